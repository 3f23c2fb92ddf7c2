// Host-side evaluation of the polynomial potential U(q) of Eq. (3)-(4) PAPER.md:49-54 and of its gradient for the setup
// tables (step a0): the monomial list of chfpe_desc is folded once into a dense coefficient tensor C[e1][e2][e3]
// (degree <= 4 per coordinate), the gradient tensors are G_s[e] = (e_s + 1) C[e + e_s], and values are taken by nested
// Horner evaluation.  (Deliberately not the term-by-term power loop of the CPU oracle: the two table generators share
// neither code nor algorithm.)
#pragma once
#include "../../include/chfpe.h"

struct ChfpePoly {
  static constexpr int D = 5;                     // exponents 0..4
  double c[D][D][D];
  double g[3][D][D][D];

  void build(const chfpe_monomial* U, int n_terms, int M) {
    for (int a = 0; a < D; a++) for (int b = 0; b < D; b++) for (int e = 0; e < D; e++) {
      c[a][b][e] = 0.0;
      for (int s = 0; s < 3; s++) g[s][a][b][e] = 0.0;
    }
    for (int t = 0; t < n_terms; t++) {
      int e[3] = {0, 0, 0};
      for (int s = 0; s < M; s++) e[s] = U[t].expo[s];
      c[e[0]][e[1]][e[2]] += U[t].coef;
    }
    for (int a = 0; a < D; a++) for (int b = 0; b < D; b++) for (int e = 0; e < D; e++) {
      if (a + 1 < D) g[0][a][b][e] = (a + 1) * c[a + 1][b][e];
      if (b + 1 < D) g[1][a][b][e] = (b + 1) * c[a][b + 1][e];
      if (e + 1 < D) g[2][a][b][e] = (e + 1) * c[a][b][e + 1];
    }
  }
  static double horner(const double (&t)[D][D][D], const double q[3]) {
    double r1 = 0.0;
    for (int a = D - 1; a >= 0; a--) {
      double r2 = 0.0;
      for (int b = D - 1; b >= 0; b--) {
        double r3 = 0.0;
        for (int e = D - 1; e >= 0; e--) r3 = r3 * q[2] + t[a][b][e];
        r2 = r2 * q[1] + r3;
      }
      r1 = r1 * q[0] + r2;
    }
    return r1;
  }
  double value(const double q[3]) const { return horner(c, q); }
  double grad(int s, const double q[3]) const { return horner(g[s], q); }
};
