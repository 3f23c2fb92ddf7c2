/*
 * chfpe_ref.c -- CPU ORACLE (test infrastructure; see chfpe_ref.h for scope, citations and pins).
 * Plain nested loops in fp64.  The only concession to speed is an OpenMP "parallel for" over the
 * outermost loop; there is no blocking, fusion or reordering beyond the formulas cited.
 */
#include "chfpe_ref.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define MAXAX 6
#define MAXK 4096

struct chfpe_ref_handle {
  chfpe_ref_desc d;
  chfpe_ref_monomial* U;       /* owned copy */
  int M, nax, K;
  int n[MAXAX];                /* points per axis, axis a = 2s (q_s) or 2s+1 (p_s) */
  int64_t st[MAXAX];           /* canonical strides, last axis fastest */
  double h[MAXAX], x0[MAXAX];  /* spacing and first coordinate per axis */
  int64_t cells, nqcells;
  double dV;
  int (*elem)[3];              /* n(k) */
  int (*up)[3], (*dn)[3];      /* neighbour element index or -1 */
  double* Gamma;               /* sum_s n_s gamma_s */
  double* Utab;                /* U(q) on the q-subgrid, q1 slowest */
  double* dUtab[3];            /* dU/dq_s on the q-subgrid */
  double kup[3], kdn[3], cdn[3];
  double* X;                   /* state, K*cells */
  double *k1, *Y, *acc;        /* RK4 scratch */
  double *D0, *D1;             /* derivative scratch (one element each) */
};
typedef struct chfpe_ref_handle H;

static double ipow(double x, int e) { double r = 1.0; for (int i = 0; i < e; i++) r *= x; return r; }

static double coord(const H* h, int a, int i) { return h->x0[a] + i * h->h[a]; }

/* U(q) = sum of monomials, Eq. (3)-(4) PAPER.md:49-54 (general polynomial) */
static double U_eval(const H* h, const double q[3]) {
  double u = 0;
  for (int t = 0; t < h->d.n_terms; t++) {
    double v = h->U[t].coef;
    for (int s = 0; s < h->M; s++) v *= ipow(q[s], h->U[t].expo[s]);
    u += v;
  }
  return u;
}
static double dU_eval(const H* h, const double q[3], int s) {
  double u = 0;
  for (int t = 0; t < h->d.n_terms; t++) {
    int e = h->U[t].expo[s];
    if (e == 0) continue;
    double v = h->U[t].coef * e * ipow(q[s], e - 1);
    for (int r = 0; r < h->M; r++) if (r != s) v *= ipow(q[r], h->U[t].expo[r]);
    u += v;
  }
  return u;
}
/* dV_s/dq_s with V_s = V_LL q + V_SL q^2/2 */
static double Vprime(const H* h, int s, double q) { return h->d.V_LL[s] + h->d.V_SL[s] * q; }

static int64_t qlinear(const H* h, const int idx[MAXAX]) {
  int64_t l = 0;
  for (int s = 0; s < h->M; s++) l = l * h->n[2 * s] + idx[2 * s];
  return l;
}
static void decode(const H* h, int64_t cell, int idx[MAXAX]) {
  for (int a = h->nax - 1; a >= 0; a--) { idx[a] = (int)(cell % h->n[a]); cell /= h->n[a]; }
}

/* hierarchy elements: all n in N^M with sum <= depth; graded, ties by descending lexicographic (reading R5, R6) */
static int enumerate(int M, int depth, int (*out)[3]) {
  int K = 0;
  for (int lev = 0; lev <= depth; lev++) {
    if (M == 1) { if (out) { out[K][0] = lev; out[K][1] = 0; out[K][2] = 0; } K++; }
    else if (M == 2) {
      for (int a = lev; a >= 0; a--) { if (out) { out[K][0] = a; out[K][1] = lev - a; out[K][2] = 0; } K++; }
    } else {
      for (int a = lev; a >= 0; a--) for (int b = lev - a; b >= 0; b--) {
        if (out) { out[K][0] = a; out[K][1] = b; out[K][2] = lev - a - b; } K++;
      }
    }
  }
  return K;
}
static int find_elem(const H* h, const int n[3]) {
  for (int k = 0; k < h->K; k++)
    if (h->elem[k][0] == n[0] && h->elem[k][1] == n[1] && h->elem[k][2] == n[2]) return k;
  return -1;
}

int chfpe_ref_set_threads(int32_t n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
  return omp_get_max_threads();
#else
  (void)n; return 1;
#endif
}

int chfpe_ref_create(const chfpe_ref_desc* d, chfpe_ref_handle** out) {
  if (!d || !out) return -1;
  if (d->n_modes < 1 || d->n_modes > 3 || d->depth < 0 || d->beta <= 0) return -1;
  if (d->scheme < 0 || d->scheme > 2 || d->gauge < 0 || d->gauge > 1 || d->closure < 0 || d->closure > 1) return -1;
  H* h = (H*)calloc(1, sizeof(H));
  h->d = *d; h->M = d->n_modes; h->nax = 2 * h->M;
  h->U = (chfpe_ref_monomial*)malloc(sizeof(chfpe_ref_monomial) * (d->n_terms > 0 ? d->n_terms : 1));
  for (int t = 0; t < d->n_terms; t++) {
    h->U[t] = d->U[t];
    int deg = 0;
    for (int s = 0; s < 3; s++) { if (d->U[t].expo[s] < 0) { free(h->U); free(h); return -1; } if (s < h->M) deg += d->U[t].expo[s]; }
    if (deg > 4) { free(h->U); free(h); return -1; }
  }
  h->d.U = h->U;
  for (int s = 0; s < h->M; s++) {
    if (d->nq[s] < 5 || d->np[s] < 5 || d->mass[s] <= 0 || d->gamma[s] <= 0 || d->zeta[s] < 0) { free(h->U); free(h); return -1; }
    h->n[2 * s] = d->nq[s]; h->n[2 * s + 1] = d->np[s];
    h->x0[2 * s] = d->qmin[s]; h->x0[2 * s + 1] = d->pmin[s];
    h->h[2 * s] = (d->qmax[s] - d->qmin[s]) / (d->nq[s] - 1);      /* nodal grid, end points included (R8) */
    h->h[2 * s + 1] = (d->pmax[s] - d->pmin[s]) / (d->np[s] - 1);
  }
  h->cells = 1; h->nqcells = 1; h->dV = 1;
  for (int a = h->nax - 1; a >= 0; a--) { h->st[a] = h->cells; h->cells *= h->n[a]; h->dV *= h->h[a]; }
  for (int s = 0; s < h->M; s++) h->nqcells *= h->n[2 * s];
  h->K = enumerate(h->M, d->depth, NULL);
  h->elem = malloc(sizeof(int[3]) * h->K); h->up = malloc(sizeof(int[3]) * h->K); h->dn = malloc(sizeof(int[3]) * h->K);
  h->Gamma = malloc(sizeof(double) * h->K);
  enumerate(h->M, d->depth, h->elem);
  for (int k = 0; k < h->K; k++) {
    h->Gamma[k] = 0;
    for (int s = 0; s < 3; s++) {
      h->up[k][s] = h->dn[k][s] = -1;
      if (s >= h->M) continue;
      h->Gamma[k] += h->elem[k][s] * d->gamma[s];          /* sum_s n_s gamma_s, Eq. (8) :77 */
      int n[3] = { h->elem[k][0], h->elem[k][1], h->elem[k][2] };
      n[s] += 1; h->up[k][s] = find_elem(h, n);            /* -1 beyond the truncation (R5) */
      n[s] -= 2; if (n[s] >= 0) h->dn[k][s] = find_elem(h, n);
    }
  }
  for (int s = 0; s < h->M; s++) {
    h->cdn[s] = d->zeta[s] * d->gamma[s] * d->mass[s] / d->beta;   /* m zeta gamma / beta, Eq. (12) :100 */
    if (d->gauge == 1) { h->kup[s] = 0.0; h->kdn[s] = d->beta / d->mass[s]; }
    else { h->kup[s] = -d->beta / (2 * d->mass[s]); h->kdn[s] = d->beta / (2 * d->mass[s]); }
  }
  /* tables of U and dU/dq_s on the q-subgrid */
  h->Utab = malloc(sizeof(double) * h->nqcells);
  for (int s = 0; s < h->M; s++) h->dUtab[s] = malloc(sizeof(double) * h->nqcells);
  for (int64_t l = 0; l < h->nqcells; l++) {
    int iq[3] = {0, 0, 0}; int64_t r = l;
    for (int s = h->M - 1; s >= 0; s--) { iq[s] = (int)(r % h->n[2 * s]); r /= h->n[2 * s]; }
    double q[3] = {0, 0, 0};
    for (int s = 0; s < h->M; s++) q[s] = coord(h, 2 * s, iq[s]);
    h->Utab[l] = U_eval(h, q);
    for (int s = 0; s < h->M; s++) h->dUtab[s][l] = dU_eval(h, q, s);
  }
  size_t tot = (size_t)h->K * h->cells;
  h->X = calloc(tot, sizeof(double));
  if (!h->X) { chfpe_ref_destroy(h); return -2; }
  *out = h;
  return 0;
}

void chfpe_ref_destroy(chfpe_ref_handle* h) {
  if (!h) return;
  free(h->U); free(h->elem); free(h->up); free(h->dn); free(h->Gamma); free(h->Utab);
  for (int s = 0; s < 3; s++) free(h->dUtab[s]);
  free(h->X); free(h->k1); free(h->Y); free(h->acc); free(h->D0); free(h->D1);
  free(h);
}

int chfpe_ref_num_elements(const chfpe_ref_handle* h, int32_t* K) { *K = h->K; return 0; }
int64_t chfpe_ref_num_cells(const chfpe_ref_handle* h) { return h->cells; }
int chfpe_ref_element_index(const chfpe_ref_handle* h, int32_t k, int32_t n_out[3]) {
  if (k < 0 || k >= h->K) return -1;
  for (int s = 0; s < 3; s++) n_out[s] = h->elem[k][s];
  return 0;
}
int chfpe_ref_neighbor(const chfpe_ref_handle* h, int32_t k, int32_t s, int32_t* up, int32_t* dn) {
  if (k < 0 || k >= h->K || s < 0 || s >= h->M) return -1;
  *up = h->up[k][s]; *dn = h->dn[k][s]; return 0;
}

/* ---- derivative at one point, explicit schemes, zero ghost values outside the grid (R9) ---- */
static inline double fetch(const double* f, int64_t cell, int64_t st, int i, int n, int off) {
  int j = i + off;
  return (j < 0 || j >= n) ? 0.0 : f[cell + off * st];
}
static inline double D_point(const H* h, const double* f, int64_t cell, int a, int i) {
  int n = h->n[a]; int64_t st = h->st[a]; double hh = h->h[a];
  if (h->d.scheme == 0)      /* fourth-order central: [8(f+1 - f-1) - (f+2 - f-2)]/(12h) */
    return (8.0 * (fetch(f, cell, st, i, n, 1) - fetch(f, cell, st, i, n, -1))
            - (fetch(f, cell, st, i, n, 2) - fetch(f, cell, st, i, n, -2))) / (12.0 * hh);
  return (fetch(f, cell, st, i, n, 1) - fetch(f, cell, st, i, n, -1)) / (2.0 * hh);
}

/* ---- derivative of a whole element array along one axis (all schemes) ---- */
int chfpe_ref_deriv_axis(const chfpe_ref_handle* h, const double* f, int32_t a, double* out) {
  if (a < 0 || a >= h->nax) return -1;
  int n = h->n[a]; int64_t st = h->st[a]; double hh = h->h[a];
  int64_t nlines = h->cells / n;
  #pragma omp parallel
  {
    double* r = malloc(sizeof(double) * n); double* c = malloc(sizeof(double) * n);
    #pragma omp for
    for (int64_t line = 0; line < nlines; line++) {
      /* base cell of the line: insert index 0 at axis a */
      int64_t outer = line / st, inner = line % st;
      int64_t base = outer * st * n + inner;
      if (h->d.scheme != 2) {
        for (int i = 0; i < n; i++) out[base + i * st] = D_point(h, f, base + i * st, a, i);
      } else {
        /* Pade scheme Eq. (25)-(31): (1/3) d_{i-1} + d_i + (1/3) d_{i+1} = [a (f+1 - f-1) + b (f+2 - f-2)]/h,
           a = 7/9, b = 1/36 (reading R4), matrices truncated as printed in Eq. (28)-(29). */
        const double al = 1.0 / 3.0, ca = 7.0 / 9.0, cb = 1.0 / 36.0;
        for (int i = 0; i < n; i++) {
          int64_t cell = base + i * st;
          r[i] = (ca * (fetch(f, cell, st, i, n, 1) - fetch(f, cell, st, i, n, -1))
                  + cb * (fetch(f, cell, st, i, n, 2) - fetch(f, cell, st, i, n, -2))) / hh;
        }
        /* Thomas algorithm for tridiag(al, 1, al) */
        double bet = 1.0; c[0] = 0; r[0] = r[0] / bet;
        for (int i = 1; i < n; i++) {
          c[i] = al / bet;
          bet = 1.0 - al * c[i];
          r[i] = (r[i] - al * r[i - 1]) / bet;
        }
        for (int i = n - 2; i >= 0; i--) r[i] -= c[i + 1] * r[i + 1];
        for (int i = 0; i < n; i++) out[base + i * st] = r[i];
      }
    }
    free(r); free(c);
  }
  return 0;
}

/* ---- one entry of the right-hand side of Eq. (8), central schemes ---- */
static double rhs_point(const H* h, const double* X, int k, int64_t cell, const int idx[MAXAX]) {
  const double* Xk = X + (size_t)k * h->cells;
  int64_t ql = qlinear(h, idx);
  double acc = -h->Gamma[k] * Xk[cell];                              /* -(sum_s n_s gamma_s) W^(n) */
  for (int s = 0; s < h->M; s++) {
    int aq = 2 * s, ap = 2 * s + 1;
    double q = coord(h, aq, idx[aq]), p = coord(h, ap, idx[ap]);
    /* L W = sum_s [ dU/dq_s dW/dp_s - (p_s/m_s) dW/dq_s ], Eq. (9)-(10) */
    acc += -(p / h->d.mass[s]) * D_point(h, Xk, cell, aq, idx[aq]);
    acc += h->dUtab[s][ql] * D_point(h, Xk, cell, ap, idx[ap]);
    double Vp = Vprime(h, s, q);
    int ku = h->up[k][s], kd = h->dn[k][s];
    if (ku >= 0) {                                                   /* Phi_s W^(n+e_s), Eq. (11) */
      const double* Xu = X + (size_t)ku * h->cells;
      acc += Vp * (D_point(h, Xu, cell, ap, idx[ap]) + h->kup[s] * p * Xu[cell]);
    }
    if (kd >= 0) {                                                   /* n_s Theta_s W^(n-e_s), Eq. (12) + R1 */
      const double* Xd = X + (size_t)kd * h->cells;
      acc += h->elem[k][s] * h->cdn[s] * Vp * (D_point(h, Xd, cell, ap, idx[ap]) + h->kdn[s] * p * Xd[cell]);
    }
  }
  return acc;
}

int chfpe_ref_rhs_at(const chfpe_ref_handle* h, const double* X, int32_t k, int64_t cell, double* out) {
  if (h->d.scheme == 2 || h->d.closure != 0 || k < 0 || k >= h->K || cell < 0 || cell >= h->cells) return -1;
  int idx[MAXAX]; decode(h, cell, idx);
  *out = rhs_point(h, X, k, cell, idx);
  return 0;
}

static void ensure(double** p, size_t n) { if (!*p) *p = malloc(sizeof(double) * n); }

static void add_terminator(chfpe_ref_handle* h, const double* X, double* F);

/* RHS through whole-array derivatives: valid for every scheme */
int chfpe_ref_rhs_deriv(chfpe_ref_handle* h, const double* X, double* F) {
  ensure(&h->D0, h->cells);
  for (int k = 0; k < h->K; k++) {
    const double* Xk = X + (size_t)k * h->cells; double* Fk = F + (size_t)k * h->cells;
    #pragma omp parallel for
    for (int64_t c = 0; c < h->cells; c++) Fk[c] = -h->Gamma[k] * Xk[c];
    for (int s = 0; s < h->M; s++) {
      int aq = 2 * s, ap = 2 * s + 1;
      for (int term = 0; term < 4; term++) {
        const double* src; int axis;
        if (term == 0) { src = Xk; axis = aq; }
        else if (term == 1) { src = Xk; axis = ap; }
        else if (term == 2) { if (h->up[k][s] < 0) continue; src = X + (size_t)h->up[k][s] * h->cells; axis = ap; }
        else { if (h->dn[k][s] < 0) continue; src = X + (size_t)h->dn[k][s] * h->cells; axis = ap; }
        chfpe_ref_deriv_axis(h, src, axis, h->D0);
        const double* D = h->D0;
        #pragma omp parallel for
        for (int64_t c = 0; c < h->cells; c++) {
          int idx[MAXAX]; decode(h, c, idx);
          double q = coord(h, aq, idx[aq]), p = coord(h, ap, idx[ap]);
          double Vp = Vprime(h, s, q);
          if (term == 0) Fk[c] += -(p / h->d.mass[s]) * D[c];
          else if (term == 1) Fk[c] += h->dUtab[s][qlinear(h, idx)] * D[c];
          else if (term == 2) Fk[c] += Vp * (D[c] + h->kup[s] * p * src[c]);
          else Fk[c] += h->elem[k][s] * h->cdn[s] * Vp * (D[c] + h->kdn[s] * p * src[c]);
        }
      }
    }
  }
  if (h->d.closure == 1) add_terminator(h, X, F);
  return 0;
}

/* Terminator closure (reading R23; the paper is silent on the truncation).  For a top-level element
 * n (|n| = depth) the element n+e_s is not propagated; Eq. (8) for it, with everything but its damping and its
 * source dropped, 0 = -Gamma_{n+e_s} W^(n+e_s) + (n_s+1) Theta_s W^(n), slaves it to W^(n).  Step by step:
 *   Y   = (n_s+1) c_s V'_s (D_{p_s} + kappa^dn_s p_s) X_n / (Gamma_n + gamma_s)       the virtual element, whole grid
 *   F_n += V'_s (D_{p_s} + kappa^up_s p_s) Y                                           its Phi_s coupling, Eq. (11)
 * with the same discrete D (any scheme) and zero ghosts for X_n and for Y.  For depth 0 this is the Kramers
 * equation with friction zeta_s V'_s^2. */
static void add_terminator(chfpe_ref_handle* h, const double* X, double* F) {
  ensure(&h->D0, h->cells); ensure(&h->D1, h->cells);
  for (int k = 0; k < h->K; k++) {
    int lev = 0;
    for (int s = 0; s < h->M; s++) lev += h->elem[k][s];
    if (lev != h->d.depth) continue;
    const double* Xk = X + (size_t)k * h->cells; double* Fk = F + (size_t)k * h->cells;
    for (int s = 0; s < h->M; s++) {
      int aq = 2 * s, ap = 2 * s + 1;
      const double fac = (h->elem[k][s] + 1) * h->cdn[s] / (h->Gamma[k] + h->d.gamma[s]);
      chfpe_ref_deriv_axis(h, Xk, ap, h->D0);
      double* Y = h->D1;
      #pragma omp parallel for
      for (int64_t c = 0; c < h->cells; c++) {
        int idx[MAXAX]; decode(h, c, idx);
        double q = coord(h, aq, idx[aq]), p = coord(h, ap, idx[ap]);
        Y[c] = fac * Vprime(h, s, q) * (h->D0[c] + h->kdn[s] * p * Xk[c]);
      }
      chfpe_ref_deriv_axis(h, Y, ap, h->D0);
      #pragma omp parallel for
      for (int64_t c = 0; c < h->cells; c++) {
        int idx[MAXAX]; decode(h, c, idx);
        double q = coord(h, aq, idx[aq]), p = coord(h, ap, idx[ap]);
        Fk[c] += Vprime(h, s, q) * (h->D0[c] + h->kup[s] * p * Y[c]);
      }
    }
  }
}

int chfpe_ref_rhs(chfpe_ref_handle* h, const double* X, double* F) {
  if (h->d.closure == 1) {                                  /* plain right-hand side, then the slaved elements */
    const int32_t keep = h->d.closure;
    h->d.closure = 0;
    int rc = chfpe_ref_rhs(h, X, F);
    h->d.closure = keep;
    if (rc) return rc;
    add_terminator(h, X, F);
    return 0;
  }
  if (h->d.scheme == 2) return chfpe_ref_rhs_deriv(h, X, F);
  int64_t n0 = h->n[0], rest = h->cells / n0;
  #pragma omp parallel for collapse(2) schedule(static)
  for (int k = 0; k < h->K; k++)
    for (int64_t i0 = 0; i0 < n0; i0++) {
      for (int64_t r = 0; r < rest; r++) {
        int64_t cell = i0 * rest + r;
        int idx[MAXAX]; decode(h, cell, idx);
        F[(size_t)k * h->cells + cell] = rhs_point(h, X, k, cell, idx);
      }
    }
  return 0;
}

/* classical RK4 (reading R13) */
static void rk4_step(H* h, double dt) {
  size_t tot = (size_t)h->K * h->cells;
  ensure(&h->k1, tot); ensure(&h->Y, tot); ensure(&h->acc, tot);
  double *X = h->X, *k = h->k1, *Y = h->Y, *A = h->acc;
  chfpe_ref_rhs(h, X, k);                                   /* k1 = F(X) */
  #pragma omp parallel for
  for (size_t i = 0; i < tot; i++) { A[i] = k[i]; Y[i] = X[i] + 0.5 * dt * k[i]; }
  chfpe_ref_rhs(h, Y, k);                                   /* k2 = F(X + dt/2 k1) */
  #pragma omp parallel for
  for (size_t i = 0; i < tot; i++) { A[i] += 2.0 * k[i]; Y[i] = X[i] + 0.5 * dt * k[i]; }
  chfpe_ref_rhs(h, Y, k);                                   /* k3 = F(X + dt/2 k2) */
  #pragma omp parallel for
  for (size_t i = 0; i < tot; i++) { A[i] += 2.0 * k[i]; Y[i] = X[i] + dt * k[i]; }
  chfpe_ref_rhs(h, Y, k);                                   /* k4 = F(X + dt k3) */
  #pragma omp parallel for
  for (size_t i = 0; i < tot; i++) X[i] = X[i] + (dt / 6.0) * (A[i] + k[i]);
}

int chfpe_ref_step(chfpe_ref_handle* h, int64_t n_steps, double dt) {
  for (int64_t i = 0; i < n_steps; i++) rk4_step(h, dt);
  return 0;
}

/* H_sys at a cell: sum_s p_s^2/(2 m_s) + U(q) */
static double Hsys(const H* h, const int idx[MAXAX]) {
  double e = h->Utab[qlinear(h, idx)];
  for (int s = 0; s < h->M; s++) { double p = coord(h, 2 * s + 1, idx[2 * s + 1]); e += p * p / (2.0 * h->d.mass[s]); }
  return e;
}

/* Neumaier-compensated accumulation */
typedef struct { double s, c; } ksum;
static inline void kadd(ksum* k, double v) {
  double t = k->s + v;
  if (fabs(k->s) >= fabs(v)) k->c += (k->s - t) + v; else k->c += (v - t) + k->s;
  k->s = t;
}

int chfpe_ref_equilibrate(chfpe_ref_handle* h, int64_t n_steps, double dt, double* residual) {
  /* X_0 <- analytic equilibrium (e^{-beta H}/Z_W, or phi/Z_f with Z_f = dV sum phi^2), X_{k>0} <- 0 (R18) */
  size_t tot = (size_t)h->K * h->cells;
  memset(h->X, 0, sizeof(double) * tot);
  ksum z = {0, 0};
  double beta = h->d.beta;
  for (int64_t c = 0; c < h->cells; c++) {
    int idx[MAXAX]; decode(h, c, idx);
    double e = Hsys(h, idx);
    if (h->d.gauge == 1) { h->X[c] = exp(-beta * e); kadd(&z, h->X[c]); }
    else { h->X[c] = exp(-0.5 * beta * e); kadd(&z, h->X[c] * h->X[c]); }
  }
  double Z = (z.s + z.c) * h->dV;
  for (int64_t c = 0; c < h->cells; c++) h->X[c] /= Z;
  chfpe_ref_step(h, n_steps, dt);
  if (residual) {
    ensure(&h->k1, tot);
    chfpe_ref_rhs(h, h->X, h->k1);
    ksum a = {0, 0}, b = {0, 0};
    for (size_t i = 0; i < tot; i++) { kadd(&a, h->k1[i] * h->k1[i]); kadd(&b, h->X[i] * h->X[i]); }
    *residual = sqrt((a.s + a.c) / (b.s + b.c));
  }
  return 0;
}

/* dX/dq_s for X(q) = c0 + sum lin_q q + 1/2 sum quad q q', Eq. (13)-(14) */
static double obs_dq(const H* h, const chfpe_ref_observable* o, int s, const double q[3]) {
  double v = o->lin_q[s];
  for (int r = 0; r < h->M; r++) v += 0.5 * (o->quad[s][r] + o->quad[r][s]) * q[r];
  return v;
}
static double obs_val(const H* h, const chfpe_ref_observable* o, const double q[3], const double p[3]) {
  double v = o->c0;
  for (int s = 0; s < h->M; s++) {
    v += o->lin_q[s] * q[s] + o->lin_p[s] * p[s];
    for (int r = 0; r < h->M; r++) v += 0.5 * o->quad[s][r] * q[s] * q[r];
  }
  return v;
}

/* Kick, Eq. (18) :131, on every element (R11); in the sqrt(W_eq) gauge d/dp -> d/dp + kup p */
int chfpe_ref_kick(chfpe_ref_handle* h, const chfpe_ref_observable* o) {
  ensure(&h->D0, h->cells); ensure(&h->D1, h->cells);
  for (int k = 0; k < h->K; k++) {
    double* Xk = h->X + (size_t)k * h->cells;
    double* out = h->D1;
    for (int64_t c = 0; c < h->cells; c++) out[c] = 0.0;
    for (int s = 0; s < h->M; s++) {
      chfpe_ref_deriv_axis(h, Xk, 2 * s + 1, h->D0);
      #pragma omp parallel for
      for (int64_t c = 0; c < h->cells; c++) {
        int idx[MAXAX]; decode(h, c, idx);
        double q[3] = {0, 0, 0};
        for (int r = 0; r < h->M; r++) q[r] = coord(h, 2 * r, idx[2 * r]);
        double p = coord(h, 2 * s + 1, idx[2 * s + 1]);
        out[c] += obs_dq(h, o, s, q) * (h->D0[c] + h->kup[s] * p * Xk[c]);
      }
    }
    memcpy(Xk, out, sizeof(double) * h->cells);
  }
  return 0;
}

/* dV * sum_cells O(q,p) w X_k, w = 1 (W gauge) or phi = e^{-beta H/2} (sqrt gauge); Eq. (15) */
int chfpe_ref_expect_element(chfpe_ref_handle* h, int32_t k, const chfpe_ref_observable* o, double* out) {
  if (k < 0 || k >= h->K) return -1;
  const double* Xk = h->X + (size_t)k * h->cells;
  int64_t n0 = h->n[0], rest = h->cells / n0;
  double* part = malloc(sizeof(double) * n0);
  #pragma omp parallel for
  for (int64_t i0 = 0; i0 < n0; i0++) {
    ksum a = {0, 0};
    for (int64_t r = 0; r < rest; r++) {
      int64_t c = i0 * rest + r;
      int idx[MAXAX]; decode(h, c, idx);
      double q[3] = {0, 0, 0}, p[3] = {0, 0, 0};
      for (int s = 0; s < h->M; s++) { q[s] = coord(h, 2 * s, idx[2 * s]); p[s] = coord(h, 2 * s + 1, idx[2 * s + 1]); }
      double w = (h->d.gauge == 1) ? 1.0 : exp(-0.5 * h->d.beta * Hsys(h, idx));
      kadd(&a, obs_val(h, o, q, p) * w * Xk[c]);
    }
    part[i0] = a.s + a.c;
  }
  ksum t = {0, 0};
  for (int64_t i0 = 0; i0 < n0; i0++) kadd(&t, part[i0]);
  free(part);
  *out = (t.s + t.c) * h->dV;
  return 0;
}
int chfpe_ref_expect(chfpe_ref_handle* h, const chfpe_ref_observable* o, double* out) {
  return chfpe_ref_expect_element(h, 0, o, out);            /* element 0 only (R12) */
}

/* R1[k] = <C> after k*stride steps from Kick(A) state; literal Eq. (15) (R3) */
int chfpe_ref_response_1d(chfpe_ref_handle* h, const chfpe_ref_observable* A, const chfpe_ref_observable* C,
                          int64_t n_samples, int64_t stride, double dt, double* R) {
  chfpe_ref_kick(h, A);
  for (int64_t k = 0; k < n_samples; k++) {
    chfpe_ref_expect(h, C, &R[k]);
    if (k + 1 < n_samples) chfpe_ref_step(h, stride, dt);
  }
  return 0;
}

/* R2[k][j]: T <- Kick(A) state; advance T to t1[k]; Y <- Kick(B) T; <C> on Y after t2[j] steps; Eq. (16) */
int chfpe_ref_response_2d(chfpe_ref_handle* h, const chfpe_ref_observable* A, const chfpe_ref_observable* B,
                          const chfpe_ref_observable* C, const int64_t* t1, int32_t n1,
                          const int64_t* t2, int32_t n2, double dt, double* R) {
  size_t tot = (size_t)h->K * h->cells;
  double* T = malloc(sizeof(double) * tot);
  if (!T) return -2;
  chfpe_ref_kick(h, A);
  int64_t now1 = 0;
  for (int k = 0; k < n1; k++) {
    if (t1[k] < now1) { free(T); return -1; }
    chfpe_ref_step(h, t1[k] - now1, dt); now1 = t1[k];
    memcpy(T, h->X, sizeof(double) * tot);                  /* keep the t1 trajectory */
    chfpe_ref_kick(h, B);
    int64_t now2 = 0;
    for (int j = 0; j < n2; j++) {
      if (t2[j] < now2) { free(T); return -1; }
      chfpe_ref_step(h, t2[j] - now2, dt); now2 = t2[j];
      chfpe_ref_expect(h, C, &R[(size_t)k * n2 + j]);
    }
    memcpy(h->X, T, sizeof(double) * tot);
  }
  free(T);
  return 0;
}

/* R3[k][j][l] (row f2 of DESIGN.md): Eq. (17) PAPER.md:126-127 written out, literal like Eq. (15)-(16) (no sign, R3):
   T1 <- Kick(A) state, advanced to t1[k]; T2 <- Kick(B) T1, advanced to t2[j]; Y <- Kick(C) T2; <D> on Y after
   t3[l] steps.  Plain triple loop; the two trajectories are kept as copies. */
int chfpe_ref_response_3d(chfpe_ref_handle* h, const chfpe_ref_observable* A, const chfpe_ref_observable* B,
                          const chfpe_ref_observable* C, const chfpe_ref_observable* D, const int64_t* t1, int32_t n1,
                          const int64_t* t2, int32_t n2, const int64_t* t3, int32_t n3, double dt, double* R) {
  size_t tot = (size_t)h->K * h->cells;
  double* T1 = malloc(sizeof(double) * tot);
  double* T2 = malloc(sizeof(double) * tot);
  if (!T1 || !T2) { free(T1); free(T2); return -2; }
  int rc = 0;
  chfpe_ref_kick(h, A);
  int64_t now1 = 0;
  for (int k = 0; k < n1 && !rc; k++) {
    if (t1[k] < now1) { rc = -1; break; }
    chfpe_ref_step(h, t1[k] - now1, dt); now1 = t1[k];
    memcpy(T1, h->X, sizeof(double) * tot);                 /* keep the t1 trajectory */
    chfpe_ref_kick(h, B);
    int64_t now2 = 0;
    for (int j = 0; j < n2 && !rc; j++) {
      if (t2[j] < now2) { rc = -1; break; }
      chfpe_ref_step(h, t2[j] - now2, dt); now2 = t2[j];
      memcpy(T2, h->X, sizeof(double) * tot);               /* keep the t2 trajectory */
      chfpe_ref_kick(h, C);
      int64_t now3 = 0;
      for (int l = 0; l < n3; l++) {
        if (t3[l] < now3) { rc = -1; break; }
        chfpe_ref_step(h, t3[l] - now3, dt); now3 = t3[l];
        chfpe_ref_expect(h, D, &R[((size_t)k * n2 + j) * n3 + l]);
      }
      memcpy(h->X, T2, sizeof(double) * tot);
    }
    memcpy(h->X, T1, sizeof(double) * tot);
  }
  free(T1); free(T2);
  return rc;
}

int chfpe_ref_export_state(const chfpe_ref_handle* h, double* dst) {
  memcpy(dst, h->X, sizeof(double) * (size_t)h->K * h->cells); return 0;
}
int chfpe_ref_import_state(chfpe_ref_handle* h, const double* src) {
  memcpy(h->X, src, sizeof(double) * (size_t)h->K * h->cells); return 0;
}

int chfpe_ref_scaled_norm2(const chfpe_ref_handle* h, double* out) {
  ksum t = {0, 0};
  for (int k = 0; k < h->K; k++) {
    double w = 1.0;
    for (int s = 0; s < h->M; s++)
      for (int j = 1; j <= h->elem[k][s]; j++) w *= j * h->cdn[s];
    const double* Xk = h->X + (size_t)k * h->cells;
    ksum a = {0, 0};
    for (int64_t c = 0; c < h->cells; c++) kadd(&a, Xk[c] * Xk[c]);
    kadd(&t, (a.s + a.c) / w);
  }
  *out = (t.s + t.c) * h->dV;
  return 0;
}
