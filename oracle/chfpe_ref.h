/*
 * chfpe_ref.h -- CPU ORACLE for the multimode CHFPE hot path (TEST INFRASTRUCTURE, not the product).
 *
 * Plain, slow, fp64, host-only restatement of what the path computes, written from PAPER.md
 * (Hoshino & Tanimura, arXiv 2509.25840) and the readings listed in DESIGN.md.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
 * It shares no code, header, table generator or helper with the CUDA path
 * (paper_2509_25840_b200/csrc); the struct layouts below are declared here independently.
 *
 * What is computed (citations are PAPER.md line numbers):
 *   state X = K hierarchy elements x phase-space grid (q1,p1,...,qM,pM), canonical layout
 *   X[k][i_q1][i_p1]...[i_qM][i_pM], last axis fastest (hierarchy-major).
 *   RHS       : Eq. (8) :77-80 with Liouvillian Eq. (9)-(10) :86-91, Phi Eq. (11) :96, Theta Eq. (12) :100,
 *               damping sum_s n_s gamma_s, and the factor n_s on the down-coupling that Appendix A1 (:345)
 *               carries (reading R1).
 *   gauges    : X = W (literal Eq. 8) or X = f = W / sqrt(W_eq), the grid analogue of the prefactor
 *               psi_0(p) exp(-beta U/2) of Eq. (22) :156-158 (reading R7).
 *   derivative: CENTRAL4 / CENTRAL2 explicit stencils with zero ghosts, or COMPACT6 = Pade scheme
 *               Eq. (25)-(31) :177-201 with a = 7/9, b = 1/36, alpha = 1/3 (reading R4), Thomas solve.
 *   step      : classical RK4 (reading R13).
 *   kick      : Eq. (18) :131 applied to every element.
 *   expect    : integral of O(q,p) W^(0), Eq. (15)-(16) :119-122, Riemann sum.
 *   responses : R1 Eq. (15), R2 Eq. (16), literal (no (-1)^N), protocol of section IV.C :229-237.
 *
 * Pins (tests/test_oracle_pins.py): closed-form Brownian-oscillator response, exact moment ODEs,
 * Boltzmann stationarity order, 2D closed form, rigid rotation, norm contraction, independent dense
 * (Kronecker) assembly, Pade order; the SL coupling V'_s = V_LL + V_SL q by the short-time
 * expansion R_phys(t) = t/m - [<U''>/m + zeta gamma <V'^2>_eq] t^3/(6m) (test_short_time_expansion_pins_Vprime).
 * Unpinned: absolute anharmonic response values at finite times (the analytic results of refs. 58-59 are
 * not in this container) and the paper's water spectra (figures only) -- "parity unpinned" for those beyond
 * stationarity, contraction, convergence, the short-time coefficient and the dense-assembly check.
 */
#ifndef CHFPE_REF_H
#define CHFPE_REF_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct { double coef; int32_t expo[3]; } chfpe_ref_monomial; /* coef * q1^e1 q2^e2 q3^e3 */

typedef struct {
  int32_t n_modes;
  double  mass[3];
  int32_t n_terms; const chfpe_ref_monomial* U;
  double  V_LL[3], V_SL[3];
  double  zeta[3], gamma[3], beta;
  int32_t nq[3], np[3];
  double  qmin[3], qmax[3], pmin[3], pmax[3];
  int32_t depth;
  int32_t scheme;   /* 0 CENTRAL4, 1 CENTRAL2, 2 COMPACT6 */
  int32_t gauge;    /* 0 sqrt(W_eq) gauge, 1 W gauge */
  int32_t batch;    /* ignored by the oracle (always one state) */
  int32_t closure;  /* 0 plain truncation (reading R5), 1 terminator: at the top level |n| = depth the missing element is
                       slaved to its source, W^(n+e_s) = (n_s+1) Theta_s W^(n) / Gamma_{n+e_s} (reading R23) */
} chfpe_ref_desc;

typedef struct { double c0, lin_q[3], quad[3][3], lin_p[3]; } chfpe_ref_observable;

typedef struct chfpe_ref_handle chfpe_ref_handle;

int     chfpe_ref_create(const chfpe_ref_desc*, chfpe_ref_handle** out);
void    chfpe_ref_destroy(chfpe_ref_handle*);
int     chfpe_ref_num_elements(const chfpe_ref_handle*, int32_t* K);
int64_t chfpe_ref_num_cells(const chfpe_ref_handle*);
int     chfpe_ref_element_index(const chfpe_ref_handle*, int32_t k, int32_t n_out[3]);
int     chfpe_ref_neighbor(const chfpe_ref_handle*, int32_t k, int32_t s, int32_t* up, int32_t* dn);
/* derivative of ONE element array (cells doubles) along grid axis a (0=q1,1=p1,2=q2,...) */
int     chfpe_ref_deriv_axis(const chfpe_ref_handle*, const double* f, int32_t axis, double* out);
/* full right-hand side, X and F are K*cells doubles, canonical layout.  _deriv works for all schemes
   (derivative arrays, then the sum of Eq. 8); _rhs uses the point formula for the central schemes. */
int     chfpe_ref_rhs(chfpe_ref_handle*, const double* X, double* F);
int     chfpe_ref_rhs_deriv(chfpe_ref_handle*, const double* X, double* F);
/* one entry of the RHS, central schemes only (used for sampled checks at full size) */
int     chfpe_ref_rhs_at(const chfpe_ref_handle*, const double* X, int32_t k, int64_t cell, double* out);
int     chfpe_ref_equilibrate(chfpe_ref_handle*, int64_t n_steps, double dt, double* residual);
int     chfpe_ref_step(chfpe_ref_handle*, int64_t n_steps, double dt);
int     chfpe_ref_kick(chfpe_ref_handle*, const chfpe_ref_observable*);
int     chfpe_ref_expect(chfpe_ref_handle*, const chfpe_ref_observable*, double* out);
/* expectation read from element k instead of 0 (moment pins need the integrals of W^(1), W^(2)) */
int     chfpe_ref_expect_element(chfpe_ref_handle*, int32_t k, const chfpe_ref_observable*, double* out);
int     chfpe_ref_response_1d(chfpe_ref_handle*, const chfpe_ref_observable* A, const chfpe_ref_observable* C,
                              int64_t n_samples, int64_t stride, double dt, double* R);
int     chfpe_ref_response_2d(chfpe_ref_handle*, const chfpe_ref_observable* A, const chfpe_ref_observable* B,
                              const chfpe_ref_observable* C, const int64_t* t1_steps, int32_t n1,
                              const int64_t* t2_steps, int32_t n2, double dt, double* R);
/* Eq. (17): R[k][j][l] = <D> after t3_steps[l] steps of Kick(C) [t2_steps[j] steps of Kick(B) [t1_steps[k] steps of
   Kick(A) X]]; row-major [n1][n2][n3] */
int     chfpe_ref_response_3d(chfpe_ref_handle*, const chfpe_ref_observable* A, const chfpe_ref_observable* B,
                              const chfpe_ref_observable* C, const chfpe_ref_observable* D,
                              const int64_t* t1_steps, int32_t n1, const int64_t* t2_steps, int32_t n2,
                              const int64_t* t3_steps, int32_t n3, double dt, double* R);
int     chfpe_ref_export_state(const chfpe_ref_handle*, double* dst);
int     chfpe_ref_import_state(chfpe_ref_handle*, const double* src);
/* sum_n ||X_n||^2 / prod_s [ n_s! (zeta_s gamma_s m_s / beta)^{n_s} ] * dV  (contraction pin P6) */
int     chfpe_ref_scaled_norm2(const chfpe_ref_handle*, double* out);
int     chfpe_ref_set_threads(int32_t n);   /* OpenMP threads used by the loops; returns the count in use */

#ifdef __cplusplus
}
#endif
#endif
