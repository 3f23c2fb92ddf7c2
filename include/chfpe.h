/*
 * chfpe.h -- C-ABI boundary of the B200-native multimode CHFPE hot path (libchfpe.so).
 *
 * Method: R. Hoshino and Y. Tanimura, "A Multimode Classical Hierarchical Fokker-Planck Equations
 * Approach to Molecular Vibrations: Simulating Two-Dimensional Spectra" (arXiv 2509.25840).
 * Citations below are line numbers of the paper text plus the equation they fall in;
 * "R<n>" are the readings of garbled / silent passages listed in DESIGN.md.
 *
 * The library time-propagates the whole hierarchy W^(n)(q1,p1,...,qM,pM), M = 1..3, on a uniform
 * phase-space grid in fp64, applies Poisson-bracket kicks, reduces phase-space expectations and runs
 * the 1D / 2D response protocols.  Every step runs in hand-written sm_100a CUDA kernels; there is no
 * CPU fallback (calls fail with CHFPE_ERR_CUDA when no device / kernel image is available).
 *
 * Conventions
 *   - All functions return int: CHFPE_OK (0) or a negative CHFPE_ERR_* code.  They never throw,
 *     abort or print.  chfpe_last_error() returns a static or handle-owned message.
 *   - "host" / "device" is stated for every pointer.  Device memory and the CUDA stream are OWNED BY
 *     THE CALLER: the library carves its state arrays, stage buffers, tables and reduction scratch out
 *     of the single workspace passed to chfpe_create and never allocates device memory itself.
 *   - Calls are asynchronous on the stream given at create time, except those that return host data
 *     (expect, response_*, equilibrate with residual_out, export to host), which synchronise that
 *     stream only.  A handle is not thread-safe; distinct handles are independent.
 *   - Canonical (import/export) layout of one replica: X[k][i_q1][i_p1]...[i_qM][i_pM], last axis
 *     fastest, hierarchy element k outermost ("hierarchy-major"), fp64.  X = W (gauge W) or
 *     X = f = W / sqrt(W_eq) (gauge SQRT_EQ, default).  The internal device layout differs (q-major /
 *     p-minor bricks) and is not exposed.
 *   - Element order (R5, R6): all n in N^M with n_1+...+n_M <= depth; ascending |n|, ties by
 *     descending lexicographic (n_1,...,n_M).
 */
#ifndef CHFPE_H
#define CHFPE_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum {
  CHFPE_OK = 0,
  CHFPE_ERR_INVALID = -1,    /* bad descriptor / argument (M not in 1..3, < 5 grid points, degree > 4, ...) */
  CHFPE_ERR_WORKSPACE = -2,  /* workspace too small or not 256-byte aligned */
  CHFPE_ERR_CUDA = -3,       /* CUDA runtime error; message from cudaGetErrorString */
  CHFPE_ERR_DIVERGED = -4,   /* non-finite expectation value, or the norm guard of chfpe_step tripped */
  CHFPE_ERR_STATE = -5       /* call sequence error (e.g. response before equilibrate/import) */
};

enum { CHFPE_CENTRAL4 = 0, CHFPE_CENTRAL2 = 1, CHFPE_COMPACT6 = 2 };   /* derivative scheme; COMPACT6 = Pade scheme Eq. (25)-(31) :177-201 with a = 7/9 (R4), one fused line pass per axis */
enum { CHFPE_GAUGE_SQRT_EQ = 0, CHFPE_GAUGE_W = 1 };                   /* propagated variable (R7) */
/* Closure of the hierarchy at the top level |n| = depth (the paper is silent; readings R5, R23):
   TRUNCATE drops W^(n+e_s); TERMINATOR slaves it to its source, W^(n+e_s) = (n_s+1) Theta_s W^(n) / Gamma_{n+e_s},
   which turns Phi_s W^(n+e_s) (Eq. 11-12 :96-100) into a second-derivative Fokker-Planck term (depth 0: the Kramers
   equation with friction zeta_s V'_s^2).  Explicit schemes only, phase-space grid representation only. */
enum { CHFPE_CLOSURE_TRUNCATE = 0, CHFPE_CLOSURE_TERMINATOR = 1 };

/* coef * q1^e1 q2^e2 q3^e3 ; total degree <= 4.  Eq. (3)-(4). */
typedef struct { double coef; int32_t expo[3]; } chfpe_monomial;

/* Model + discretisation.  Copied at create time.  Entries beyond n_modes are ignored. */
typedef struct {
  int32_t n_modes;                    /* M = 1..3 */
  double  mass[3];                    /* m_s, Eq. (2) :45 */
  int32_t n_terms; const chfpe_monomial* U;   /* host; U(q) incl. harmonic, anharmonic and mode-mode terms */
  double  V_LL[3], V_SL[3];           /* V_s = V_LL q + V_SL q^2/2 */
  double  zeta[3], gamma[3], beta;    /* Drude baths Eq. (7) :67, inverse temperature */
  int32_t nq[3], np[3];               /* grid points per axis (>= 5) */
  double  qmin[3], qmax[3], pmin[3], pmax[3];   /* nodal uniform grid, end points included (R8) */
  int32_t depth;                      /* N: elements n with sum(n) <= N */
  int32_t scheme;                     /* CHFPE_CENTRAL4 (default) | CHFPE_CENTRAL2 | CHFPE_COMPACT6 */
  int32_t gauge;                      /* CHFPE_GAUGE_SQRT_EQ (default) | CHFPE_GAUGE_W (literal Eq. 8) */
  int32_t batch;                      /* B >= 1 independent replicas (state slots) sharing the operator */
  int32_t closure;                    /* CHFPE_CLOSURE_TRUNCATE (default) | CHFPE_CLOSURE_TERMINATOR */
} chfpe_desc;

/* X(q,p) = c0 + sum lin_q[s] q_s + 1/2 sum quad[s][s'] q_s q_s' + sum lin_p[s] p_s ; Eq. (13)-(14) :108-113.
   lin_p and c0 are used by chfpe_expect only (kick needs dX/dq_s). */
typedef struct { double c0, lin_q[3], quad[3][3], lin_p[3]; } chfpe_observable;

typedef struct chfpe_handle chfpe_handle;     /* opaque, host side, owned by the library */

/* Device bytes the caller must provide for this descriptor (256-byte aligned).  out: host. */
int chfpe_workspace_bytes(const chfpe_desc* desc, size_t* bytes);

/* Build tables (setup step a0), carve the workspace, zero all replicas.  dev_workspace: device, caller-owned,
   must outlive the handle.  cuda_stream: a cudaStream_t (0 = legacy default stream).  Section IV.A, :217-219. */
int chfpe_create(const chfpe_desc* desc, void* dev_workspace, size_t bytes, void* cuda_stream, chfpe_handle** out);

/* Frees the host struct only (the workspace stays with the caller). */
int chfpe_destroy(chfpe_handle* h);

int chfpe_num_elements(const chfpe_handle* h, int32_t* K);                  /* K = C(N+M, M) */
int chfpe_element_index(const chfpe_handle* h, int32_t k, int32_t n_out[3]); /* canonical order */

/* All replicas: X_0 <- analytic equilibrium (e^{-beta H}/Z or phi/Z_f), X_{k>0} <- 0, then n_steps RK4 steps
   (section IV.B, :221-223; R18).  residual_out (host, may be NULL) <- ||F(X)||_2 / ||X||_2 of replica 0. */
int chfpe_equilibrate(chfpe_handle* h, int64_t n_steps, double dt, double* residual_out);

/* n_steps fourth-order Runge-Kutta steps of Eq. (8) :77-80 on every replica (R13: evaluated in the
   Horner form of the same degree-4 polynomial in dt*L, the generator being linear and autonomous).
   Norm guard: returns CHFPE_ERR_DIVERGED if, after the steps, the state of a replica is not finite or its sum of
   squares exceeds 1e8 times its value at the last equilibrate / import / kick / response call (the literal W gauge
   is unstable on a phase-space grid, reading R7).  The check is one reduction and synchronises the stream. */
int chfpe_step(chfpe_handle* h, int64_t n_steps, double dt);

/* Every element of every replica: X_k <- sum_s (dX/dq_s) (d/dp_s) X_k, Eq. (18) :131, literal (no sign; R3, R11). */
int chfpe_kick(chfpe_handle* h, const chfpe_observable* X);

/* out[b] (host, length batch) <- integral of O(q,p) W^(0) over phase space for replica b, Eq. (15) :119 (R10, R12). */
int chfpe_expect(chfpe_handle* h, const chfpe_observable* O, double* out);

/* Same reduction on element k of replica `replica` (tests of the hierarchy normalisation). out: host, 1 double. */
int chfpe_expect_element(chfpe_handle* h, int32_t replica, int32_t k, const chfpe_observable* O, double* out);

/* R1: replica 0 <- Kick(A) replica 0; for i in 0..n_samples-1: R[i] = <C>, then `stride` steps (none after the
   last sample).  Literal Eq. (15) :119, section IV.C.1 :229-233.  R: host, n_samples doubles.  Other replicas
   untouched.  A == NULL skips the kick and continues the trajectory replica 0 already holds. */
int chfpe_response_1d(chfpe_handle* h, const chfpe_observable* A, const chfpe_observable* C,
                      int64_t n_samples, int64_t stride, double dt, double* R);

/* R2[k][j]: T <- Kick(A) replica 0, advanced along t1; at t1_steps[k] a copy of T gets Kick(B) and is propagated
   over the t2 grid, <C> recorded after t2_steps[j] steps.  Literal Eq. (16) :121-122, section IV.C.2 :235-237.
   Step lists: host, ascending, >= 0.  R: host, row-major [n1][n2].  With batch >= 2, batch-1 replicas (different
   t1) are propagated together per launch; with batch == 1 an extra workspace slot is used sequentially. */
int chfpe_response_2d(chfpe_handle* h, const chfpe_observable* A, const chfpe_observable* B, const chfpe_observable* C,
                      const int64_t* t1_steps, int32_t n1, const int64_t* t2_steps, int32_t n2,
                      double dt, double* R);

/* R3[k][j][l] (row f2 of DESIGN.md): T1 <- Kick(A) replica 0, advanced along t1; at t1_steps[k] a copy T2 of T1 gets
   Kick(B) and is advanced along t2; at t2_steps[j] a copy of T2 gets Kick(C) and is propagated over the t3 grid, <D>
   recorded after t3_steps[l] steps.  Literal Eq. (17) :126-127 (no sign, like Eq. 15-16).  Step lists: host,
   ascending, >= 0.  R: host, row-major [n1][n2][n3].  Replicas of different t1 are propagated together per launch:
   slot 0 = T1; a group of nb t1 samples uses slots [1, 1+nb) for its t2 trajectories and [1+nb, 1+2nb) for the t3
   replicas, nb = (batch-1)/2; at the last t2 sample C is applied in place, so n2 == 1 (a fixed waiting time, the
   scan of Eq. 21) runs nb = batch-1 replicas.  CHFPE_ERR_INVALID if nb < 1 or nb*n3 exceeds the 65536-entry results
   buffer.  On return replica 0 holds T1 at t1_steps[n1-1]. */
int chfpe_response_3d(chfpe_handle* h, const chfpe_observable* A, const chfpe_observable* B, const chfpe_observable* C,
                      const chfpe_observable* D, const int64_t* t1_steps, int32_t n1, const int64_t* t2_steps,
                      int32_t n2, const int64_t* t3_steps, int32_t n3, double dt, double* R);

/* Canonical-layout copy of one replica out of / into the library (K*cells doubles). dst/src: device if *_is_device. */
int chfpe_export_state(chfpe_handle* h, int32_t replica, double* dst, int dst_is_device);
int chfpe_import_state(chfpe_handle* h, int32_t replica, const double* src, int src_is_device);

/* F(X) of replica `replica` (right-hand side of Eq. (8)), canonical layout, for operator-level parity tests. */
int chfpe_export_rhs(chfpe_handle* h, int32_t replica, double* dst, int dst_is_device);

/* Stage-level access for a slab-decomposed propagation (row f4: one propagation split along q_1 over
   several GPUs needs the two boundary planes of every element of the STAGE INPUT from its neighbours before every
   stage).  chfpe_rk4_stage runs stage `stage` = 0..3 of one RK4 step (Horner form, R13) on every replica:
     0: v_a = y + dt/4 F(y)   1: v_b = y + dt/3 F(v_a)   2: v_a = y + dt/2 F(v_b)   3: y = y + dt F(v_a)
   so four calls with stage = 0, 1, 2, 3 are exactly chfpe_step(h, 1, dt) without its norm guard.
   chfpe_stage_input returns the DEVICE pointer of the array that stage `stage` reads (y, v_a, v_b, v_a) for one replica,
   in the library's internal layout X[k][i_q1][i_q2..i_qM][i_p1..i_pM] (q-major / p-minor, last axis fastest): the q_1
   plane i of element k is the contiguous run of *plane_doubles doubles at dev + (k * nq_1 + i) * plane_doubles.  The
   caller may overwrite such planes (halo planes of a slab) on the handle's stream between stages; the pointer stays
   valid for the life of the handle. */
int chfpe_rk4_stage(chfpe_handle* h, int32_t stage, double dt);
int chfpe_stage_input(chfpe_handle* h, int32_t replica, int32_t stage, double** dev, int64_t* plane_doubles);

/* Number of kernels the library has launched on this handle since create (bench.py's gpu_launches). */
int chfpe_launch_count(const chfpe_handle* h, int64_t* n);

/* Device timing of the dominant kernel (the fused RK-stage kernel, steps a1-a3).  While enabled, every stage
   launch is bracketed by two CUDA events on the handle's stream.  chfpe_profile_read synchronises the stream,
   returns the summed duration (milliseconds) and the number of stage launches since the last read (host
   pointers), and resets both.  Off by default; the events cost about a microsecond per launch. */
int chfpe_profile_enable(chfpe_handle* h, int on);
int chfpe_profile_read(chfpe_handle* h, double* total_ms, int64_t* n_launches);

/* Spectra (row f3 of DESIGN.md): half-line Fourier integrals of sampled response functions, Eq. (19)-(21) :138-146,
   as trapezoid sums over the uniform delay grid t_k = k dt (weights 1/2, 1, ..., 1, 1/2; no window, no padding;
   reading R22) at the frequencies the caller lists.  No handle: ALL pointers are DEVICE pointers, the kernels are
   enqueued on `cuda_stream` (asynchronous), nothing is allocated.
     spectrum_1d, Eq. (19):  I[a] = omega[a] * Im sum_k w_k e^{+i omega[a] t_k} R[k] dt          (R: n, I: n_omega)
     spectrum_2d, Eq. (20):  I[a][b] = Im sum_k sum_j w_k w_j e^{i sign1 omega1[a] k dt1} e^{i sign2 omega2[b] j dt2}
                             R[k][j] dt1 dt2       (R row-major [n1][n2], I row-major [n_omega1][n_omega2]);
                             sign1 = sign2 = -1 is Eq. (20); Eq. (21) at one waiting time is sign1 = -1 (t1),
                             sign2 = +1 (t3) on R3[:, j, :].  scratch: 2*n1*n_omega2 doubles, 16-byte aligned.
   CHFPE_ERR_INVALID for null pointers, sizes < 1, dt <= 0, signs other than +-1. */
int chfpe_spectrum_1d(void* cuda_stream, const double* R, int64_t n, double dt, const double* omega, int32_t n_omega,
                      double* I);
int chfpe_spectrum_2d(void* cuda_stream, const double* R, int32_t n1, int32_t n2, double dt1, double dt2,
                      const double* omega1, int32_t n_omega1, const double* omega2, int32_t n_omega2, int32_t sign1,
                      int32_t sign2, double* scratch, double* I);

/* chfpe_spectrum_2d for callers that can neither allocate nor provide the scratch array (CUDA graph capture, serving
   loops, harnesses that forbid cudaMalloc): same arguments without `scratch`, same result.  The complex scratch
   T[n1][n_omega2] is a file-scope device array inside the library of CHFPE_SPECTRUM_STATIC_MAX entries (1 MiB, held
   by every GPU that loads the library until exit); the call allocates and frees nothing.
   CHFPE_ERR_WORKSPACE if n1 * n_omega2 > CHFPE_SPECTRUM_STATIC_MAX, CHFPE_ERR_INVALID as for chfpe_spectrum_2d.
   All calls share the array (contents of the last call remain; nothing needs clearing: the first pass writes every
   entry the second reads).  Calls that overlap on the GPU -- different streams, or one stream per thread -- RACE on
   it: serialise them.  Successive calls on one stream are safe. */
#define CHFPE_SPECTRUM_STATIC_MAX 65536
int chfpe_spectrum_2d_static(void* cuda_stream, const double* R, int32_t n1, int32_t n2, double dt1, double dt2,
                             const double* omega1, int32_t n_omega1, const double* omega2, int32_t n_omega2,
                             int32_t sign1, int32_t sign2, double* I);

/* Which kernel family runs the RK stage on this handle (host pointer), so that a test or a benchmark can assert
   that a configuration did not fall back to the generic kernel.  The cooperative multi-step kernel of tiny
   states is a property of the step call, not of the handle, and is not reported here. */
enum { CHFPE_STAGE_GENERIC = 0, CHFPE_STAGE_BRICK = 1, CHFPE_STAGE_COMPACT = 3, CHFPE_STAGE_TMA = 4 };   /* (2: a removed experiment) */
int chfpe_stage_kernel(const chfpe_handle* h, int32_t* kind);

const char* chfpe_last_error(const chfpe_handle* h);   /* h may be NULL: last create-time error */

/* ---- Hermite-in-momentum representation (row f1 of DESIGN.md): the paper's production scheme -----------------------
   Eq. (22)-(23) :156-164: W^(n)(p,q) = prod_s psi_0(p_s) e^{-beta U(q)/2} sum_k c^(n)_k(q) prod_s psi_{k_s}(p_s), psi_j the
   orthonormal Hermite functions of width sqrt(2 m_s/beta); equations of motion = de-garbled Eq. (A1)-(A4) :343-355
   (reading R19 of DESIGN.md, with the n_s factor of R1):
     d/dt c^(n)_k = sum_s [ sqrt(k_s+1) D+_s c^(n)_{k+e_s} - sqrt(k_s) D-_s c^(n)_{k-e_s} ] - Gamma_n c^(n)_k
                  + sum_s V'_s [ n_s gamma_s zeta_s sqrt(m_s/beta) sqrt(k_s+1) c^(n-e_s)_{k+e_s} - sqrt(k_s beta/m_s) c^(n+e_s)_{k-e_s} ],
     D+-_s g = (dU/dq_s) / (2 sqrt(m_s/beta)) g -+ (1/sqrt(m_s beta)) dg/dq_s.
   The same chfpe_desc is used with np[s] = number of Hermite functions of mode s (>= 1); pmin/pmax and gauge are
   ignored; scheme = CHFPE_CENTRAL4 | CHFPE_CENTRAL2 (explicit q-stencils, zero ghosts R9) | CHFPE_COMPACT6 (the paper's
   Pade q-derivative Eq. (25)-(31) :177-201 with a = 7/9 (R4): one tridiagonal line solve per slab, mode and q-line; at
   most 256 points per q axis; a stage is 1 + M launches).  State layout of one replica
   (import/export AND device): c[element][k_1]..[k_M][i_q1]..[i_qM], last axis fastest, fp64; element order as above.
   Same conventions as the grid calls: caller-owned 256-byte aligned device workspace and stream, int return codes,
   host pointers unless stated, calls returning host data synchronise the stream.  No CPU fallback. */
typedef struct chfpe_hermite_handle chfpe_hermite_handle;
int chfpe_hermite_workspace_bytes(const chfpe_desc* desc, size_t* bytes);
int chfpe_hermite_create(const chfpe_desc* desc, void* dev_workspace, size_t bytes, void* cuda_stream,
                         chfpe_hermite_handle** out);
int chfpe_hermite_destroy(chfpe_hermite_handle* h);
int chfpe_hermite_num_elements(const chfpe_hermite_handle* h, int32_t* K);
/* All replicas: c^(0)_0 <- e^{-beta U/2} / Z_q (Z_q = dV sum_q e^{-beta U}), all other coefficients 0, then n_steps
   RK4 steps (section IV.B :221-223).  residual_out (may be NULL) <- ||F(c)||_2 / ||c||_2 of replica 0. */
int chfpe_hermite_equilibrate(chfpe_hermite_handle* h, int64_t n_steps, double dt, double* residual_out);
/* n_steps RK4 steps on every replica (Horner form of the degree-4 Taylor polynomial, R13). */
int chfpe_hermite_step(chfpe_hermite_handle* h, int64_t n_steps, double dt);
/* Eq. (18) :131 on every element of every replica: c_k <- sum_s (dX/dq_s) (-sqrt(k_s beta/m_s)) c_{k-e_s}. */
int chfpe_hermite_kick(chfpe_hermite_handle* h, const chfpe_observable* X);
/* out[b] (length batch) <- int int O W^(element) dp dq = dV sum_q e^{-beta U/2} [ O(q) c_0 + sum_s lin_p[s] sqrt(m_s/beta) c_{e_s} ]
   of replica b (Eq. 15 :119 for element 0). */
int chfpe_hermite_expect(chfpe_hermite_handle* h, int32_t element, const chfpe_observable* O, double* out);
/* Same protocols as chfpe_response_1d / _2d (literal Eq. 15, 16); response_2d needs batch >= 2 (slot 0 carries the
   t1 trajectory, batch-1 replicas of different t1 advance together per launch). */
int chfpe_hermite_response_1d(chfpe_hermite_handle* h, const chfpe_observable* A, const chfpe_observable* C,
                              int64_t n_samples, int64_t stride, double dt, double* R);
int chfpe_hermite_response_2d(chfpe_hermite_handle* h, const chfpe_observable* A, const chfpe_observable* B,
                              const chfpe_observable* C, const int64_t* t1_steps, int32_t n1, const int64_t* t2_steps,
                              int32_t n2, double dt, double* R);
/* Same protocol as chfpe_response_3d (literal Eq. 17 :126-127; R row-major [n1][n2][n3]): slot 0 = t1 trajectory, a group
   of nb = (batch-1)/2 t1 samples (batch-1 if n2 == 1) owns nb slots for its t2 trajectories and nb for the t3 replicas.
   CHFPE_ERR_INVALID if nb < 1 or nb*n3 exceeds the 65536-entry results buffer. */
int chfpe_hermite_response_3d(chfpe_hermite_handle* h, const chfpe_observable* A, const chfpe_observable* B,
                              const chfpe_observable* C, const chfpe_observable* D, const int64_t* t1_steps, int32_t n1,
                              const int64_t* t2_steps, int32_t n2, const int64_t* t3_steps, int32_t n3, double dt,
                              double* R);
/* K * prod(np) * prod(nq) doubles; dst/src: device if *_is_device, else host. */
int chfpe_hermite_export_state(chfpe_hermite_handle* h, int32_t replica, double* dst, int dst_is_device);
int chfpe_hermite_import_state(chfpe_hermite_handle* h, int32_t replica, const double* src, int src_is_device);
int chfpe_hermite_export_rhs(chfpe_hermite_handle* h, int32_t replica, double* dst, int dst_is_device);
int chfpe_hermite_launch_count(const chfpe_hermite_handle* h, int64_t* n);
/* Which kernel family runs the RK stage on this handle (benchmark records and tests; the results do not depend on it):
   per-value kernel | column kernel (one mode) | patch kernel | COMPACT6 pointwise + line passes | bulk-copy march kernel
   (three modes on an n_1 x 32 x 32 mesh with n_1 even: the default there, for the explicit stencils and for COMPACT6). */
enum { CHFPE_HERMITE_STAGE_VALUE = 0, CHFPE_HERMITE_STAGE_COLUMN = 1, CHFPE_HERMITE_STAGE_PATCH = 2,
       CHFPE_HERMITE_STAGE_COMPACT = 3, CHFPE_HERMITE_STAGE_TMA = 4,
       CHFPE_HERMITE_STAGE_COMPACT_TMA = 5 };   /* COMPACT6 on such a mesh: march kernel with the q_2, q_3 line solves inside + q_1 line pass */
int chfpe_hermite_stage_kernel(const chfpe_hermite_handle* h, int32_t* kind);
const char* chfpe_hermite_last_error(const chfpe_hermite_handle* h);   /* h may be NULL: last create-time error */

/* ---------------------------------------------------------------------------------------------------------------
   Tunables.  The library reads the following environment variables once per chfpe_create / chfpe_hermite_create.
   They select among kernel variants and launch plans that compute THE SAME results (every one is covered by a parity
   test); they exist for measurements and for the tests that force the variants small inputs would not reach.
   Unset = the measured default.  A value without an instantiated kernel falls back to the next kernel family.
     Stage kernel family (phase-space grid, M >= 2, explicit schemes)
       CHFPE_BRICK=0          generic one-thread-per-value stage kernel instead of the brick / bulk-copy kernels
       CHFPE_TMA=0            three modes, CENTRAL4: k_stage_brick3 (register-staged loads) instead of k_stage_tma
       CHFPE_TMA_NPART=1|2    p_1 parts per brick of k_stage_tma (default 2 from 12 planes on)
       CHFPE_TMA_NSEG=n       thread groups (p_1 segments) per part
       CHFPE_TMA_SLOTS=4|5    ring slots (default 5; 4 for 20^3 bricks)
       CHFPE_TMA_RING=0       load the q_3 neighbour bricks as chunks instead of carrying them in registers
       CHFPE_BRICK_SPLIT=n, CHFPE_BRICK_MINB=n, CHFPE_BRICK_NPASS=n   thread decomposition of k_stage_brick3
       CHFPE_BPC=n            consecutive bricks per CTA of k_stage_brick3
     Sweep order and L2 policy (both brick kernels)
       CHFPE_GROUP=g          hierarchy elements swept in lock-step (default: 4 with k_stage_tma, else 2, if they fit)
       CHFPE_Q2CHUNK=r        q_2 rows per sweep chunk
       CHFPE_L2_WINDOW_MB=m   L2 budget of the reuse window (default 64)
       CHFPE_L2MODE=bits      bit 0: once-touched data evict_first, bit 1: window data evict_last (default 3 / 1)
     Other kernels
       CHFPE_COOP=0|1|2       persistent cooperative step kernel: off | states <= 1 MB (default) | states <= 24 MB
       CHFPE_KICK_BRICK=0     generic kick kernel + copy back instead of the in-place brick kick
       CHFPE_COMPACT_CUBE=0   run-time-shaped brick pass also for 16^3 / 48^2 bricks and line passes for 20^3 bricks
                              (default there: brick pass with a compile-time shape)
       CHFPE_COMPACT_QPLANE=0 COMPACT6, three modes: one line pass per q axis instead of the fused (q_2, q_3) plane pass (16- and
                              20-point axes)
       CHFPE_COMPACT_PCOLUMN=0 COMPACT6, 16^3 / 20^3 bricks: k_compact_pbrick instead of the thread-per-column brick pass
       CHFPE_COMPACT_QLINE=0  COMPACT6: generic line kernel also for 16-, 20- and (two modes) 48-point q lines (default there:
                              k_compact_qline / k_compact_qline_long)
       CHFPE_EXPECT_PBRICK=0  generic reduction (index decode per cell) instead of the factorised expectation kernel
       CHFPE_COMPACT_PBRICK=0|1|2   COMPACT6 p-derivatives: one line pass per momentum axis | one brick pass for bricks of
                              up to 4096 cells (default) | brick pass for bricks of up to 8192 cells as well
     Hermite representation
       CHFPE_HERMITE_KC=0|4|8 per-value kernel | column kernel with 4 / 8 Hermite indices per thread
       CHFPE_HERMITE_PATCH=AB patch kernel with A x B points of (q_1, q_2) per thread (0: off)
       CHFPE_HERMITE_FIXED=0, CHFPE_HERMITE_TILE=0, CHFPE_HERMITE_PCOL=0   32^3 specialisation / CTA tile remap / column
                              walk off
       CHFPE_HERMITE_CONTIG=0 strided instead of transposing COMPACT6 line kernel on the contiguous axis
       CHFPE_HERMITE_TMA=0    patch kernel (COMPACT6: pointwise pass + three line passes) instead of the bulk-copy march
                              kernel (n_1 x 32 x 32 meshes of three modes; an explicit CHFPE_HERMITE_KC / CHFPE_HERMITE_PATCH
                              request also turns it off)
   --------------------------------------------------------------------------------------------------------------- */

#ifdef __cplusplus
}
#endif
#endif
