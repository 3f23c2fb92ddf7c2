// COMPACT6 derivative path (step a9 of DESIGN.md): the sixth-order Pade scheme of PAPER.md Eq. (25)-(31) :177-201,
//     (1/3) d_{i-1} + d_i + (1/3) d_{i+1} = [ a (f_{i+1} - f_{i-1}) + b (f_{i+2} - f_{i-2}) ] / h,
// a = 7/9, b = 1/36 (reading R4: the printed a = 7/18 is not consistent), matrices truncated as printed in
// Eq. (28)-(29) (zero ghosts, R9).  The tridiagonal systems are solved per grid line by the Thomas recurrence with the
// elimination factors of the constant matrix tridiag(1/3, 1, 1/3) tabulated once per axis on the host; the paper's own
// choice for this step is parallel cyclic reduction on Ampere-class GPUs (section III.C :203-207) -- at line lengths
// of 16..128 one thread per line is enough to occupy the GPU (a 16^6 grid has 10^6 lines per element and axis).
//
// This is the conditional, correctness-first path of SURVEY.md 8(a9): the RHS is assembled element by element from
// whole-array derivatives (one line solve per (element, axis) on X_k along q_s, one on the combination
// G_s = (dU/dq_s) X_k + V'_s X_up + n_s c_s V'_s X_dn along p_s), not fused; the explicit CENTRAL4 scheme is the
// performance path.
#include "chfpe_internal.cuh"

namespace {

template <int NAX>
__device__ __forceinline__ void cdecode(const DevOp& op, unsigned cell, int (&idx)[NAX]) {
#pragma unroll
  for (int a = NAX - 1; a >= 0; a--) {
    const unsigned q = cell / (unsigned)op.n[a];
    idx[a] = (int)(cell - q * (unsigned)op.n[a]);
    cell = q;
  }
}

// d = A^{-1} B f along `axis` for every grid line of one element array; one thread per line.
// bet[i], cfac[i]: elimination factors of tridiag(1/3,1,1/3) with n rows (host-tabulated per axis).
__global__ void __launch_bounds__(128) k_compact_deriv(const double* __restrict__ f, double* __restrict__ d, long long nlines,
                                                       int n, long long st, double inv_h, const double* __restrict__ bet,
                                                       const double* __restrict__ cfac) {
  const long long line = (long long)blockIdx.x * 128 + threadIdx.x;
  if (line >= nlines) return;
  const long long outer = line / st, inner = line - outer * st;
  const long long base = outer * st * n + inner;
  const double al = 1.0 / 3.0, ca = 7.0 / 9.0, cb = 1.0 / 36.0;
  double fm2 = 0.0, fm1 = 0.0, f0 = f[base], fp1 = (n > 1) ? f[base + st] : 0.0, prev = 0.0;
  for (int i = 0; i < n; i++) {                                    // forward elimination, r'_i stored in d
    const double fp2 = (i + 2 < n) ? f[base + (long long)(i + 2) * st] : 0.0;
    const double r = (ca * (fp1 - fm1) + cb * (fp2 - fm2)) * inv_h;
    prev = (i == 0) ? r / __ldg(bet) : (r - al * prev) / __ldg(bet + i);
    d[base + (long long)i * st] = prev;
    fm2 = fm1; fm1 = f0; f0 = fp1; fp1 = fp2;
  }
  double next = prev;                                              // back substitution
  for (int i = n - 2; i >= 0; i--) {
    next = d[base + (long long)i * st] - __ldg(cfac + i + 1) * next;
    d[base + (long long)i * st] = next;
  }
}

// G_s = (dU/dq_s) X_k + V'_s X_up + n_s c_s V'_s X_dn  (per cell)
template <int M>
__global__ void __launch_bounds__(256) k_compact_G(DevOp op, const double* __restrict__ X, int k, int s, double* __restrict__ G) {
  const long long cell = (long long)blockIdx.x * 256 + threadIdx.x;
  if (cell >= op.cells) return;
  int idx[2 * M];
  cdecode<2 * M>(op, (unsigned)cell, idx);
  const long long ql = (long long)((unsigned)cell / (unsigned)op.pb);
  const double q = op.x0[s] + idx[s] * op.h[s];
  const double Vp = fma(op.VSL[s], q, op.VLL[s]);
  double g = __ldg(op.dU[s] + ql) * X[(size_t)k * op.cells + cell];
  const int ku = __ldg(op.up + 3 * k + s), kd = __ldg(op.dn + 3 * k + s);
  if (ku >= 0) g = fma(Vp, X[(size_t)ku * op.cells + cell], g);
  if (kd >= 0) g = fma(__ldg(op.nvec + 3 * k + s) * op.cdn[s] * Vp, X[(size_t)kd * op.cells + cell], g);
  G[cell] = g;
}

// F = -Gamma_k X_k + sum_s p_s V'_s (kup_s X_up + n_s c_s kdn_s X_dn)   (damping and the gauge terms, pointwise)
template <int M>
__global__ void __launch_bounds__(256) k_compact_init(DevOp op, const double* __restrict__ X, int k, double* __restrict__ F) {
  const long long cell = (long long)blockIdx.x * 256 + threadIdx.x;
  if (cell >= op.cells) return;
  int idx[2 * M];
  cdecode<2 * M>(op, (unsigned)cell, idx);
  double acc = -__ldg(op.Gamma + k) * X[(size_t)k * op.cells + cell];
#pragma unroll
  for (int s = 0; s < M; s++) {
    const double q = op.x0[s] + idx[s] * op.h[s];
    const double p = op.x0[M + s] + idx[M + s] * op.h[M + s];
    const double Vp = fma(op.VSL[s], q, op.VLL[s]);
    const int ku = __ldg(op.up + 3 * k + s), kd = __ldg(op.dn + 3 * k + s);
    if (ku >= 0) acc = fma(Vp * op.kup[s] * p, X[(size_t)ku * op.cells + cell], acc);
    if (kd >= 0) acc = fma(__ldg(op.nvec + 3 * k + s) * op.cdn[s] * Vp * op.kdn[s] * p, X[(size_t)kd * op.cells + cell], acc);
  }
  F[cell] = acc;
}

// F += coef(cell) * D, coef = -(p_s / m_s) (mode 0, the q_s-derivative of X_k) or 1 (mode 1, the p_s-derivative of G_s)
template <int M>
__global__ void __launch_bounds__(256) k_compact_accum(DevOp op, const double* __restrict__ D, int s, int mode, double* __restrict__ F) {
  const long long cell = (long long)blockIdx.x * 256 + threadIdx.x;
  if (cell >= op.cells) return;
  double c = 1.0;
  if (mode == 0) {
    int idx[2 * M];
    cdecode<2 * M>(op, (unsigned)cell, idx);
    c = -(op.x0[M + s] + idx[M + s] * op.h[M + s]) * op.inv_mass[s];
  }
  F[cell] = fma(c, D[cell], F[cell]);
}

// kick (Eq. 18): F (+)= dX/dq_s (D + kup_s p_s X_k)
template <int M>
__global__ void __launch_bounds__(256) k_compact_kick_accum(DevOp op, DevObs ob, const double* __restrict__ Xk,
                                                            const double* __restrict__ D, int s, int first, double* __restrict__ F) {
  const long long cell = (long long)blockIdx.x * 256 + threadIdx.x;
  if (cell >= op.cells) return;
  int idx[2 * M];
  cdecode<2 * M>(op, (unsigned)cell, idx);
  double g = ob.lin_q[s];
#pragma unroll
  for (int r = 0; r < M; r++) g = fma(0.5 * (ob.quad[s][r] + ob.quad[r][s]), op.x0[r] + idx[r] * op.h[r], g);
  const double p = op.x0[M + s] + idx[M + s] * op.h[M + s];
  const double v = g * fma(op.kup[s] * p, Xk[cell], D[cell]);
  F[cell] = first ? v : F[cell] + v;
}

__global__ void __launch_bounds__(256) k_compact_combine(const double* __restrict__ F, const double* y, double* out, long long n,
                                                         double a, double c) {
  const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
  if (i < n) out[i] = fma(c, F[i], a * y[i]);
}

}  // namespace

#define CDISPATCH(M, CALL) do { if ((M) == 1) { CALL(1); } else if ((M) == 2) { CALL(2); } else { CALL(3); } } while (0)

static int compact_deriv(const DevOp& op, const CompactTables& ct, const double* f, int axis, double* d, cudaStream_t s) {
  const int n = op.n[axis];
  const long long nlines = op.cells / n;
  k_compact_deriv<<<(unsigned)((nlines + 127) / 128), 128, 0, s>>>(f, d, nlines, n, op.st[axis], 1.0 / op.h[axis],
                                                                   ct.bet[axis], ct.cfac[axis]);
  return 1;
}

// out = a*y + c*F(in) for slots [0, nb); scratch: three element-sized arrays (G, D, F)
int launch_stage_compact(const DevOp& op, const CompactTables& ct, const double* in, const double* y, double* out, double a,
                         double c, int nb, size_t slot_stride, double* scratch, cudaStream_t s) {
  int launches = 0;
  const unsigned blocks = (unsigned)((op.cells + 255) / 256);
  double *G = scratch, *D = scratch + op.cells, *F = scratch + 2 * op.cells;
  for (int b = 0; b < nb; b++) {
    const double* X = in + (size_t)b * slot_stride;
    for (int k = 0; k < op.K; k++) {
#define CALL(MM) k_compact_init<MM><<<blocks, 256, 0, s>>>(op, X, k, F)
      CDISPATCH(op.M, CALL);
#undef CALL
      launches++;
      for (int sI = 0; sI < op.M; sI++) {
        launches += compact_deriv(op, ct, X + (size_t)k * op.cells, sI, D, s);            // d/dq_s of X_k
#define CALL(MM) k_compact_accum<MM><<<blocks, 256, 0, s>>>(op, D, sI, 0, F)
        CDISPATCH(op.M, CALL);
#undef CALL
#define CALL(MM) k_compact_G<MM><<<blocks, 256, 0, s>>>(op, X, k, sI, G)
        CDISPATCH(op.M, CALL);
#undef CALL
        launches += 2 + compact_deriv(op, ct, G, op.M + sI, D, s);                        // d/dp_s of G_s
#define CALL(MM) k_compact_accum<MM><<<blocks, 256, 0, s>>>(op, D, sI, 1, F)
        CDISPATCH(op.M, CALL);
#undef CALL
        launches++;
      }
      const size_t o = (size_t)b * slot_stride + (size_t)k * op.cells;
      k_compact_combine<<<blocks, 256, 0, s>>>(F, y + o, out + o, op.cells, a, c);
      launches++;
    }
  }
  return launches;
}

// out_k = Kick_obs(in_k) for every element of slots [0, nb)
int launch_kick_compact(const DevOp& op, const CompactTables& ct, const DevObs& o, const double* in, double* out, int nb,
                        size_t slot_stride, double* scratch, cudaStream_t s) {
  int launches = 0;
  const unsigned blocks = (unsigned)((op.cells + 255) / 256);
  double* D = scratch + op.cells;
  for (int b = 0; b < nb; b++)
    for (int k = 0; k < op.K; k++) {
      const size_t off = (size_t)b * slot_stride + (size_t)k * op.cells;
      for (int sI = 0; sI < op.M; sI++) {
        launches += compact_deriv(op, ct, in + off, op.M + sI, D, s);
#define CALL(MM) k_compact_kick_accum<MM><<<blocks, 256, 0, s>>>(op, o, in + off, D, sI, sI == 0 ? 1 : 0, out + off)
        CDISPATCH(op.M, CALL);
#undef CALL
        launches++;
      }
    }
  return launches;
}
