// sm_100a kernels of the CHFPE hot path: RK stage (Liouvillian stencil + hierarchy couplings + stage combine),
// kick, expectation reduction, equilibrium initialisation, layout conversion.
// Equations: PAPER.md Eq. (8)-(12) :77-100, (15)-(18) :119-131; readings R1, R3, R7, R9-R13 of DESIGN.md.
#include <cooperative_groups.h>
#include "chfpe_internal.cuh"

namespace {

// cell -> per-axis indices; 32-bit arithmetic (chfpe_create rejects grids of 2^31 cells or more): a 64-bit
// division costs ~80 instructions, and these kernels are instruction-bound
template <int NAX>
__device__ __forceinline__ void decode(const DevOp& op, long long cell64, int (&idx)[NAX]) {
  unsigned cell = (unsigned)cell64;
#pragma unroll
  for (int a = NAX - 1; a >= 0; a--) {
    const unsigned q = cell / (unsigned)op.n[a];
    idx[a] = (int)(cell - q * (unsigned)op.n[a]);
    cell = q;
  }
}
__device__ __forceinline__ long long qlinear(const DevOp& op, long long cell) {   // index of the q-point of a cell
  return (long long)((unsigned)cell / (unsigned)op.pb);
}

// explicit antisymmetric stencil with zero ghosts (R9): c1 (f[+1]-f[-1]) + c2 (f[+2]-f[-2])
__device__ __forceinline__ double dstencil(const double* __restrict__ f, long long cell, long long st, int i, int n,
                                           double c1, double c2, bool wide) {
  double fp1 = (i + 1 < n) ? __ldg(f + cell + st) : 0.0;
  double fm1 = (i >= 1) ? __ldg(f + cell - st) : 0.0;
  double d = c1 * (fp1 - fm1);
  if (wide) {
    double fp2 = (i + 2 < n) ? __ldg(f + cell + 2 * st) : 0.0;
    double fm2 = (i >= 2) ? __ldg(f + cell - 2 * st) : 0.0;
    d = fma(c2, fp2 - fm2, d);
  }
  return d;
}

// Loads of the stage input: read-only path inside one-stage launches, L2-coherent (.cg) inside the persistent
// multi-stage kernel, where other SMs have just written the array.
template <bool COHERENT>
__device__ __forceinline__ double ldx(const double* p) { return COHERENT ? __ldcg(p) : __ldg(p); }

template <bool COHERENT>
__device__ __forceinline__ double dstencil_x(const double* __restrict__ f, long long cell, long long st, int i, int n,
                                             double c1, double c2, bool wide) {
  double fp1 = (i + 1 < n) ? ldx<COHERENT>(f + cell + st) : 0.0;
  double fm1 = (i >= 1) ? ldx<COHERENT>(f + cell - st) : 0.0;
  double d = c1 * (fp1 - fm1);
  if (wide) {
    double fp2 = (i + 2 < n) ? ldx<COHERENT>(f + cell + 2 * st) : 0.0;
    double fm2 = (i >= 2) ? ldx<COHERENT>(f + cell - 2 * st) : 0.0;
    d = fma(c2, fp2 - fm2, d);
  }
  return d;
}

// Terminator closure (reading R23) for a top-level element k, mode s: the element n+e_s that is not propagated is
//   Y = (n_s+1) c_s V'_s (D_{p_s} + kappa^dn_s p_s) X_k / (Gamma_k + gamma_s)        (Eq. 12 with its damping only)
// and feeds back through Phi_s (Eq. 11): V'_s (D_{p_s} + kappa^up_s p_s) Y, with zero ghosts for X_k and for Y (R9).
// One value: nine points of X_k along p_s.
template <bool COHERENT>
__device__ __forceinline__ double terminator_value(const DevOp& op, const double* __restrict__ Xk, long long cell, int ap,
                                                   int i, double Vp, double fac, double kup, double kdn, bool wide) {
  const int n = op.n[ap];
  const long long st = op.st[ap];
  const double c1 = op.c1[ap], c2 = wide ? op.c2[ap] : 0.0;
  const double p0 = op.x0[ap], h = op.h[ap];
  double v[9];
#pragma unroll
  for (int j = -4; j <= 4; j++) v[j + 4] = (i + j >= 0 && i + j < n) ? ldx<COHERENT>(Xk + cell + j * st) : 0.0;
  double A[5];                                                      // (D + kdn p) X at i-2..i+2, zero outside the grid
#pragma unroll
  for (int j = -2; j <= 2; j++) {
    const double d = fma(c2, v[j + 6] - v[j + 2], c1 * (v[j + 5] - v[j + 3]));
    A[j + 2] = (i + j >= 0 && i + j < n) ? fma(kdn * fma((double)(i + j), h, p0), v[j + 4], d) : 0.0;
  }
  const double dA = fma(c2, A[4] - A[0], c1 * (A[3] - A[1]));
  return fac * Vp * Vp * fma(kup * fma((double)i, h, p0), A[2], dA);
}

// F_k(X)(cell), right-hand side of Eq. (8) :77-80 for one (element, cell): Liouvillian Eq. (9)-(10), Phi Eq. (11),
// n_s Theta Eq. (12) + R1, damping.  X points at element 0 of the replica.
template <int M, bool COHERENT>
__device__ __forceinline__ double rhs_value(const DevOp& op, const double* __restrict__ X, int k, long long cell) {
  const double* Xk = X + (size_t)k * op.cells;
  int idx[2 * M];
  decode<2 * M>(op, cell, idx);
  const long long ql = qlinear(op, cell);
  const bool wide = (op.scheme == CHFPE_CENTRAL4);
  double acc = -__ldg(op.Gamma + k) * ldx<COHERENT>(Xk + cell);
#pragma unroll
  for (int s = 0; s < M; s++) {
    const int aq = s, ap = M + s;
    const double q = op.x0[aq] + idx[aq] * op.h[aq];
    const double p = op.x0[ap] + idx[ap] * op.h[ap];
    const double dq = dstencil_x<COHERENT>(Xk, cell, op.st[aq], idx[aq], op.n[aq], op.c1[aq], op.c2[aq], wide);
    const double dp = dstencil_x<COHERENT>(Xk, cell, op.st[ap], idx[ap], op.n[ap], op.c1[ap], op.c2[ap], wide);
    acc = fma(-(p * op.inv_mass[s]), dq, acc);                      // -(p_s/m_s) dW/dq_s
    acc = fma(__ldg(op.dU[s] + ql), dp, acc);                       // +(dU/dq_s) dW/dp_s
    const double Vp = fma(op.VSL[s], q, op.VLL[s]);
    const int ku = __ldg(op.up + 3 * k + s), kd = __ldg(op.dn + 3 * k + s);
    if (ku >= 0) {                                                  // Phi_s W^(n+e_s)
      const double* Xu = X + (size_t)ku * op.cells;
      double d = dstencil_x<COHERENT>(Xu, cell, op.st[ap], idx[ap], op.n[ap], op.c1[ap], op.c2[ap], wide);
      acc = fma(Vp, fma(op.kup[s] * p, ldx<COHERENT>(Xu + cell), d), acc);
    }
    if (kd >= 0) {                                                  // n_s Theta_s W^(n-e_s)
      const double* Xd = X + (size_t)kd * op.cells;
      double d = dstencil_x<COHERENT>(Xd, cell, op.st[ap], idx[ap], op.n[ap], op.c1[ap], op.c2[ap], wide);
      acc = fma(__ldg(op.nvec + 3 * k + s) * op.cdn[s] * Vp, fma(op.kdn[s] * p, ldx<COHERENT>(Xd + cell), d), acc);
    }
    if (op.closure == CHFPE_CLOSURE_TERMINATOR && ku < 0) {         // top level: the missing element is slaved (R23)
      const double fac = (__ldg(op.nvec + 3 * k + s) + 1) * op.cdn[s] / (__ldg(op.Gamma + k) + op.gam[s]);
      acc += terminator_value<COHERENT>(op, Xk, cell, ap, idx[ap], Vp, fac, op.kup[s], op.kdn[s], wide);
    }
  }
  return acc;
}

// out += c * (terminator terms of element k) for the stage kernels that evaluate plain truncation only
template <int M>
__global__ void __launch_bounds__(256) k_terminator_add(DevOp op, const double* __restrict__ in, double* out, double c,
                                                        size_t slot_stride) {
  long long cell = (long long)blockIdx.x * 256 + threadIdx.x;
  if (cell >= op.cells) return;
  const int k = blockIdx.y;
  int lev = 0;
#pragma unroll
  for (int s = 0; s < M; s++) lev += __ldg(op.nvec + 3 * k + s);
  if (lev != op.depth) return;                                      // (simplex truncation: up(k, s) is missing for every s)
  const size_t boff = (size_t)blockIdx.z * slot_stride + (size_t)k * op.cells;
  const double* Xk = in + boff;
  int idx[2 * M];
  decode<2 * M>(op, cell, idx);
  const bool wide = (op.scheme == CHFPE_CENTRAL4);
  double acc = 0.0;
#pragma unroll
  for (int s = 0; s < M; s++) {
    const double q = op.x0[s] + idx[s] * op.h[s];
    const double Vp = fma(op.VSL[s], q, op.VLL[s]);
    const double fac = (__ldg(op.nvec + 3 * k + s) + 1) * op.cdn[s] / (__ldg(op.Gamma + k) + op.gam[s]);
    acc += terminator_value<false>(op, Xk, cell, M + s, idx[M + s], Vp, fac, op.kup[s], op.kdn[s], wide);
  }
  out[boff + cell] = fma(c, acc, out[boff + cell]);
}

// ------------------------------------------------------------------------------------------------
// Generic RK stage: out = a*y + c*F(in), one thread per (cell, element, slot).  Correct for every M, grid
// and explicit scheme; the brick kernels replace it where they apply.
// ------------------------------------------------------------------------------------------------
template <int M>
__global__ void __launch_bounds__(256) k_stage_generic(DevOp op, const double* __restrict__ in,
                                                       const double* y, double* out,
                                                       double a, double c, size_t slot_stride) {
  long long cell = (long long)blockIdx.x * 256 + threadIdx.x;
  if (cell >= op.cells) return;
  const int k = blockIdx.y;
  const size_t boff = (size_t)blockIdx.z * slot_stride;
  const double acc = rhs_value<M, false>(op, in + boff, k, cell);
  const size_t o = boff + (size_t)k * op.cells + cell;
  out[o] = fma(c, acc, a * y[o]);
}

// Kick, Eq. (18): out_k = sum_s dX/dq_s (D_{p_s} + kup_s p_s) in_k
template <int M>
__global__ void __launch_bounds__(256) k_kick_generic(DevOp op, DevObs ob, const double* __restrict__ in,
                                                      double* __restrict__ out, size_t slot_stride) {
  long long cell = (long long)blockIdx.x * 256 + threadIdx.x;
  if (cell >= op.cells) return;
  const int k = blockIdx.y;
  const size_t boff = (size_t)blockIdx.z * slot_stride + (size_t)k * op.cells;
  const double* Xk = in + boff;
  int idx[2 * M];
  decode<2 * M>(op, cell, idx);
  const bool wide = (op.scheme == CHFPE_CENTRAL4);
  double q[M];
#pragma unroll
  for (int s = 0; s < M; s++) q[s] = op.x0[s] + idx[s] * op.h[s];
  const double xc = __ldg(Xk + cell);
  double acc = 0.0;
#pragma unroll
  for (int s = 0; s < M; s++) {
    const int ap = M + s;
    const double p = op.x0[ap] + idx[ap] * op.h[ap];
    double g = ob.lin_q[s];
#pragma unroll
    for (int r = 0; r < M; r++) g = fma(0.5 * (ob.quad[s][r] + ob.quad[r][s]), q[r], g);
    double d = dstencil(Xk, cell, op.st[ap], idx[ap], op.n[ap], op.c1[ap], op.c2[ap], wide);
    acc = fma(g, fma(op.kup[s] * p, xc, d), acc);
  }
  out[boff + cell] = acc;
}

// Kick in place on the brick layout (M >= 2): one CTA per p-brick (all momenta of one (element, q-point), contiguous).
// The kick is local to the brick -- p-derivatives only, dX/dq_s depends on q alone -- so the brick is staged in shared
// memory, every cell is formed from it and written back to where it came from: one read and one write of the state,
// no second array and no copy back (the generic kernel above needs both).
template <int M>
__global__ void __launch_bounds__(256) k_kick_brick(DevOp op, DevObs ob, double* x, size_t slot_stride) {
  extern __shared__ __align__(16) double kb[];
  const long long ql = blockIdx.x;
  const int k = blockIdx.y;
  const int pb = (int)op.pb;
  double* X = x + (size_t)blockIdx.z * slot_stride + (size_t)k * op.cells + (size_t)ql * pb;
  for (int i = threadIdx.x; i < pb / 2; i += 256)
    reinterpret_cast<double2*>(kb)[i] = __ldcs(reinterpret_cast<const double2*>(X) + i);
  if ((pb & 1) && threadIdx.x == 0) kb[pb - 1] = X[pb - 1];
  int iq[M];
  {
    long long r = ql;
#pragma unroll
    for (int s = M - 1; s >= 0; s--) { iq[s] = (int)(r % op.n[s]); r /= op.n[s]; }
  }
  double g[M];                                                      // dX/dq_s at this q-point, Eq. (13)-(14), (18)
#pragma unroll
  for (int s = 0; s < M; s++) {
    g[s] = ob.lin_q[s];
#pragma unroll
    for (int r = 0; r < M; r++) g[s] = fma(0.5 * (ob.quad[s][r] + ob.quad[r][s]), op.x0[r] + iq[r] * op.h[r], g[s]);
  }
  const bool wide = (op.scheme == CHFPE_CENTRAL4);
  __syncthreads();
  for (int c = threadIdx.x; c < pb; c += 256) {
    int r = c;
    const double xc = kb[c];
    double acc = 0.0;
#pragma unroll
    for (int s = M - 1; s >= 0; s--) {                              // p_M is the fastest axis of the brick
      const int ap = M + s, n = op.n[ap], st = (int)op.st[ap];
      const int i = r % n;
      r /= n;
      const double fp1 = (i + 1 < n) ? kb[c + st] : 0.0, fm1 = (i >= 1) ? kb[c - st] : 0.0;
      double d = op.c1[ap] * (fp1 - fm1);
      if (wide) {
        const double fp2 = (i + 2 < n) ? kb[c + 2 * st] : 0.0, fm2 = (i >= 2) ? kb[c - 2 * st] : 0.0;
        d = fma(op.c2[ap], fp2 - fm2, d);
      }
      acc = fma(g[s], fma(op.kup[s] * (op.x0[ap] + i * op.h[ap]), xc, d), acc);
    }
    X[c] = acc;
  }
}

// The same with 128-bit shared accesses (even fastest momentum axis): a thread owns a pair of cells adjacent along
// the fastest axis and marches along p_1 with a five-deep register window, so a pair costs 1 + 2 (+ 4 for M = 3)
// LDS.128 instead of 2 x 13 LDS.64, and no index division per cell.
template <int M>
__global__ void __launch_bounds__(256) k_kick_brick_pairs(DevOp op, DevObs ob, double* x, size_t slot_stride) {
  extern __shared__ __align__(16) double kb[];
  const long long ql = blockIdx.x;
  const int k = blockIdx.y;
  const int pb = (int)op.pb;
  double* X = x + (size_t)blockIdx.z * slot_stride + (size_t)k * op.cells + (size_t)ql * pb;
  for (int i = threadIdx.x; i < pb / 2; i += 256)
    reinterpret_cast<double2*>(kb)[i] = __ldcs(reinterpret_cast<const double2*>(X) + i);
  int iq[M];
  {
    long long r = ql;
#pragma unroll
    for (int s = M - 1; s >= 0; s--) { iq[s] = (int)(r % op.n[s]); r /= op.n[s]; }
  }
  double g[M];                                                      // dX/dq_s at this q-point, Eq. (13)-(14), (18)
#pragma unroll
  for (int s = 0; s < M; s++) {
    g[s] = ob.lin_q[s];
#pragma unroll
    for (int r = 0; r < M; r++) g[s] = fma(0.5 * (ob.quad[s][r] + ob.quad[r][s]), op.x0[r] + iq[r] * op.h[r], g[s]);
  }
  const bool wide = (op.scheme == CHFPE_CENTRAL4);
  const int n1 = op.n[M], nf = op.n[2 * M - 1], nm = (M == 3) ? op.n[M + 1] : 1;   // slowest, fastest, middle momentum axis
  const int plane = nm * nf, plane2 = plane / 2, nf2 = nf / 2;
  const int af = 2 * M - 1, am = M + 1;
  const double c1a = op.c1[M] * g[0], c2a = wide ? op.c2[M] * g[0] : 0.0;            // p_1
  const double c1f = op.c1[af] * g[M - 1], c2f = wide ? op.c2[af] * g[M - 1] : 0.0;  // fastest axis
  const double c1m = (M == 3) ? op.c1[am] * g[1] : 0.0, c2m = (M == 3 && wide) ? op.c2[am] * g[1] : 0.0;
  __syncthreads();
  const double2* K2 = reinterpret_cast<const double2*>(kb);
  double2* X2 = reinterpret_cast<double2*>(X);
  const double2 z = make_double2(0.0, 0.0);
  for (int pos = threadIdx.x; pos < plane2; pos += 256) {
    const int im = pos / nf2, jf = pos - im * nf2;                  // middle index, pair index along the fastest axis
    const double pfa = op.x0[af] + (2 * jf) * op.h[af], pfb = pfa + op.h[af];
    // pointwise part kappa^up (g_f p_f + g_m p_m) x, and g_1 kappa^up p_1 x per plane
    double ka = g[M - 1] * op.kup[M - 1] * pfa, kbb = g[M - 1] * op.kup[M - 1] * pfb;
    if (M == 3) { const double pm = g[1] * op.kup[1] * (op.x0[am] + im * op.h[am]); ka += pm; kbb += pm; }
    double2 w0 = z, w1 = z, w2 = K2[pos], w3 = (n1 > 1) ? K2[plane2 + pos] : z, w4;   // planes i1-2 .. i1+2
    for (int i1 = 0; i1 < n1; i1++) {
      w4 = (i1 + 2 < n1) ? K2[(i1 + 2) * plane2 + pos] : z;
      const int c = i1 * plane2 + pos;
      const double p1k = g[0] * op.kup[0] * (op.x0[M] + i1 * op.h[M]);
      double ax = fma(c2a, w4.x - w0.x, c1a * (w3.x - w1.x)) + (ka + p1k) * w2.x;
      double ay = fma(c2a, w4.y - w0.y, c1a * (w3.y - w1.y)) + (kbb + p1k) * w2.y;
      {                                                             // fastest axis: pairs to the left and right
        const double2 l = (jf >= 1) ? K2[c - 1] : z, r = (jf + 1 < nf2) ? K2[c + 1] : z;
        // cells (a, b) = (2 jf, 2 jf + 1): neighbours of a: l.y | b ; of b: a | r.x ; second neighbours: l.x | r.x ; l.y | r.y
        ax = fma(c1f, w2.y - l.y, ax); ay = fma(c1f, r.x - w2.x, ay);
        ax = fma(c2f, r.x - l.x, ax);  ay = fma(c2f, r.y - l.y, ay);
      }
      if (M == 3) {
        const double2 u1 = (im + 1 < nm) ? K2[c + nf2] : z, d1 = (im >= 1) ? K2[c - nf2] : z;
        ax = fma(c1m, u1.x - d1.x, ax); ay = fma(c1m, u1.y - d1.y, ay);
        if (wide) {
          const double2 u2 = (im + 2 < nm) ? K2[c + 2 * nf2] : z, d2 = (im >= 2) ? K2[c - 2 * nf2] : z;
          ax = fma(c2m, u2.x - d2.x, ax); ay = fma(c2m, u2.y - d2.y, ay);
        }
      }
      __stcs(X2 + c, make_double2(ax, ay));
      w0 = w1; w1 = w2; w2 = w3; w3 = w4;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Deterministic reductions: per-block partials (warp shuffle -> shared) then a fixed-order final pass.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double block_sum_256(double v) {
  __shared__ double sm[8];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
  __syncthreads();
  double r = 0.0;
  if (threadIdx.x < 32) {
    r = (threadIdx.x < 8) ? sm[threadIdx.x] : 0.0;
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) r += __shfl_down_sync(0xffffffffu, r, o);
  }
  __syncthreads();
  return r;   // valid in thread 0
}

// O(q,p) * w(q,p) at one cell: observable polynomial Eq. (13)-(14) times the gauge weight (1 or phi = e^{-beta H/2})
template <int M>
__device__ __forceinline__ double expect_weight(const DevOp& op, const DevObs& ob, long long cell) {
  int idx[2 * M];
  decode<2 * M>(op, cell, idx);
  double O = ob.c0, w = 1.0;
  double q[M];
#pragma unroll
  for (int s = 0; s < M; s++) q[s] = op.x0[s] + idx[s] * op.h[s];
#pragma unroll
  for (int s = 0; s < M; s++) {
    const double p = op.x0[M + s] + idx[M + s] * op.h[M + s];
    O = fma(ob.lin_q[s], q[s], O);
    O = fma(ob.lin_p[s], p, O);
#pragma unroll
    for (int r = 0; r < M; r++) O = fma(0.5 * ob.quad[s][r] * q[s], q[r], O);
    if (op.gauge == CHFPE_GAUGE_SQRT_EQ) w *= __ldg(op.ep[s] + idx[M + s]);
  }
  if (op.gauge == CHFPE_GAUGE_SQRT_EQ) w *= __ldg(op.eU + qlinear(op, cell));
  return O * w;
}

template <int M>
__global__ void __launch_bounds__(256) k_reduce_partial(DevOp op, DevObs ob, int mode, const double* __restrict__ x,
                                                        long long elem_off, long long ncells, size_t slot_stride,
                                                        double* __restrict__ partial) {
  const double* X = x + (size_t)blockIdx.y * slot_stride + elem_off;
  // contiguous chunk per block so that the summation order is fixed by (ncells, gridDim.x) alone
  const long long per = (ncells + gridDim.x - 1) / gridDim.x;
  const long long lo = (long long)blockIdx.x * per;
  long long hi = lo + per; if (hi > ncells) hi = ncells;
  double acc = 0.0;
  for (long long c = lo + threadIdx.x; c < hi; c += 256) {
    const double v = X[c];
    if (mode == RED_SUMSQ) { acc = fma(v, v, acc); continue; }
    if (mode == RED_SUM) { acc += v; continue; }
    acc = fma(expect_weight<M>(op, ob, c), v, acc);   // RED_EXPECT: ncells == op.cells
  }
  const double r = block_sum_256(acc);
  if (threadIdx.x == 0) partial[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = r;
}

// <O> on the p-brick layout (RED_EXPECT only; p-bricks of up to EXPECT_MAXPB cells).  The observable of Eq. (13)-(14) is
// O(q, p) = A(q) + sum_s lin_p[s] p_s and the gauge weight factorises as eU(q) * prod_s ep_s(p_s), so a CTA tabulates the
// momentum factors of one brick once in shared memory -- wp[c] = prod_s ep_s, lp[c] = sum_s lin_p[s] p_s -- and then
// streams its contiguous run of bricks: per cell one coalesced load, two shared loads and two FMAs instead of a full
// index decode (six divisions) and four table loads.  Summation order: fixed by (nqc, gridDim.x, 256) alone.
constexpr int EXPECT_MAXPB = 8192;
template <int M>
__global__ void __launch_bounds__(256) k_expect_pbrick(DevOp op, DevObs ob, const double* __restrict__ x, long long elem_off,
                                                       size_t slot_stride, double* __restrict__ partial) {
  extern __shared__ double ex_tab[];                  // wp[pb], lp[pb]
  const int pb = (int)op.pb;
  double* wp = ex_tab;
  double* lp = ex_tab + pb;
  for (int c = threadIdx.x; c < pb; c += 256) {
    unsigned r = (unsigned)c;
    double w = 1.0, l = 0.0;
#pragma unroll
    for (int s = M - 1; s >= 0; s--) {
      const unsigned q = r / (unsigned)op.n[M + s];
      const int i = (int)(r - q * (unsigned)op.n[M + s]);
      r = q;
      l = fma(ob.lin_p[s], op.x0[M + s] + i * op.h[M + s], l);
      if (op.gauge == CHFPE_GAUGE_SQRT_EQ) w *= __ldg(op.ep[s] + i);
    }
    wp[c] = w; lp[c] = l;
  }
  __syncthreads();
  const double* X = x + (size_t)blockIdx.y * slot_stride + elem_off;
  const long long per = (op.nqc + gridDim.x - 1) / gridDim.x;
  const long long lo = (long long)blockIdx.x * per;
  long long hi = lo + per; if (hi > op.nqc) hi = op.nqc;
  double acc = 0.0;
  for (long long qi = lo; qi < hi; qi++) {
    unsigned r = (unsigned)qi;
    double q[M];
#pragma unroll
    for (int s = M - 1; s >= 0; s--) {
      const unsigned d = r / (unsigned)op.n[s];
      q[s] = op.x0[s] + (int)(r - d * (unsigned)op.n[s]) * op.h[s];
      r = d;
    }
    double A = ob.c0;
#pragma unroll
    for (int s = 0; s < M; s++) {
      A = fma(ob.lin_q[s], q[s], A);
#pragma unroll
      for (int t = 0; t < M; t++) A = fma(0.5 * ob.quad[s][t] * q[s], q[t], A);
    }
    const double e = (op.gauge == CHFPE_GAUGE_SQRT_EQ) ? __ldg(op.eU + qi) : 1.0;
    const double* B = X + qi * pb;
    double a = 0.0;
    for (int c = threadIdx.x; c < pb; c += 256) a = fma((A + lp[c]) * wp[c], B[c], a);
    acc = fma(e, a, acc);
  }
  const double r = block_sum_256(acc);
  if (threadIdx.x == 0) partial[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = r;
}

__global__ void __launch_bounds__(256) k_reduce_final(const double* __restrict__ partial, int nblocks, double scale,
                                                      double* __restrict__ results, long long res_stride) {
  const double* P = partial + (size_t)blockIdx.x * nblocks;
  double acc = 0.0;
  for (int i = threadIdx.x; i < nblocks; i += 256) acc += P[i];
  const double r = block_sum_256(acc);
  if (threadIdx.x == 0) results[(long long)blockIdx.x * res_stride] = r * scale;
}

// element 0 <- exp factor tables product (phi or e^{-beta H}), others <- 0
template <int M>
__global__ void __launch_bounds__(256) k_init_eq(DevOp op, double* __restrict__ x) {
  long long cell = (long long)blockIdx.x * 256 + threadIdx.x;
  if (cell >= op.cells) return;
  const int k = blockIdx.y;
  double v = 0.0;
  if (k == 0) {
    int idx[2 * M];
    decode<2 * M>(op, cell, idx);
    v = __ldg(op.eU + qlinear(op, cell));
#pragma unroll
    for (int s = 0; s < M; s++) v *= __ldg(op.ep[s] + idx[M + s]);
  }
  x[(size_t)k * op.cells + cell] = v;
}

__global__ void __launch_bounds__(256) k_scale(double* __restrict__ x, long long n, const double* __restrict__ denom,
                                               double mult) {
  const double f = mult / denom[0];
  for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < n; i += (long long)gridDim.x * 256) x[i] *= f;
}

template <int M>
__global__ void __launch_bounds__(256) k_permute(DevOp op, const double* __restrict__ src, double* __restrict__ dst,
                                                 int to_internal) {
  long long cell = (long long)blockIdx.x * 256 + threadIdx.x;
  if (cell >= op.cells) return;
  int idx[2 * M];
  decode<2 * M>(op, cell, idx);
  long long canon = 0;                       // canonical order q1,p1,...,qM,pM, last fastest
#pragma unroll
  for (int s = 0; s < M; s++) {
    canon = canon * op.n[s] + idx[s];
    canon = canon * op.n[M + s] + idx[M + s];
  }
  const size_t e = (size_t)blockIdx.y * op.cells;
  if (to_internal) dst[e + cell] = src[e + canon];
  else dst[e + canon] = src[e + cell];
}

// ------------------------------------------------------------------------------------------------
// Persistent multi-step kernel for states that live in L2 (configs 1-2 and small grids): all four RK stages of
// `stride` steps and, optionally, one expectation sample per `stride` steps in ONE cooperative launch; stages are
// separated by grid-wide barriers instead of kernel boundaries (6 launches of ~9 us per step otherwise).
// ------------------------------------------------------------------------------------------------
template <int M>
__device__ __forceinline__ void coop_stage(const DevOp& op, const double* in, const double* y, double* out, double c,
                                           long long total) {
  for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < total; v += (long long)gridDim.x * blockDim.x) {
    const int k = (int)(v / op.cells);
    const long long cell = v - (long long)k * op.cells;
    const double acc = rhs_value<M, true>(op, in, k, cell);
    out[v] = fma(c, acc, __ldcg(y + v));
  }
}

template <int M>
__global__ void __launch_bounds__(256) k_steps_coop(DevOp op, DevObs ob, double* y, double* va, double* vb, double dt,
                                                    long long n_samples, long long stride, int do_expect,
                                                    double* partial, double* results) {
  namespace cg = cooperative_groups;
  cg::grid_group grid = cg::this_grid();
  const long long total = (long long)op.K * op.cells;
  for (long long smp = 0; smp < n_samples; smp++) {
    for (long long st = 0; st < stride; st++) {                    // Horner form of RK4 (R13)
      coop_stage<M>(op, y, y, va, dt / 4.0, total);  grid.sync();
      coop_stage<M>(op, va, y, vb, dt / 3.0, total); grid.sync();
      coop_stage<M>(op, vb, y, va, dt / 2.0, total); grid.sync();
      coop_stage<M>(op, va, y, y, dt, total);        grid.sync();
    }
    if (do_expect) {                                               // <O> on element 0, fixed summation order
      const long long per = (op.cells + gridDim.x - 1) / gridDim.x;
      const long long lo = (long long)blockIdx.x * per;
      long long hi = lo + per; if (hi > op.cells) hi = op.cells;
      double acc = 0.0;
      for (long long c = lo + threadIdx.x; c < hi; c += 256) acc = fma(expect_weight<M>(op, ob, c), __ldcg(y + c), acc);
      const double r = block_sum_256(acc);
      if (threadIdx.x == 0) partial[blockIdx.x] = r;
      grid.sync();
      if (blockIdx.x == 0) {
        double a2 = 0.0;
        for (int i = threadIdx.x; i < (int)gridDim.x; i += 256) a2 += __ldcg(partial + i);
        const double r2 = block_sum_256(a2);
        if (threadIdx.x == 0) results[smp] = r2 * op.dV;
      }
      if (stride == 0) grid.sync();                                // no stage barrier follows: block 0 must be done with `partial`
    }
  }
}

}  // namespace

#define DISPATCH_M(M, CALL)            \
  do {                                 \
    if ((M) == 1) { CALL(1); }         \
    else if ((M) == 2) { CALL(2); }    \
    else { CALL(3); }                  \
  } while (0)

int launch_stage(const DevOp& op, const double* in, const double* y, double* out, double a, double c, int nb,
                 size_t slot_stride, cudaStream_t s) {
  dim3 grid((unsigned)((op.cells + 255) / 256), op.K, nb);
#define CALL(MM) k_stage_generic<MM><<<grid, 256, 0, s>>>(op, in, y, out, a, c, slot_stride)
  DISPATCH_M(op.M, CALL);
#undef CALL
  return 1;
}

// in-place kick on the brick layout; returns 0 (nothing launched) where it does not apply
int launch_kick_brick(const DevOp& op, const DevObs& o, double* x, int nb, size_t slot_stride, cudaStream_t s) {
  const size_t smem = sizeof(double) * (size_t)op.pb;
  if (op.M < 2 || op.scheme == CHFPE_COMPACT6 || smem > 200 * 1024 || op.nqc > 0x7fffffffLL) return 0;
  static bool optin[4] = {false, false, false, false};
  if (!optin[op.M]) {
    if (op.M == 2) cudaFuncSetAttribute(k_kick_brick<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    else cudaFuncSetAttribute(k_kick_brick<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    optin[op.M] = true;
  }
  dim3 grid((unsigned)op.nqc, op.K, nb);
  if (op.n[2 * op.M - 1] % 2 == 0 && ((op.cells * sizeof(double)) % 16) == 0 && (slot_stride % 2) == 0) {   // 128-bit pairs
    if (!optin[op.M - 2]) {
      if (op.M == 2) cudaFuncSetAttribute(k_kick_brick_pairs<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
      else cudaFuncSetAttribute(k_kick_brick_pairs<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
      optin[op.M - 2] = true;
    }
    if (op.M == 2) k_kick_brick_pairs<2><<<grid, 256, smem, s>>>(op, o, x, slot_stride);
    else k_kick_brick_pairs<3><<<grid, 256, smem, s>>>(op, o, x, slot_stride);
    return 1;
  }
  if (op.M == 2) k_kick_brick<2><<<grid, 256, smem, s>>>(op, o, x, slot_stride);
  else k_kick_brick<3><<<grid, 256, smem, s>>>(op, o, x, slot_stride);
  return 1;
}

int launch_terminator_add(const DevOp& op, const double* in, double* out, double c, int nb, size_t slot_stride,
                          cudaStream_t s) {
  dim3 grid((unsigned)((op.cells + 255) / 256), op.K, nb);
#define CALL(MM) k_terminator_add<MM><<<grid, 256, 0, s>>>(op, in, out, c, slot_stride)
  DISPATCH_M(op.M, CALL);
#undef CALL
  return 1;
}

int launch_kick(const DevOp& op, const DevObs& o, const double* in, double* out, int nb, size_t slot_stride,
                cudaStream_t s) {
  dim3 grid((unsigned)((op.cells + 255) / 256), op.K, nb);
#define CALL(MM) k_kick_generic<MM><<<grid, 256, 0, s>>>(op, o, in, out, slot_stride)
  DISPATCH_M(op.M, CALL);
#undef CALL
  return 1;
}

int launch_reduce(const DevOp& op, const DevObs& o, int mode, const double* x, int k, long long ncells, int nb,
                  size_t slot_stride, double scale, double* partial, int red_blocks, double* results,
                  long long res_stride, cudaStream_t s) {
  dim3 grid(red_blocks, nb);
  const long long off = (long long)k * op.cells;
  if (mode == RED_EXPECT && ncells == op.cells && op.pb <= EXPECT_MAXPB && op.pb >= 256 && op.expect_pbrick) {
    const size_t sm = 2 * sizeof(double) * (size_t)op.pb;
    cudaError_t e = cudaSuccess;
    if (sm > 48 * 1024) {
      switch (op.M) {
        case 1: e = cudaFuncSetAttribute(k_expect_pbrick<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm); break;
        case 2: e = cudaFuncSetAttribute(k_expect_pbrick<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm); break;
        default: e = cudaFuncSetAttribute(k_expect_pbrick<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm); break;
      }
    }
    if (e == cudaSuccess) {
#define CALL(MM) k_expect_pbrick<MM><<<grid, 256, sm, s>>>(op, o, x, off, slot_stride, partial)
      DISPATCH_M(op.M, CALL);
#undef CALL
      k_reduce_final<<<nb, 256, 0, s>>>(partial, red_blocks, scale, results, res_stride);
      return 2;
    }
    cudaGetLastError();
  }
#define CALL(MM) k_reduce_partial<MM><<<grid, 256, 0, s>>>(op, o, mode, x, off, ncells, slot_stride, partial)
  DISPATCH_M(op.M, CALL);
#undef CALL
  k_reduce_final<<<nb, 256, 0, s>>>(partial, red_blocks, scale, results, res_stride);
  return 2;
}

int launch_init_eq(const DevOp& op, double* x, cudaStream_t s) {
  dim3 grid((unsigned)((op.cells + 255) / 256), op.K);
#define CALL(MM) k_init_eq<MM><<<grid, 256, 0, s>>>(op, x)
  DISPATCH_M(op.M, CALL);
#undef CALL
  return 1;
}

int launch_scale(double* x, long long n, const double* denom_dev, double mult, cudaStream_t s) {
  long long blocks = (n + 255) / 256;
  if (blocks > 148 * 16) blocks = 148 * 16;
  k_scale<<<(unsigned)blocks, 256, 0, s>>>(x, n, denom_dev, mult);
  return 1;
}

int launch_permute(const DevOp& op, const double* src, double* dst, int to_internal, cudaStream_t s) {
  dim3 grid((unsigned)((op.cells + 255) / 256), op.K);
#define CALL(MM) k_permute<MM><<<grid, 256, 0, s>>>(op, src, dst, to_internal)
  DISPATCH_M(op.M, CALL);
#undef CALL
  return 1;
}

// n_samples x (stride RK4 steps [+ one expectation sample]) on ONE replica in one cooperative launch.  Returns the
// number of launches (1) or 0 when the device cannot co-schedule the grid (the caller then uses per-stage launches).
int launch_steps_coop(const DevOp& op, const DevObs& o, double* y, double* va, double* vb, double dt,
                      long long n_samples, long long stride, int do_expect, double* partial, int max_blocks,
                      double* results, cudaStream_t s) {
  int dev = 0, coop = 0, sms = 0, per_sm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return 0;
  cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (!coop) return 0;
  const void* fn = nullptr;
  if (op.M == 1) fn = (const void*)k_steps_coop<1>;
  else if (op.M == 2) fn = (const void*)k_steps_coop<2>;
  else fn = (const void*)k_steps_coop<3>;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, 256, 0) != cudaSuccess || per_sm < 1) return 0;
  if (per_sm > 8) per_sm = 8;
  const long long total = (long long)op.K * op.cells;
  long long blocks = (total + 255) / 256;
  if (blocks > (long long)sms * per_sm) blocks = (long long)sms * per_sm;
  if (blocks > max_blocks) blocks = max_blocks;                    // one partial sum per block: `partial` holds max_blocks
  DevOp opv = op; DevObs ov = o;
  void* args[] = {&opv, &ov, &y, &va, &vb, &dt, &n_samples, &stride, &do_expect, &partial, &results};
  if (cudaLaunchCooperativeKernel(fn, dim3((unsigned)blocks), dim3(256), args, 0, s) != cudaSuccess) {
    cudaGetLastError();
    return 0;
  }
  return 1;
}
