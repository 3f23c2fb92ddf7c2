// COMPACT6 derivative path (step a9 of DESIGN.md): the sixth-order Pade scheme of PAPER.md Eq. (25)-(31) :177-201,
//     (1/3) d_{i-1} + d_i + (1/3) d_{i+1} = [ a (f_{i+1} - f_{i-1}) + b (f_{i+2} - f_{i-2}) ] / h,
// a = 7/9, b = 1/36 (reading R4: the printed a = 7/18 is not consistent), matrices truncated as printed in
// Eq. (28)-(29) (zero ghosts, R9).  The tridiagonal systems are solved per grid line by the Thomas recurrence with the
// elimination factors of the constant matrix tridiag(1/3, 1, 1/3) tabulated once per axis on the host; the paper's own
// choice for this step is parallel cyclic reduction on Ampere-class GPUs (section III.C :203-207) -- at line lengths
// of 16..128 one thread per line is enough to occupy the GPU (a 16^6 grid has 10^6 lines per element and axis).
//
// This is the conditional path of SURVEY.md 8(a9); the explicit CENTRAL4 scheme is the performance path.  A stage is
// 2M line passes, each ONE launch over all elements and replica slots (grid.y, grid.z):
//   q_s pass: d = A^{-1} B X_k along q_s, accumulated as  out (+)= c * (-(p_s/m_s)) d
//   p_s pass: d = A^{-1} B G_s along p_s with G_s = (dU/dq_s) X_k + V'_s X_up + n_s c_s V'_s X_dn formed on the fly
//             (its coefficients are constant along a p-line),  out += c * d; the pass has X_up and X_dn in hand, so
//             it also adds the pointwise gauge terms c * p_s V'_s (kup_s X_up + n_s c_s kdn_s X_dn) of its mode, and
//             the last one the damping -c * Gamma_k X_k
// The first pass writes out = a*y + c*(...), so no right-hand-side array exists; the forward-elimination values of a
// line stay in thread-local memory for lines of up to 128 points (all BASELINE configs), longer lines keep
// them in an element-sized scratch array and run element by element.  (First version: whole-array derivatives,
// 17 launches per element, 37.4 ms per stage at config 4.)
#include <cstdlib>
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
// bet[i], cfac[i]: RECIPROCAL pivots and elimination factors of tridiag(1/3,1,1/3) with n rows (host-tabulated per
// axis; multiplying by the tabulated reciprocal replaces a division per point: q passes 2.33 -> see DESIGN.md).
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
    prev = (i == 0) ? r * __ldg(bet) : (r - al * prev) * __ldg(bet + i);   // bet[]: reciprocal pivots
    d[base + (long long)i * st] = prev;
    fm2 = fm1; fm1 = f0; f0 = fp1; fp1 = fp2;
  }
  double next = prev;                                              // back substitution
  for (int i = n - 2; i >= 0; i--) {
    next = d[base + (long long)i * st] - __ldg(cfac + i + 1) * next;
    d[base + (long long)i * st] = next;
  }
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

constexpr int CLINE_MAX = 128;    // longest line whose elimination values stay in thread-local memory

// One Pade line solve per thread, fused with the formation of its operand and with the accumulation into `out`.
// PAXIS = 0: line along q_s of X_k; PAXIS = 1: line along p_s of G_s.  grid = (line blocks, elements, slots).
// NF = 0: run-time length <= CLINE_MAX, elimination values in a thread-local array; NF = -1: element-sized scratch D.
// (NF > 0, a compile-time length with the values in registers, was measured slower at 16 points: 30.4 vs 22.5 ms
// per stage at config 4 -- 100 registers per thread leave too few warps to hide the line's dependent loads.)
template <int M, int PAXIS, int NF>
__global__ void __launch_bounds__(128) k_compact_line(DevOp op, const double* __restrict__ in, const double* y, double* out,
                                                      double a, double c, int s, int first, int k0, int b0,
                                                      size_t slot_stride, const double* __restrict__ bet,
                                                      const double* __restrict__ cfac, double* __restrict__ D) {
  const int axis = PAXIS ? M + s : s;
  constexpr bool LOCAL = NF >= 0;
  const int n = NF > 0 ? NF : op.n[axis];
  const long long st = op.st[axis];
  const long long line = (long long)blockIdx.x * 128 + threadIdx.x;
  if (line >= op.cells / n) return;
  const int k = k0 + blockIdx.y;
  const size_t eoff = (size_t)(b0 + blockIdx.z) * slot_stride + (size_t)k * op.cells;
  const long long outer = line / st, inner = line - outer * st;
  const long long base = outer * st * n + inner;                   // cell of point 0 of the line
  int idx[2 * M];
  cdecode<2 * M>(op, (unsigned)base, idx);
  const double* Xk = in + eoff + base;
  const double* Xu = Xk;
  const double* Xd = Xk;
  double ck = 1.0, cu = 0.0, cd = 0.0, coef = 1.0, gam = 0.0;
  if (PAXIS) {                                                     // G_s: coefficients depend on q only
    const long long ql = base / op.pb;
    const double q = op.x0[s] + idx[s] * op.h[s];
    const double Vp = fma(op.VSL[s], q, op.VLL[s]);
    ck = __ldg(op.dU[s] + ql);
    const int ku = __ldg(op.up + 3 * k + s), kd = __ldg(op.dn + 3 * k + s);
    if (ku >= 0) { cu = Vp; Xu = Xk + ((long long)ku - k) * op.cells; }
    if (kd >= 0) { cd = __ldg(op.nvec + 3 * k + s) * op.cdn[s] * Vp; Xd = Xk + ((long long)kd - k) * op.cells; }
    if (s == M - 1) gam = __ldg(op.Gamma + k);                     // the damping term rides on the last p pass
  } else {
    coef = -(op.x0[M + s] + idx[M + s] * op.h[M + s]) * op.inv_mass[s];
  }
  auto f = [&](int i) -> double {
    const long long o = (long long)i * st;
    double v = PAXIS ? ck * Xk[o] : Xk[o];
    if (PAXIS) { if (cu != 0.0) v = fma(cu, Xu[o], v); if (cd != 0.0) v = fma(cd, Xd[o], v); }
    return v;
  };
  double rl[NF > 0 ? NF : (NF == 0 ? CLINE_MAX : 1)];
  double* rg = D + base;                                           // element-sized scratch (LOCAL == false)
  const double al = 1.0 / 3.0, ca = 7.0 / 9.0, cb = 1.0 / 36.0, inv_h = 1.0 / op.h[axis];
  double fm2 = 0.0, fm1 = 0.0, f0 = f(0), fp1 = (n > 1) ? f(1) : 0.0, prev = 0.0;
#pragma unroll
  for (int i = 0; i < n; i++) {                                    // forward elimination
    const double fp2 = (i + 2 < n) ? f(i + 2) : 0.0;
    const double r = (ca * (fp1 - fm1) + cb * (fp2 - fm2)) * inv_h;
    prev = (i == 0) ? r * __ldg(bet) : (r - al * prev) * __ldg(bet + i);   // bet[]: reciprocal pivots
    if (LOCAL) rl[LOCAL ? i : 0] = prev; else rg[(long long)i * st] = prev;
    fm2 = fm1; fm1 = f0; f0 = fp1; fp1 = fp2;
  }
  const double cc = c * coef;
  const double* Y = y + eoff + base;
  double* O = out + eoff + base;
  double next = 0.0;
#pragma unroll
  for (int i = n - 1; i >= 0; i--) {                               // back substitution + accumulation
    const double ri = LOCAL ? rl[LOCAL ? i : 0] : rg[(long long)i * st];
    next = (i == n - 1) ? ri : ri - __ldg(cfac + i + 1) * next;
    const long long o = (long long)i * st;
    double t = cc * next;
    if (PAXIS) {                                                   // pointwise terms of mode s (gauge) and the damping
      const double p = op.x0[M + s] + i * op.h[M + s];
      double pw = 0.0;
      if (cu != 0.0) pw = op.kup[s] * cu * Xu[o];
      if (cd != 0.0) pw = fma(op.kdn[s] * cd, Xd[o], pw);
      pw *= p;
      if (s == M - 1) pw = fma(-gam, Xk[o], pw);
      t = fma(c, pw, t);
    }
    O[o] = first ? fma(a, Y[o], t) : O[o] + t;
  }
}

// q_2 and q_3 passes of three modes in ONE launch: a CTA owns the whole (q_2, q_3) plane of NQ x NQ points for PC
// consecutive momentum cells of one (element, q_1) -- PC * 8 bytes contiguous per q-point, so every global access is a
// full 128-byte run.  The plane goes into a shared tile X once (instead of once per axis); NQ * PC threads then take one
// q_3 line each (Thomas recurrence as in k_compact_line, operand from shared memory, forward values in registers) and
// leave coef_3 d_3 in a second tile A, take one q_2 line each from the same X and add coef_2 d_2 to their cells of A, and
// the tile is added to `out` in one coalesced read-modify-write (instead of one per axis): 8.05 GB of compulsory traffic
// for both axes at config 4 against 2 x 9.3 GB measured for the two line passes.
template <int NQ, int PC>
__global__ void __launch_bounds__(NQ * PC, (NQ * NQ * PC * 16 <= 72 * 1024) ? 3 : 2) k_compact_qplane(
    DevOp op, const double* __restrict__ in, const double* y, double* out, double a, double c, int first, size_t slot_stride,
    const double* __restrict__ ib2, const double* __restrict__ cf2, const double* __restrict__ ib3, const double* __restrict__ cf3) {
  extern __shared__ double qp_s[];
  constexpr int NT = NQ * PC, PTS = NQ * NQ, TILE = PTS * PC;
  double* X = qp_s;
  double* A = qp_s + TILE;
  const int t = threadIdx.x;
  const int pb = (int)op.pb, nch = pb / PC;
  const int chunk = blockIdx.x % nch;
  const int kq = blockIdx.x / nch;                                   // (element, q_1 index)
  const int iq1 = kq % op.n[0], k = kq / op.n[0];
  const size_t eoff = (size_t)blockIdx.z * slot_stride + (size_t)k * op.cells + (size_t)iq1 * PTS * pb + (size_t)chunk * PC;
  const double* Xg = in + eoff;
  {                                                                  // NQ loads per thread, all in flight before the first use
    double v[NQ];
#pragma unroll
    for (int j = 0; j < NQ; j++) { const int i = t + j * NT; v[j] = __ldg(Xg + (size_t)(i / PC) * pb + (i % PC)); }
    if ((t & 15) == 0) {                                             // the lines of the final read-modify-write: ask L2 now
      const double* Pg = (first ? y : out) + eoff;
#pragma unroll
      for (int j = 0; j < NQ; j++) { const int i = t + j * NT; asm volatile("prefetch.global.L2 [%0];" ::"l"(Pg + (size_t)(i / PC) * pb + (i % PC))); }
    }
#pragma unroll
    for (int j = 0; j < NQ; j++) X[t + j * NT] = v[j];
  }
  __syncthreads();
  const int line = t / PC, pc = t - line * PC;
  double coef2, coef3;
  {
    int r = chunk * PC + pc;
    const int i3 = r % op.n[5]; r /= op.n[5];
    const int i2 = r % op.n[4];
    coef2 = -(op.x0[4] + i2 * op.h[4]) * op.inv_mass[1];
    coef3 = -(op.x0[5] + i3 * op.h[5]) * op.inv_mass[2];
  }
  const double al = 1.0 / 3.0, ca = 7.0 / 9.0, cb = 1.0 / 36.0;
  auto solve = [&](const int base, const int st, const double inv_h, const double* __restrict__ ib, const double* __restrict__ cf,
                   double (&d)[NQ]) {                                // d <- A^{-1} B f / h along the line X[base + i * st]
    double fm2 = 0.0, fm1 = 0.0, f0 = X[base], fp1 = X[base + st], prev = 0.0;
#pragma unroll
    for (int i = 0; i < NQ; i++) {
      const double fp2 = (i + 2 < NQ) ? X[base + (i + 2) * st] : 0.0;
      const double r = (ca * ((i + 1 < NQ ? fp1 : 0.0) - fm1) + cb * (fp2 - fm2)) * inv_h;
      prev = (i == 0) ? r * __ldg(ib) : (r - al * prev) * __ldg(ib + i);
      d[i] = prev;
      fm2 = fm1; fm1 = f0; f0 = fp1; fp1 = fp2;
    }
#pragma unroll
    for (int i = NQ - 2; i >= 0; i--) d[i] = d[i] - __ldg(cf + i + 1) * d[i + 1];
  };
  {
    double d[NQ];                                                    // q_3 line (q_2 = line): points line * NQ + i
    solve(line * NQ * PC + pc, PC, 1.0 / op.h[2], ib3, cf3, d);
#pragma unroll
    for (int i = 0; i < NQ; i++) A[(line * NQ + i) * PC + pc] = coef3 * d[i];
  }
  __syncthreads();
  {
    double d[NQ];                                                    // q_2 line (q_3 = line): points i * NQ + line
    solve(line * PC + pc, NQ * PC, 1.0 / op.h[1], ib2, cf2, d);
#pragma unroll
    for (int i = 0; i < NQ; i++) A[(i * NQ + line) * PC + pc] += coef2 * d[i];
  }
  __syncthreads();
  const double* Yg = y + eoff;
  double* Og = out + eoff;
  {
    double v[NQ];
#pragma unroll
    for (int j = 0; j < NQ; j++) {
      const int i = t + j * NT;
      const size_t g = (size_t)(i / PC) * pb + (i % PC);
      v[j] = first ? Yg[g] : Og[g];
    }
#pragma unroll
    for (int j = 0; j < NQ; j++) {
      const int i = t + j * NT;
      const size_t g = (size_t)(i / PC) * pb + (i % PC);
      Og[g] = first ? fma(a, v[j], c * A[i]) : v[j] + c * A[i];
    }
  }
}

// One q-line of compile-time length NQ per thread (q axes only): all NQ loads of the line are issued before the first use,
// the recurrence runs in registers, then all NQ loads of the output (or of y) are issued before the first store -- the
// memory-level parallelism of a thread is NQ instead of the one or two loads the generic kernel has in flight.
template <int M, int NQ>
__global__ void __launch_bounds__(128) k_compact_qline(DevOp op, const double* __restrict__ in, const double* y, double* out,
                                                       double a, double c, int s, int first, size_t slot_stride,
                                                       const double* __restrict__ ib, const double* __restrict__ cf) {
  const long long st = op.st[s];
  const long long line = (long long)blockIdx.x * 128 + threadIdx.x;
  if (line >= op.cells / NQ) return;
  const int k = blockIdx.y;
  const size_t eoff = (size_t)blockIdx.z * slot_stride + (size_t)k * op.cells;
  const long long outer = line / st, inner = line - outer * st;
  const long long base = outer * st * NQ + inner;
  int idx[2 * M];
  cdecode<2 * M>(op, (unsigned)base, idx);
  const double coef = -(op.x0[M + s] + idx[M + s] * op.h[M + s]) * op.inv_mass[s];
  const double* Xk = in + eoff + base;
  double f[NQ + 2];
#pragma unroll
  for (int i = 0; i < NQ; i++) f[i] = __ldg(Xk + (long long)i * st);
  f[NQ] = 0.0; f[NQ + 1] = 0.0;
  const double al = 1.0 / 3.0, ca = 7.0 / 9.0, cb = 1.0 / 36.0, inv_h = 1.0 / op.h[s];
  double d[NQ];
  double prev = 0.0;
#pragma unroll
  for (int i = 0; i < NQ; i++) {
    const double fm1 = (i >= 1) ? f[i - 1] : 0.0, fm2 = (i >= 2) ? f[i - 2] : 0.0;
    const double r = (ca * (f[i + 1] - fm1) + cb * (f[i + 2] - fm2)) * inv_h;
    prev = (i == 0) ? r * __ldg(ib) : (r - al * prev) * __ldg(ib + i);
    d[i] = prev;
  }
#pragma unroll
  for (int i = NQ - 2; i >= 0; i--) d[i] = d[i] - __ldg(cf + i + 1) * d[i + 1];
  const double cc = c * coef;
  const double* Y = y + eoff + base;
  double* O = out + eoff + base;
  double o[NQ];
#pragma unroll
  for (int i = 0; i < NQ; i++) o[i] = first ? Y[(long long)i * st] : O[(long long)i * st];
#pragma unroll
  for (int i = 0; i < NQ; i++) O[(long long)i * st] = first ? fma(a, o[i], cc * d[i]) : o[i] + cc * d[i];
}

// The same for long lines (NQ a multiple of 8, e.g. the 48-point axes of config 3): the operand streams through a window
// of three blocks of 8 points -- the block two ahead is requested before the current one is used -- while the NQ forward
// values stay in registers; the output is read-modify-written in blocks of 8 with the loads ahead of the stores.
template <int M, int NQ>
__global__ void __launch_bounds__(128) k_compact_qline_long(DevOp op, const double* __restrict__ in, const double* y, double* out,
                                                            double a, double c, int s, int first, size_t slot_stride,
                                                            const double* __restrict__ ib, const double* __restrict__ cf) {
  static_assert(NQ % 8 == 0 && NQ >= 24, "blocks of 8 points");
  constexpr int B = 8, NB = NQ / B;
  const long long st = op.st[s];
  const long long line = (long long)blockIdx.x * 128 + threadIdx.x;
  if (line >= op.cells / NQ) return;
  const int k = blockIdx.y;
  const size_t eoff = (size_t)blockIdx.z * slot_stride + (size_t)k * op.cells;
  const long long outer = line / st, inner = line - outer * st;
  const long long base = outer * st * NQ + inner;
  int idx[2 * M];
  cdecode<2 * M>(op, (unsigned)base, idx);
  const double coef = -(op.x0[M + s] + idx[M + s] * op.h[M + s]) * op.inv_mass[s];
  const double* Xk = in + eoff + base;
  const double al = 1.0 / 3.0, ca = 7.0 / 9.0, cb = 1.0 / 36.0, inv_h = 1.0 / op.h[s];
  double d[NQ];
  double cur[B], nxt[B], nn[B];
#pragma unroll
  for (int j = 0; j < B; j++) { cur[j] = __ldg(Xk + (long long)j * st); nxt[j] = __ldg(Xk + (long long)(B + j) * st); }
  double fm2 = 0.0, fm1 = 0.0, prev = 0.0;
#pragma unroll
  for (int b = 0; b < NB; b++) {
#pragma unroll
    for (int j = 0; j < B; j++) nn[j] = (b + 2 < NB) ? __ldg(Xk + (long long)((b + 2) * B + j) * st) : 0.0;
#pragma unroll
    for (int j = 0; j < B; j++) {
      const int i = b * B + j;
      const double fp1 = (j + 1 < B) ? cur[j + 1] : nxt[0];          // (nxt is zero past the end of the line)
      const double fp2 = (j + 2 < B) ? cur[j + 2] : nxt[j + 2 - B];
      const double r = (ca * (fp1 - fm1) + cb * (fp2 - fm2)) * inv_h;
      prev = (i == 0) ? r * __ldg(ib) : (r - al * prev) * __ldg(ib + i);
      d[i] = prev;
      fm2 = fm1; fm1 = cur[j];
    }
#pragma unroll
    for (int j = 0; j < B; j++) { cur[j] = nxt[j]; nxt[j] = nn[j]; }
  }
#pragma unroll
  for (int i = NQ - 2; i >= 0; i--) d[i] = d[i] - __ldg(cf + i + 1) * d[i + 1];
  const double cc = c * coef;
  const double* Y = y + eoff + base;
  double* O = out + eoff + base;
#pragma unroll
  for (int b = 0; b < NB; b++) {
    double o[B];
#pragma unroll
    for (int j = 0; j < B; j++) o[j] = first ? Y[(long long)(b * B + j) * st] : O[(long long)(b * B + j) * st];
#pragma unroll
    for (int j = 0; j < B; j++) O[(long long)(b * B + j) * st] = first ? fma(a, o[j], cc * d[b * B + j]) : o[j] + cc * d[b * B + j];
  }
}

// p_M pass (the contiguous axis): one thread per line would read 8 bytes per 128-byte line and request.  A warp
// therefore takes 32 consecutive lines (32 n contiguous doubles), loads them coalesced, forms G_M on the way and
// transposes through a padded shared tile [32][n+1]; every lane then runs the Thomas recurrence on its row in place,
// and the tile is written back coalesced.  Needs n <= 32 and cells % (32 n) == 0.
template <int M>
__global__ void __launch_bounds__(128) k_compact_pline_s1(DevOp op, const double* __restrict__ in, const double* y,
                                                          double* out, double a, double c, int first,
                                                          size_t slot_stride, const double* __restrict__ bet,
                                                          const double* __restrict__ cfac) {
  constexpr int s = M - 1, axis = 2 * M - 1;
  extern __shared__ double tiles[];
  const int n = op.n[axis], lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long line0 = ((long long)blockIdx.x * 4 + warp) * 32;
  if (line0 >= op.cells / n) return;
  double* tile = tiles + warp * 64 * (n + 1);                      // [32][n+1] G_M, then [32][n+1] pointwise terms
  double* ptile = tile + 32 * (n + 1);
  const int k = blockIdx.y;
  const size_t eoff = (size_t)blockIdx.z * slot_stride + (size_t)k * op.cells;
  const long long base = line0 * n;                                // first cell of the tile
  const double* Xk = in + eoff + base;
  const int ku = __ldg(op.up + 3 * k + s), kd = __ldg(op.dn + 3 * k + s);
  const double* Xu = Xk + ((long long)(ku >= 0 ? ku : k) - k) * op.cells;
  const double* Xd = Xk + ((long long)(kd >= 0 ? kd : k) - k) * op.cells;
  const double ncd = (kd >= 0) ? __ldg(op.nvec + 3 * k + s) * op.cdn[s] : 0.0;
  const double gam = __ldg(op.Gamma + k);
  for (int j = 0; j < n; j++) {                                    // coalesced load, G_M formed per cell
    const int e = j * 32 + lane;
    const int ln = e / n, i = e - ln * n;
    const long long ql = (base + e) / op.pb;
    const double q = op.x0[s] + (double)(ql % op.n[s]) * op.h[s];
    const double Vp = fma(op.VSL[s], q, op.VLL[s]);
    const double xk = Xk[e];
    double v = __ldg(op.dU[s] + ql) * xk, pw = 0.0;
    if (ku >= 0) { const double xu = Xu[e]; v = fma(Vp, xu, v); pw = op.kup[s] * Vp * xu; }
    if (kd >= 0) { const double xd = Xd[e]; v = fma(ncd * Vp, xd, v); pw = fma(op.kdn[s] * ncd * Vp, xd, pw); }
    tile[ln * (n + 1) + i] = v;
    ptile[ln * (n + 1) + i] = fma(-gam, xk, pw * (op.x0[axis] + i * op.h[axis]));   // gauge terms of mode M, damping
  }
  __syncwarp();
  double* row = tile + lane * (n + 1);
  const double al = 1.0 / 3.0, ca = 7.0 / 9.0, cb = 1.0 / 36.0, inv_h = 1.0 / op.h[axis];
  double fm2 = 0.0, fm1 = 0.0, f0 = row[0], fp1 = (n > 1) ? row[1] : 0.0, prev = 0.0;
  for (int i = 0; i < n; i++) {                                    // forward elimination, in place
    const double fp2 = (i + 2 < n) ? row[i + 2] : 0.0;
    const double r = (ca * (fp1 - fm1) + cb * (fp2 - fm2)) * inv_h;
    prev = (i == 0) ? r * __ldg(bet) : (r - al * prev) * __ldg(bet + i);   // bet[]: reciprocal pivots
    row[i] = prev;
    fm2 = fm1; fm1 = f0; f0 = fp1; fp1 = fp2;
  }
  double next = 0.0;
  for (int i = n - 1; i >= 0; i--) {                               // back substitution, in place
    next = (i == n - 1) ? row[i] : row[i] - __ldg(cfac + i + 1) * next;
    row[i] = next;
  }
  __syncwarp();
  const double* Y = y + eoff + base;
  double* O = out + eoff + base;
  for (int j = 0; j < n; j++) {                                    // coalesced accumulation into the stage output
    const int e = j * 32 + lane;
    const int ln = e / n, i = e - ln * n;
    const double d = tile[ln * (n + 1) + i] + ptile[ln * (n + 1) + i];
    O[e] = first ? fma(a, Y[e], c * d) : fma(c, d, O[e]);
  }
}

// All p-derivative terms of one (element, q-point) in ONE pass over its p-brick (M >= 2; second solver design of step
// a9).  Everything that needs a p_s-derivative is local to the brick: for every mode s the operand
//   G_s = (dU/dq_s) X_k + V'_s X_up(k,s) + n_s c_s V'_s X_dn(k,s)
// is formed from coalesced loads into a shared tile (brick layout with the rows of the contiguous axis padded to n + 1,
// so that lines along every axis are bank-conflict free); the right-hand side B G_s / h of Eq. (29) is taken by all
// threads in parallel into a second tile, and only the two Thomas recurrences of tridiag(1/3, 1, 1/3) run one thread
// per line, in place, one dependent FMA per point (elimination factors and reciprocal pivots tabulated by the host:
// no division, no thread-local array).  Every thread collects the result for the cells it owns in registers together
// with the pointwise gauge terms and the damping: one read of X_k, X_up, X_dn and one read-modify-write of `out` per
// stage instead of one such pass per momentum axis.  The K elements of a q-point run in consecutive CTAs, so the bricks
// of hierarchy neighbours are served by L2.  CPT cells per thread: pb <= CPT * blockDim.x.
// NP > 0: cubic bricks of NP points per momentum axis with NP^M = CPT * 512 cells known at compile time (every index
// decode, stride and loop bound becomes a constant); NP = 0: run-time brick shape.
__host__ __device__ constexpr int pbrick_ipow(int b, int e) { return e <= 0 ? 1 : b * pbrick_ipow(b, e - 1); }
__host__ __device__ constexpr int pbrick_nt(int m, int cpt, int np) {   // threads per CTA of a compile-time shape (0: run time, <= 512)
  return np ? ((pbrick_ipow(np, m) + cpt - 1) / cpt + 31) / 32 * 32 : 512;
}
template <int M, int PBRICK_CPT, int NP>
__global__ void __launch_bounds__(pbrick_nt(M, PBRICK_CPT, NP), (PBRICK_CPT == 8) ? 2 : 1) k_compact_pbrick(DevOp op, CompactTables ct, const double* __restrict__ in,
                                                         double* out, double c, size_t slot_stride) {
  extern __shared__ double ptile_s[];
  const int NT = NP ? pbrick_nt(M, PBRICK_CPT, NP) : blockDim.x, t = threadIdx.x;
  const int pb = NP ? pbrick_ipow(NP, M) : (int)op.pb, nl = NP ? NP : op.n[2 * M - 1];
  double* tile = ptile_s;                                           // G_s
  double* rt = ptile_s + (pb + pb / nl);                            // B G_s / h, then d = A^{-1} B G_s
  const long long ql = blockIdx.x / op.K;
  const int k = (int)(blockIdx.x - ql * op.K);
  const size_t eoff = (size_t)blockIdx.z * slot_stride + (size_t)k * op.cells + (size_t)ql * pb;
  const double* Xk = in + eoff;
  int iq[M];
  {
    long long r = ql;
#pragma unroll
    for (int s = M - 1; s >= 0; s--) { iq[s] = (int)(r % op.n[s]); r /= op.n[s]; }
  }
  const double gam = __ldg(op.Gamma + k);
  double acc[PBRICK_CPT];                                           // (X_k is re-read per mode: L1 / L2 hits, 16 registers less)
  int pcs[PBRICK_CPT], pidx[PBRICK_CPT];                            // padded tile index, packed momentum indices (10 bits each)
#pragma unroll
  for (int j = 0; j < PBRICK_CPT; j++) {
    const int cell = t + j * NT;
    acc[j] = (cell < pb) ? -gam * Xk[cell] : 0.0;                   // damping -Gamma_k X_k
    pcs[j] = cell + cell / nl;
    int r = cell, pk = 0;
#pragma unroll
    for (int s = M - 1; s >= 0; s--) { const int n = NP ? NP : op.n[M + s]; const int q = r / n; pk |= (r - q * n) << (10 * s); r = q; }
    pidx[j] = pk;
  }
  const double al = 1.0 / 3.0, ca = 7.0 / 9.0, cb = 1.0 / 36.0;
#pragma unroll
  for (int s = 0; s < M; s++) {
    const int ap = M + s, n = NP ? NP : op.n[ap], stb = NP ? pbrick_ipow(NP, M - 1 - s) : (int)op.st[ap];   // stride of p_s inside the brick
    const double q = op.x0[s] + iq[s] * op.h[s];
    const double Vp = fma(op.VSL[s], q, op.VLL[s]);
    const double ck = __ldg(op.dU[s] + ql);
    const int ku = __ldg(op.up + 3 * k + s), kd = __ldg(op.dn + 3 * k + s);
    const double cu = (ku >= 0) ? Vp : 0.0;
    const double cd = (kd >= 0) ? __ldg(op.nvec + 3 * k + s) * op.cdn[s] * Vp : 0.0;
    const double* Xu = Xk + ((long long)(ku >= 0 ? ku : k) - k) * op.cells;
    const double* Xd = Xk + ((long long)(kd >= 0 ? kd : k) - k) * op.cells;
    const int pitch = (stb == 1) ? 1 : stb + stb / nl;              // padded stride of p_s
    const double inv_h = 1.0 / op.h[ap];
#pragma unroll
    for (int j = 0; j < PBRICK_CPT; j++) {
      const int cell = t + j * NT;
      if (cell < pb) {
        double v = ck * Xk[cell], pw = 0.0;
        if (ku >= 0) { const double xu = Xu[cell]; v = fma(cu, xu, v); pw = op.kup[s] * cu * xu; }
        if (kd >= 0) { const double xd = Xd[cell]; v = fma(cd, xd, v); pw = fma(op.kdn[s] * cd, xd, pw); }
        const int i = (pidx[j] >> (10 * s)) & 1023;
        acc[j] = fma(op.x0[ap] + i * op.h[ap], pw, acc[j]);         // gauge terms p_s V'_s (kup X_up + n c kdn X_dn)
        tile[pcs[j]] = v;
      }
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < PBRICK_CPT; j++) {                          // right-hand side of Eq. (29), zero ghosts (R9)
      const int cell = t + j * NT;
      if (cell < pb) {
        const int i = (pidx[j] >> (10 * s)) & 1023, pc = pcs[j];
        const double fp1 = (i + 1 < n) ? tile[pc + pitch] : 0.0, fm1 = (i >= 1) ? tile[pc - pitch] : 0.0;
        const double fp2 = (i + 2 < n) ? tile[pc + 2 * pitch] : 0.0, fm2 = (i >= 2) ? tile[pc - 2 * pitch] : 0.0;
        rt[pc] = (ca * (fp1 - fm1) + cb * (fp2 - fm2)) * inv_h;
      }
    }
    __syncthreads();
    {                                                               // A d = r along p_s, in place in rt
      const double* ibet = ct.ibet[ap];
      const double* cfac = ct.cfac[ap];
      const int nlines = pb / n;
      for (int L = t; L < nlines; L += NT) {
        const int outer = L / stb, inner = L - outer * stb;
        const int base = outer * stb * n + inner;
        double* row = rt + base + base / nl;
        double prev = row[0] * __ldg(ibet);
        row[0] = prev;
#pragma unroll(NP ? NP : 4)
        for (int i = 1; i < n; i++) {                               // forward elimination: r'_i = (r_i - r'_{i-1}/3) / bet_i
          const double ib = __ldg(ibet + i);
          prev = fma(-al * ib, prev, row[i * pitch] * ib);
          row[i * pitch] = prev;
        }
#pragma unroll(NP ? NP : 4)
        for (int i = n - 2; i >= 0; i--) {                          // back substitution
          prev = fma(-__ldg(cfac + i + 1), prev, row[i * pitch]);
          row[i * pitch] = prev;
        }
      }
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < PBRICK_CPT; j++) {
      const int cell = t + j * NT;
      if (cell < pb) acc[j] += rt[pcs[j]];
    }
  }
  double* O = out + eoff;
#pragma unroll
  for (int j = 0; j < PBRICK_CPT; j++) {
    const int cell = t + j * NT;
    if (cell < pb) O[cell] = fma(c, acc[j], O[cell]);
  }
}

// The brick pass for cubic three-mode bricks of NP^3 cells (NP = 16: config 4, NP = 20: config 5), thread-per-column form:
// thread (i_2, i_3) owns the NP cells of its p_1 column in registers.  Per mode s it forms G_s on its column; the p_1 lines
// ARE the columns, so their right-hand sides and Thomas recurrences run in registers with no shared memory and no barrier;
// for p_2 and p_3 the columns go through one shared tile [i_1][i_2][i_3 + pad], thread (i_1, i_3) resp. (i_1, i_2) takes
// one line into registers, solves it and puts it back, and the owners add their cells.  Same arithmetic as
// k_compact_pbrick; about a quarter of its instructions (no index decode, no ghost predicates on shared loads, every
// thread busy in the recurrences of modes 2 and 3).
template <int NP>
__global__ void __launch_bounds__((NP * NP + 31) / 32 * 32, (NP == 16) ? 2 : 1) k_compact_pcolumn(
    DevOp op, CompactTables ct, const double* __restrict__ in, double* out, double c, size_t slot_stride) {
  extern __shared__ double pcol_s[];
  constexpr int M = 3, LD = NP + 1, PL = NP * NP, PB = NP * PL;
  const int t = threadIdx.x;
  const bool active = t < PL;
  const int ta = active ? t : 0;
  const int ia = ta / NP, ib = ta - ia * NP;                        // (i_2, i_3) as owner; (i_1, i_3) / (i_1, i_2) as line solver
  const long long ql = blockIdx.x / op.K;
  const int k = (int)(blockIdx.x - ql * op.K);
  const size_t eoff = (size_t)blockIdx.z * slot_stride + (size_t)k * op.cells + (size_t)ql * PB;
  const double* Xk = in + eoff + ta;                                // cell (i_1, i_2, i_3) = i_1 * PL + t
  int iq[M];
  {
    long long r = ql;
#pragma unroll
    for (int s = M - 1; s >= 0; s--) { iq[s] = (int)(r % op.n[s]); r /= op.n[s]; }
  }
  if (t == 0) {
    // the bricks this CTA will read later -- hierarchy neighbours of the three modes, the output -- are contiguous runs of
    // PB doubles: ask L2 for them now, so that the three mode phases and the final read-modify-write do not each pay a
    // DRAM latency with only two CTAs per SM to hide it
    const double* base = in + eoff;
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(out + eoff), "r"((unsigned)(PB * sizeof(double))) : "memory");
#pragma unroll
    for (int s = 0; s < M; s++) {
      const int ku = __ldg(op.up + 3 * k + s), kd = __ldg(op.dn + 3 * k + s);
      if (ku >= 0) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(base + ((long long)ku - k) * op.cells), "r"((unsigned)(PB * sizeof(double))) : "memory");
      if (kd >= 0) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(base + ((long long)kd - k) * op.cells), "r"((unsigned)(PB * sizeof(double))) : "memory");
    }
  }
  const double gam = __ldg(op.Gamma + k);
  double acc[NP];
#pragma unroll
  for (int i = 0; i < NP; i++) acc[i] = -gam * Xk[i * PL];
  const double al = 1.0 / 3.0, ca = 7.0 / 9.0, cb = 1.0 / 36.0;
  auto solve = [&](double (&f)[NP], const int ap) {                 // f <- A^{-1} B f / h along one line
    const double* __restrict__ ibet = ct.ibet[ap];
    const double* __restrict__ cfac = ct.cfac[ap];
    const double inv_h = 1.0 / op.h[ap];
    double fm2 = 0.0, fm1 = 0.0, prev = 0.0;
#pragma unroll
    for (int i = 0; i < NP; i++) {
      const double fp1 = (i + 1 < NP) ? f[i + 1] : 0.0, fp2 = (i + 2 < NP) ? f[i + 2] : 0.0;
      const double r = (ca * (fp1 - fm1) + cb * (fp2 - fm2)) * inv_h;
      const double ibi = __ldg(ibet + i);
      fm2 = fm1; fm1 = f[i];
      prev = (i == 0) ? r * ibi : fma(-al * ibi, prev, r * ibi);
      f[i] = prev;
    }
#pragma unroll
    for (int i = NP - 2; i >= 0; i--) f[i] = fma(-__ldg(cfac + i + 1), f[i + 1], f[i]);
  };
#pragma unroll
  for (int s = 0; s < M; s++) {
    const int ap = M + s;
    const double q = op.x0[s] + iq[s] * op.h[s];
    const double Vp = fma(op.VSL[s], q, op.VLL[s]);
    const double ck = __ldg(op.dU[s] + ql);
    const int ku = __ldg(op.up + 3 * k + s), kd = __ldg(op.dn + 3 * k + s);
    const double cu = (ku >= 0) ? Vp : 0.0;
    const double cd = (kd >= 0) ? __ldg(op.nvec + 3 * k + s) * op.cdn[s] * Vp : 0.0;
    const double* Xu = Xk + ((long long)(ku >= 0 ? ku : k) - k) * op.cells;
    const double* Xd = Xk + ((long long)(kd >= 0 ? kd : k) - k) * op.cells;
    const double pu = op.kup[s] * cu, pd = op.kdn[s] * cd;
    double g[NP];
#pragma unroll
    for (int i = 0; i < NP; i++) {                                  // G_s and the gauge terms p_s V'_s (kup X_up + n c kdn X_dn)
      double v = ck * Xk[i * PL], pw = 0.0;
      if (ku >= 0) { const double xu = Xu[i * PL]; v = fma(cu, xu, v); pw = pu * xu; }
      if (kd >= 0) { const double xd = Xd[i * PL]; v = fma(cd, xd, v); pw = fma(pd, xd, pw); }
      const int ip = (s == 0) ? i : (s == 1 ? ia : ib);
      acc[i] = fma(op.x0[ap] + ip * op.h[ap], pw, acc[i]);
      g[i] = v;
    }
    if (s == 0) {                                                   // p_1 lines: the thread's own column
      solve(g, ap);
#pragma unroll
      for (int i = 0; i < NP; i++) acc[i] += g[i];
    } else {
      if (s == 2) __syncthreads();                                  // the owners have read the p_2 results
      if (active) {
#pragma unroll
        for (int i = 0; i < NP; i++) pcol_s[(i * NP + ia) * LD + ib] = g[i];
      }
      __syncthreads();
      // line of thread (ia, ib): s = 1: (i_1 = ia, i_3 = ib) along i_2; s = 2: (i_1 = ia, i_2 = ib) along i_3
      double* L = (s == 1) ? pcol_s + ia * NP * LD + ib : pcol_s + (ia * NP + ib) * LD;
      constexpr int one = 1;
      const int st = (s == 1) ? LD : one;
#pragma unroll
      for (int i = 0; i < NP; i++) g[i] = L[i * st];
      solve(g, ap);
      if (active) {
#pragma unroll
        for (int i = 0; i < NP; i++) L[i * st] = g[i];
      }
      __syncthreads();
#pragma unroll
      for (int i = 0; i < NP; i++) acc[i] += pcol_s[(i * NP + ia) * LD + ib];
    }
  }
  if (active) {
    double* O = out + eoff + ta;
    double o[NP];
#pragma unroll
    for (int i = 0; i < NP; i++) o[i] = O[i * PL];
#pragma unroll
    for (int i = 0; i < NP; i++) O[i * PL] = fma(c, acc[i], o[i]);
  }
}

}  // namespace

#define CDISPATCH(M, CALL) do { if ((M) == 1) { CALL(1); } else if ((M) == 2) { CALL(2); } else { CALL(3); } } while (0)

static int compact_deriv(const DevOp& op, const CompactTables& ct, const double* f, int axis, double* d, cudaStream_t s) {
  const int n = op.n[axis];
  const long long nlines = op.cells / n;
  k_compact_deriv<<<(unsigned)((nlines + 127) / 128), 128, 0, s>>>(f, d, nlines, n, op.st[axis], 1.0 / op.h[axis],
                                                                   ct.ibet[axis], ct.cfac[axis]);
  return 1;
}

// out = a*y + c*F(in) for slots [0, nb); scratch: three element-sized arrays (the second one holds the elimination
// values of lines longer than CLINE_MAX)
int launch_stage_compact(const DevOp& op, const CompactTables& ct, const double* in, const double* y, double* out, double a,
                         double c, int nb, size_t slot_stride, double* scratch, cudaStream_t s) {
  int launches = 0;
  double* D = scratch + op.cells;
  int first = 1;
  // p part in one brick pass (M >= 2, brick <= 16 cells per thread of a 512-thread CTA and <= 200 KB padded);
  // CHFPE_COMPACT_PBRICK=0 keeps one line pass per momentum axis (the first design; profiles/r02_compact_*.txt)
  static const bool pbrick_on = []() { const char* e = getenv("CHFPE_COMPACT_PBRICK"); return !(e && e[0] == '0'); }();
  const int nl = op.n[2 * op.M - 1];
  const size_t tile_bytes = 2 * sizeof(double) * (size_t)(op.pb + op.pb / nl);   // operand tile + right-hand-side tile
  // (measured per stage, brick pass vs line passes: config 4 16.8 vs 18.3 ms, config 3 3.56 vs 4.58 ms; 20^3 bricks with
  // 16 cells per thread lose, 83.3 vs 74.9 ms, so they stay on the line passes unless CHFPE_COMPACT_PBRICK=2)
  static const bool pbrick_big = []() { const char* e = getenv("CHFPE_COMPACT_PBRICK"); return e && e[0] == '2'; }();
  static const bool cube_on = []() { const char* e = getenv("CHFPE_COMPACT_CUBE"); return !(e && e[0] == '0'); }();
  // (with the compile-time 20^3 shape the brick pass wins there as well: 55.4 vs 69.3 ms per stage at config 5)
  const bool is20 = cube_on && op.M == 3 && op.n[3] == 20 && op.n[4] == 20 && op.n[5] == 20;
  bool pbrick = pbrick_on && op.M >= 2 && op.pb <= ((pbrick_big || is20) ? 16 : 8) * 512 && tile_bytes <= 200 * 1024 && op.nqc * op.K <= 0x7fffffffLL;
  for (int s2 = 0; s2 < op.M; s2++) if (op.n[op.M + s2] > 1023) pbrick = false;
  // q_2 and q_3 of three modes in one launch where the plane tile fits (CHFPE_COMPACT_QPLANE=0: one line pass per axis)
  static const bool qplane_on = []() { const char* e = getenv("CHFPE_COMPACT_QPLANE"); return !(e && e[0] == '0'); }();
  const int qp = (qplane_on && op.M == 3 && op.n[1] == op.n[2] && op.pb % 16 == 0 && (size_t)op.K * op.n[0] * (op.pb / 16) <= 0x7fffffffULL)
                     ? ((op.n[1] == 16 || op.n[1] == 20) ? op.n[1] : 0) : 0;
  for (int pa = 0; pa < (pbrick ? 1 : 2); pa++)
    for (int sI = 0; sI < op.M; sI++) {
      if (pa == 0 && qp && sI >= 1) {
        if (sI == 1) {
          const dim3 grid((unsigned)((size_t)op.K * op.n[0] * (op.pb / 16)), 1, nb);
          const size_t sm = 2 * sizeof(double) * (size_t)qp * qp * 16;
          static bool optin = false;
          if (!optin) {
            cudaFuncSetAttribute(k_compact_qplane<16, 16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(2 * 8 * 16 * 16 * 16));
            cudaFuncSetAttribute(k_compact_qplane<20, 16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(2 * 8 * 20 * 20 * 16));
            optin = true;
          }
          if (qp == 16) k_compact_qplane<16, 16><<<grid, 16 * 16, sm, s>>>(op, in, y, out, a, c, first, slot_stride, ct.ibet[1], ct.cfac[1], ct.ibet[2], ct.cfac[2]);
          else k_compact_qplane<20, 16><<<grid, 20 * 16, sm, s>>>(op, in, y, out, a, c, first, slot_stride, ct.ibet[1], ct.cfac[1], ct.ibet[2], ct.cfac[2]);
          launches++;
          first = 0;
        }
        continue;
      }
      const int axis = pa ? op.M + sI : sI;
      const int n = op.n[axis];
      static const bool qline_on = []() { const char* e = getenv("CHFPE_COMPACT_QLINE"); return !(e && e[0] == '0'); }();
      if (pa == 0 && qline_on && n == 48 && op.M == 2) {                // config 3's lines: blocked window
        const dim3 grid((unsigned)((op.cells / n + 127) / 128), op.K, nb);
        k_compact_qline_long<2, 48><<<grid, 128, 0, s>>>(op, in, y, out, a, c, sI, first, slot_stride, ct.ibet[axis], ct.cfac[axis]);
        launches++;
        first = 0;
        continue;
      }
      if (pa == 0 && qline_on && (n == 16 || n == 20) && op.M >= 2) {   // q lines of the BASELINE lengths: loads ahead of the recurrence
        const dim3 grid((unsigned)((op.cells / n + 127) / 128), op.K, nb);
#define CALLQ(MM)                                                                                                     \
  do {                                                                                                                \
    if (n == 16) k_compact_qline<MM, 16><<<grid, 128, 0, s>>>(op, in, y, out, a, c, sI, first, slot_stride, ct.ibet[axis], ct.cfac[axis]); \
    else k_compact_qline<MM, 20><<<grid, 128, 0, s>>>(op, in, y, out, a, c, sI, first, slot_stride, ct.ibet[axis], ct.cfac[axis]);       \
  } while (0)
        CDISPATCH(op.M, CALLQ);
#undef CALLQ
        launches++;
        first = 0;
        continue;
      }
      const unsigned lb = (unsigned)((op.cells / n + 127) / 128);
      const bool local = n <= CLINE_MAX;
#define LINE(MM, PA, NFV, GRID, K0, B0)                                                                               \
  k_compact_line<MM, PA, NFV><<<GRID, 128, 0, s>>>(op, in, y, out, a, c, sI, first, K0, B0, slot_stride, ct.ibet[axis],  \
                                                   ct.cfac[axis], D)
#define LINE_PA(MM, NFV, GRID, K0, B0)                                                                                \
  do { if (pa) LINE(MM, 1, NFV, GRID, K0, B0); else LINE(MM, 0, NFV, GRID, K0, B0); } while (0)
#define CALL(MM)                                                                                                      \
  do {                                                                                                                \
    if (pa && sI == MM - 1 && n <= 32 && op.cells % (32 * n) == 0) {       /* contiguous axis: transposing kernel */    \
      const unsigned wb = (unsigned)((op.cells / n / 32 + 3) / 4);                                                    \
      static bool optin_##MM = false;                                      /* n >= 24 needs more than 48 KB */          \
      if (!optin_##MM) {                                                                                              \
        cudaFuncSetAttribute(k_compact_pline_s1<MM>, cudaFuncAttributeMaxDynamicSharedMemorySize,                     \
                             (int)(sizeof(double) * 4 * 64 * 33));                                                    \
        optin_##MM = true;                                                                                            \
      }                                                                                                               \
      k_compact_pline_s1<MM><<<dim3(wb, op.K, nb), 128, sizeof(double) * 4 * 64 * (n + 1), s>>>(                      \
          op, in, y, out, a, c, first, slot_stride, ct.ibet[axis], ct.cfac[axis]);                                     \
      launches++;                                                                                                     \
    } else if (local) {                                                                                               \
      const dim3 grid(lb, op.K, nb);                                                                                  \
      LINE_PA(MM, 0, grid, 0, 0);                                                                                     \
      launches++;                                                                                                     \
    } else {                                                                                                          \
      for (int b = 0; b < nb; b++)                                                                                    \
        for (int k = 0; k < op.K; k++) {                                                                              \
          LINE_PA(MM, -1, dim3(lb, 1, 1), k, b);                                                                      \
          launches++;                                                                                                 \
        }                                                                                                             \
    }                                                                                                                 \
  } while (0)
      CDISPATCH(op.M, CALL);
#undef CALL
#undef LINE_PA
#undef LINE
      first = 0;
    }
  if (pbrick) {
    const int cpt = (op.pb <= 8 * 512) ? 8 : 16;                      // cells per thread
    int nt = (int)((op.pb + cpt - 1) / cpt);
    nt = (nt + 31) / 32 * 32;
    if (nt < 64) nt = 64;
    static bool optin = false;
    if (!optin) {
      cudaFuncSetAttribute(k_compact_pbrick<2, 8, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
      cudaFuncSetAttribute(k_compact_pbrick<2, 16, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
      cudaFuncSetAttribute(k_compact_pbrick<3, 8, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
      cudaFuncSetAttribute(k_compact_pbrick<3, 16, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
      cudaFuncSetAttribute(k_compact_pbrick<3, 8, 16>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
      cudaFuncSetAttribute(k_compact_pbrick<3, 16, 20>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
      cudaFuncSetAttribute(k_compact_pbrick<2, 8, 48>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
      optin = true;
    }
    const dim3 grid((unsigned)(op.nqc * op.K), 1, nb);                // element fastest: hierarchy neighbours meet in L2
    const bool cube16 = cube_on && op.M == 3 && op.n[3] == 16 && op.n[4] == 16 && op.n[5] == 16 && nt == 512;
    const bool cube20 = cube_on && op.M == 3 && op.n[3] == 20 && op.n[4] == 20 && op.n[5] == 20 && nt == 512 && cpt == 16;
    const bool sq48 = cube_on && op.M == 2 && op.n[2] == 48 && op.n[3] == 48 && nt == 288 && cpt == 8;
    static const bool pcol_on = []() { const char* e = getenv("CHFPE_COMPACT_PCOLUMN"); return !(e && e[0] == '0'); }();
    static bool pcol_optin = false;
    if (!pcol_optin) {
      cudaFuncSetAttribute(k_compact_pcolumn<20>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(double) * 20 * 20 * 21));
      pcol_optin = true;
    }
    if (pcol_on && cube16) k_compact_pcolumn<16><<<grid, 256, sizeof(double) * 16 * 16 * 17, s>>>(op, ct, in, out, c, slot_stride);
    else if (pcol_on && cube20) k_compact_pcolumn<20><<<grid, 416, sizeof(double) * 20 * 20 * 21, s>>>(op, ct, in, out, c, slot_stride);
    else if (sq48) k_compact_pbrick<2, 8, 48><<<grid, nt, tile_bytes, s>>>(op, ct, in, out, c, slot_stride);
    else if (cube20) k_compact_pbrick<3, 16, 20><<<grid, nt, tile_bytes, s>>>(op, ct, in, out, c, slot_stride);
    else if (op.M == 2 && cpt == 8) k_compact_pbrick<2, 8, 0><<<grid, nt, tile_bytes, s>>>(op, ct, in, out, c, slot_stride);
    else if (op.M == 2) k_compact_pbrick<2, 16, 0><<<grid, nt, tile_bytes, s>>>(op, ct, in, out, c, slot_stride);
    else if (cube16) k_compact_pbrick<3, 8, 16><<<grid, nt, tile_bytes, s>>>(op, ct, in, out, c, slot_stride);
    else if (cpt == 8) k_compact_pbrick<3, 8, 0><<<grid, nt, tile_bytes, s>>>(op, ct, in, out, c, slot_stride);
    else k_compact_pbrick<3, 16, 0><<<grid, nt, tile_bytes, s>>>(op, ct, in, out, c, slot_stride);
    launches++;
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
