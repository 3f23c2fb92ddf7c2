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
    prev = (i == 0) ? r / __ldg(bet) : (r - al * prev) / __ldg(bet + i);
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
    prev = (i == 0) ? r / __ldg(bet) : (r - al * prev) / __ldg(bet + i);
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

}  // namespace

#define CDISPATCH(M, CALL) do { if ((M) == 1) { CALL(1); } else if ((M) == 2) { CALL(2); } else { CALL(3); } } while (0)

static int compact_deriv(const DevOp& op, const CompactTables& ct, const double* f, int axis, double* d, cudaStream_t s) {
  const int n = op.n[axis];
  const long long nlines = op.cells / n;
  k_compact_deriv<<<(unsigned)((nlines + 127) / 128), 128, 0, s>>>(f, d, nlines, n, op.st[axis], 1.0 / op.h[axis],
                                                                   ct.bet[axis], ct.cfac[axis]);
  return 1;
}

// out = a*y + c*F(in) for slots [0, nb); scratch: three element-sized arrays (the second one holds the elimination
// values of lines longer than CLINE_MAX)
int launch_stage_compact(const DevOp& op, const CompactTables& ct, const double* in, const double* y, double* out, double a,
                         double c, int nb, size_t slot_stride, double* scratch, cudaStream_t s) {
  int launches = 0;
  double* D = scratch + op.cells;
  int first = 1;
  for (int pa = 0; pa < 2; pa++)
    for (int sI = 0; sI < op.M; sI++) {
      const int axis = pa ? op.M + sI : sI;
      const int n = op.n[axis];
      const unsigned lb = (unsigned)((op.cells / n + 127) / 128);
      const bool local = n <= CLINE_MAX;
#define LINE(MM, PA, NFV, GRID, K0, B0)                                                                               \
  k_compact_line<MM, PA, NFV><<<GRID, 128, 0, s>>>(op, in, y, out, a, c, sI, first, K0, B0, slot_stride, ct.bet[axis],  \
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
          op, in, y, out, a, c, first, slot_stride, ct.bet[axis], ct.cfac[axis]);                                     \
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
