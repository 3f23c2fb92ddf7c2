// Brick kernel of the RK stage (steps a1-a3 of DESIGN.md) for two and three modes on sm_100a.
//
// Internal layout [k][q_1..q_M][p_1..p_M] makes all momenta of one (element, q-point) a contiguous "p-brick".
// Everything in Eq. (8) :77-80 except the q-derivatives of Eq. (9)-(10) :86-91 is local to the bricks of one
// q-point: the p_s-derivatives of W^(n) (Eq. 10), of W^(n+e_s) (Phi, Eq. 11 :96) and of W^(n-e_s) (Theta, Eq. 12
// :100) have q-only coefficients, so they are taken ONCE on the combination
//     G_s = (dU/dq_s) X_k + V'_s X_up(k,s) + n_s c_s V'_s X_dn(k,s)                      (per cell, 3 flops)
// The gauge terms kappa p_s X_{up,dn} are pointwise.  The q-derivatives are pointwise in the brick: coalesced loads
// of the same cell of the 12 neighbouring bricks of the same element, which the L2 serves (CTAs are ordered q_1-plane
// by q_1-plane, element group by group).  A CTA walks a short run of bricks; two-mode grids run as three-mode
// ones with a one-point middle mode (P2 == 1).  Grids without a compile-time specialisation run the
// generic kernel of chfpe_kernels.cu (a run-time-shaped brick kernel was measured slower than it and removed).
#include <type_traits>
#include "chfpe_internal.cuh"

namespace {

// L2 eviction policies (createpolicy + ld/st .L2::cache_hint): the stage input of the elements of the current
// group must survive in L2 for five q_1 planes, everything that is touched once (y, out, bricks of elements outside
// the group) is marked evict_first so that it cannot push the window out.
__device__ __forceinline__ unsigned long long l2_policy(int kind) {   // 0 normal, 1 evict_first, 2 evict_last
  unsigned long long p;
  if (kind == 1) asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  else if (kind == 2) asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  else asm("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ void bulk_prefetch_l2(const void* src, unsigned bytes) {   // bytes: multiple of 16
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}

// ------------------------------------------------------------------------------------------------
// Specialised M = 3 brick kernel with compile-time momentum extents (P1, P2, P3), 128-bit accesses.
// A thread owns a PAIR of cells adjacent along p_3 (one double2) on NC = P1/SPLIT consecutive p_1 planes; the SPLIT
// thread groups of a CTA share one brick.  The p_1 stencil of G_1 runs in registers in scatter form (each G_1 value
// is added to its four neighbours' accumulators as soon as it is formed; segment edges are exchanged through shared
// memory); G_2 and G_3 go to two shared arrays padded along their own axis only, so one __syncthreads per brick
// suffices.  The kernel is latency-bound at 16 warps per SM, so its time follows its instruction count: every load
// is "one 64-bit base per brick and direction + compile-time byte offset", the brick decode is 32-bit, and ghost
// bricks (R9) are handled by CTA-uniform branches (an all-interior fast path per q axis), not by selects.
// ------------------------------------------------------------------------------------------------
template <int OFF>   // OFF in double2 units, folded into the instruction as an immediate byte offset
__device__ __forceinline__ double2 ldg2o(const double2* base, unsigned long long pol) {
  double2 v;
  asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0, %1}, [%2+%4], %3;"
      : "=d"(v.x), "=d"(v.y) : "l"(base), "l"(pol), "n"(OFF * 16));
  return v;
}
// L1-allocating form (MODE 2) for the bricks of the q_3 line a CTA walks along: brick i_3+1 re-reads four of the
// five bricks that brick i_3 read, and the L1 (what the shared arrays leave of 256 KB) can hold small ones.
template <int OFF, int MODE>
__device__ __forceinline__ double2 ldg2o_l1(const double2* base, unsigned long long pol) {
  double2 v;
  if (MODE == 2)
    asm("ld.global.nc.L2::cache_hint.v2.f64 {%0, %1}, [%2+%4], %3;"
        : "=d"(v.x), "=d"(v.y) : "l"(base), "l"(pol), "n"(OFF * 16));
  else
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0, %1}, [%2+%4], %3;"
        : "=d"(v.x), "=d"(v.y) : "l"(base), "l"(pol), "n"(OFF * 16));
  return v;
}
template <int OFF>
__device__ __forceinline__ double2 ld2o(const double2* base, unsigned long long pol) {   // may alias the output
  double2 v;
  asm volatile("ld.global.L2::cache_hint.v2.f64 {%0, %1}, [%2+%4], %3;"
               : "=d"(v.x), "=d"(v.y) : "l"(base), "l"(pol), "n"(OFF * 16) : "memory");
  return v;
}
template <int OFF>
__device__ __forceinline__ void st2o(double2* base, double2 v, unsigned long long pol) {
  asm volatile("st.global.L2::cache_hint.v2.f64 [%0+%4], {%1, %2}, %3;" ::"l"(base), "d"(v.x), "d"(v.y), "l"(pol), "n"(OFF * 16) : "memory");
}
__device__ __forceinline__ double2 fma2(double c, double2 a, double2 b) { return make_double2(fma(c, a.x, b.x), fma(c, a.y, b.y)); }

// compile-time loop helpers (the load offsets must be template arguments)
template <int J, int N> struct Unroll {
  template <typename F> __device__ __forceinline__ static void run(F&& f) { f(std::integral_constant<int, J>()); Unroll<J + 1, N>::run(f); }
};
template <int N> struct Unroll<N, N> {
  template <typename F> __device__ __forceinline__ static void run(F&&) {}
};

// registers per thread that let MINB CTAs of NT threads share the 64 K registers of an SM
constexpr int brick3_maxreg(int nt, int minb) {
  const int warps = ((nt + 127) / 128) * 4;                        // warps are allocated in groups of four
  const int r = (65536 / (minb * warps * 32)) & ~7;
  return r > 255 ? 255 : r;
}

// true if the P3/2 pairs of a p_3 row are a power-of-two lane group of a warp and warps hold whole rows
__host__ __device__ constexpr bool brick3_shfl3(int p2, int p3, int split) {
  return (32 % (p3 / 2) == 0) && ((split * p2 * p3 / 2) % 32 == 0) && ((p2 * p3 / 2) % (p3 / 2) == 0);
}

// NPASS > 1: a brick is processed in NPASS passes over blocks of P1/NPASS consecutive p_1 planes (large bricks: keeps
// the per-thread state small); G_1 of the two planes beyond a block edge is recomputed from three extra loads.
template <int P1, int P2, int P3, int SPLIT, int MINB, int NPASS>
__global__ void __launch_bounds__(SPLIT * P2 * P3 / 2) __maxnreg__(brick3_maxreg(SPLIT * P2 * P3 / 2, MINB))
k_stage_brick3(DevOp op, BrickPlan bp, const double* __restrict__ in, const double* y, double* out, double a,
               double cc, size_t slot_stride, int y_is_in) {
  static_assert(P3 % 2 == 0 && P1 % (SPLIT * NPASS) == 0 && P1 / (SPLIT * NPASS) >= 2, "unsupported brick shape");
  constexpr int PLANE = P2 * P3, PL2 = PLANE / 2, NTT = SPLIT * PL2, P1P = P1 / NPASS, NC = P1P / SPLIT;
  // P2 == 1: two-mode systems run as a three-mode one whose middle mode has a single q and a single p point and no
  // couplings (same memory layout); everything that belongs to that mode is compiled out.
  constexpr bool SKIP1 = (P2 == 1);
  // bricks of the q_3 line go through L1 when five of them fit beside the shared arrays (measured: two-mode 48 x 48
  // bricks 0.79 -> 0.75 ms per stage; 16^3 bricks, 160 KB per five, gain nothing and keep L1::no_allocate)
  constexpr int L1Q3 = (5 * P1 * P2 * P3 * (int)sizeof(double) <= 100 * 1024) ? 2 : 0;
  constexpr int G2_ROW = P3, G2_PLANE = SKIP1 ? 0 : (P2 + 4) * P3;  // G_2[i1][i2+2][i3]
  // p_3 rows of P3/2 pairs that tile a warp: the p_3 stencil of G_3 runs on warp shuffles as soon as G_3 is formed
  // (no shared array, no copy kept in registers); other shapes stage G_3 in shared memory like G_2.
  constexpr bool SHFL3 = brick3_shfl3(P2, P3, SPLIT);
  constexpr int G3_ROW = P3 + 4, G3_PLANE = SHFL3 ? 0 : P2 * (P3 + 4);   // G_3[i1][i2][i3+2]
  extern __shared__ __align__(16) double sm[];
  double* g2 = sm;
  double* g3 = sm + P1P * G2_PLANE;
  double* xg = g3 + P1P * G3_PLANE;                                 // [SPLIT][4][PLANE]: first/last two G_1 planes of a segment
  const int seg = (SPLIT == 1) ? 0 : threadIdx.x / PL2;
  const int tid = threadIdx.x - seg * PL2;                          // pair index inside the plane
  const int jbase = seg * NC;                                       // first p_1 plane of this thread
  const int i2 = tid / (P3 / 2), i3 = 2 * (tid - i2 * (P3 / 2));

  // zero the ghost rows / columns of the two shared bricks
  for (int i = threadIdx.x; i < (SKIP1 ? 0 : P1P * 4 * P3); i += NTT) {   // G_2: rows i2 = -2,-1,P2,P2+1 of every plane
    const int pl = i / (4 * P3), rr = i - pl * (4 * P3), row = rr / P3, col = rr - row * P3;
    g2[pl * G2_PLANE + (row < 2 ? row : P2 + row) * G2_ROW + col] = 0.0;
  }
  for (int i = threadIdx.x; i < (SHFL3 ? 0 : P1P * P2 * 4); i += NTT) {   // G_3: columns i3 = -2,-1,P3,P3+1 of every row
    const int rw = i >> 2, c4 = i & 3;
    g3[rw * G3_ROW + (c4 < 2 ? c4 : P3 + c4)] = 0.0;
  }

  const unsigned long long pol_own = l2_policy((bp.l2mode & 2) ? 2 : 0);
  const unsigned long long pol_str = l2_policy((bp.l2mode & 1) ? 1 : 0);
  const bool wide = (op.scheme == CHFPE_CENTRAL4);
  const double h1 = op.h[3];
  const double p2 = op.x0[4] + i2 * op.h[4];
  const double p3a = op.x0[5] + i3 * op.h[5], p3b = op.x0[5] + (i3 + 1) * op.h[5];
  // ---- bricks of this CTA: bp.bpc consecutive entries of the brick order (setup above is paid once) ----
  const long long n_bricks = (long long)op.K * op.nqc;
  for (long long L = (long long)blockIdx.x * bp.bpc, Lend = L + bp.bpc; L < Lend && L < n_bricks; L++) {
  const BrickId bid = decode_brick_id(op, bp, L);
  const int k = bid.k;
  const unsigned ql = (unsigned)bid.ql;
  const size_t boff = (size_t)blockIdx.y * slot_stride;
  const double2* X2 = reinterpret_cast<const double2*>(in + boff);  // replica base
  const unsigned cells2 = (unsigned)(op.cells >> 1);                // element stride in double2
#pragma unroll 1
  for (int pass = 0; pass < NPASS; pass++) {
  const int pofs = pass * P1P;                                      // first p_1 plane of this pass
  const double p1_0 = op.x0[3] + (pofs + jbase) * h1;
  const unsigned tpart = (unsigned)((pofs + jbase) * PL2 + tid);    // this thread's first pair inside a brick
  const unsigned brick2 = ql * (unsigned)(P1 * PL2);                // brick offset inside an element
  const double2* Xk = X2 + ((size_t)k * cells2 + brick2 + tpart);   // own pairs: Xk[j * PL2]

  const double Gam = __ldg(op.Gamma + k);
  int kup[3], kdn[3];
#pragma unroll
  for (int s = 0; s < 3; s++) { kup[s] = __ldg(op.up + 3 * k + s); kdn[s] = __ldg(op.dn + 3 * k + s); }

  // Everything this brick needs from HBM (its own stage input, the bricks of its hierarchy neighbours, y) is
  // requested into L2 now -- one bulk prefetch per array, issued by one thread -- and consumed after the
  // q-derivative part, whose loads are L2 hits on the q_1-plane window and cover the DRAM latency.
  if (threadIdx.x == 0 && pass == 0) {
    constexpr unsigned BB = P1 * PLANE * sizeof(double);
    const double* Xd = in + boff;
    const size_t b0 = (size_t)ql * (P1 * PLANE);
    bulk_prefetch_l2(Xd + (size_t)k * op.cells + b0, BB);
    if (!y_is_in) bulk_prefetch_l2(y + boff + (size_t)k * op.cells + b0, BB);
#pragma unroll
    for (int s = 0; s < 3; s++) {
      if (SKIP1 && s == 1) continue;
      if (kup[s] >= 0) bulk_prefetch_l2(Xd + (size_t)kup[s] * op.cells + b0, BB);
      if (kdn[s] >= 0) bulk_prefetch_l2(Xd + (size_t)kdn[s] * op.cells + b0, BB);
    }
  }
  double2 acc[NC];
#pragma unroll
  for (int j = 0; j < NC; j++) acc[j] = make_double2(0.0, 0.0);

  // ---- -(p_s/m_s) dW/dq_s: same pair of the 4 neighbouring bricks of this element along every q axis ----
#pragma unroll
  for (int s = 0; s < 3; s++) {
    if (SKIP1 && s == 1) continue;
    const long long st2 = op.st[s] >> 1;                            // brick stride of q_s in double2 (even)
    const int i = bid.iq[s], n = op.n[s];
    const double wq = -(wide ? -op.c2[s] : op.c1[s]) * op.inv_mass[s];   // -(1/m_s) / (12 h) or / (2 h)
    const double cqa = wq * (s == 1 ? p2 : p3a), cqb = wq * (s == 1 ? p2 : p3b);
    const double2* bp1 = Xk + st2;
    const double2* bm1 = Xk - st2;
    if (wide && i >= 2 && i + 2 < n) {                              // interior in q_s: all four neighbours exist
      const double2* bp2 = Xk + 2 * st2;
      const double2* bm2 = Xk - 2 * st2;
      constexpr int CH = (NC <= 5) ? NC : 4;                        // planes per load batch (<= 20 loads), last one partial
      Unroll<0, (NC + CH - 1) / CH>::run([&](auto C0) {
        constexpr int j0 = decltype(C0)::value * CH;
        constexpr int CN = (NC - j0 < CH) ? NC - j0 : CH;
        double2 vp1[CN], vm1[CN], vp2[CN], vm2[CN];
        Unroll<0, CN>::run([&](auto J) {
          constexpr int j = decltype(J)::value;
          if (s == 2) {
            vp1[j] = ldg2o_l1<(j0 + j) * PL2, L1Q3>(bp1, pol_own);
            vm1[j] = ldg2o_l1<(j0 + j) * PL2, L1Q3>(bm1, pol_own);
            vp2[j] = ldg2o_l1<(j0 + j) * PL2, L1Q3>(bp2, pol_own);
            vm2[j] = ldg2o_l1<(j0 + j) * PL2, L1Q3>(bm2, pol_own);
          } else {
            vp1[j] = ldg2o<(j0 + j) * PL2>(bp1, pol_own);
            vm1[j] = ldg2o<(j0 + j) * PL2>(bm1, pol_own);
            vp2[j] = ldg2o<(j0 + j) * PL2>(bp2, pol_own);
            vm2[j] = ldg2o<(j0 + j) * PL2>(bm2, pol_own);
          }
        });
#pragma unroll
        for (int j = 0; j < CN; j++) {
          const double ex = fma(8.0, vp1[j].x - vm1[j].x, -(vp2[j].x - vm2[j].x));
          const double ey = fma(8.0, vp1[j].y - vm1[j].y, -(vp2[j].y - vm2[j].y));
          const double c1 = wq * fma((double)(j0 + j), h1, p1_0);
          acc[j0 + j].x = fma(s == 0 ? c1 : cqa, ex, acc[j0 + j].x);
          acc[j0 + j].y = fma(s == 0 ? c1 : cqb, ey, acc[j0 + j].y);
        }
      });
    } else {                                                        // edge of the q_s axis: one direction at a time
#pragma unroll
      for (int d = 0; d < 4; d++) {
        const int off = (d == 0) ? 1 : (d == 1 ? -1 : (d == 2 ? 2 : -2));
        if (i + off < 0 || i + off >= n || (!wide && d >= 2)) continue;          // ghost brick: contributes zero
        const double wd = wide ? ((d == 0) ? 8.0 : (d == 1 ? -8.0 : (d == 2 ? -1.0 : 1.0))) : ((d == 0) ? 1.0 : -1.0);
        const double2* b = Xk + off * st2;
        double2 v[NC];
        Unroll<0, NC>::run([&](auto J) {
          constexpr int j = decltype(J)::value;
          v[j] = (s == 2) ? ldg2o_l1<j * PL2, L1Q3>(b, pol_own) : ldg2o<j * PL2>(b, pol_own);
        });
#pragma unroll
        for (int j = 0; j < NC; j++) {
          const double c1 = wq * fma((double)j, h1, p1_0);
          acc[j].x = fma((s == 0 ? c1 : cqa) * wd, v[j].x, acc[j].x);
          acc[j].y = fma((s == 0 ? c1 : cqb) * wd, v[j].y, acc[j].y);
        }
      }
    }
  }

  // ---- own brick, hierarchy neighbours: G_s and the pointwise gauge terms ----
  double2 xk[NC];
  Unroll<0, NC>::run([&](auto J) { constexpr int j = decltype(J)::value; xk[j] = ldg2o_l1<j * PL2, L1Q3>(Xk, pol_own); });
#pragma unroll
  for (int j = 0; j < NC; j++) acc[j] = fma2(-Gam, xk[j], acc[j]);

  double w2 = 0.0, w3 = 0.0;                                        // 1/(12h) or 1/(2h) of p_2, p_3
  constexpr bool KEEP_G3 = (NC <= 8) && !SHFL3;                    // else re-read the own G_3 pair from shared memory
  double2 g3own[KEEP_G3 ? NC : 1];
#pragma unroll
  for (int s = 0; s < 3; s++) {
    if (SKIP1 && s == 1) continue;
    const double qs = op.x0[s] + bid.iq[s] * op.h[s];
    const double Vp = fma(op.VSL[s], qs, op.VLL[s]);
    const double dUs = __ldg(op.dU[s] + ql);
    const int ku = kup[s], kd = kdn[s];
    const double cu = Vp;
    const double cd = __ldg(op.nvec + 3 * k + s) * op.cdn[s] * Vp;
    const double pu = cu * op.kup[s], pd = cd * op.kdn[s];
    const double wp = wide ? -op.c2[3 + s] : op.c1[3 + s];
    if (s == 1) w2 = wp;
    if (s == 2) w3 = wp;
    const double wp8 = wide ? 8.0 * wp : wp, wp1 = wide ? wp : 0.0;
    const double2* Xu = X2 + ((size_t)(ku >= 0 ? ku : k) * cells2 + brick2 + tpart);
    const double2* Xd = X2 + ((size_t)(kd >= 0 ? kd : k) * cells2 + brick2 + tpart);
    const unsigned long long pol_u = ((bid.own >> (2 * s)) & 1) ? pol_own : pol_str;
    const unsigned long long pol_d = ((bid.own >> (2 * s + 1)) & 1) ? pol_own : pol_str;
    constexpr int CH = (NC <= 5) ? NC : (NC % 5 == 0 ? 5 : (NC % 4 == 0 ? 4 : (NC % 3 == 0 ? 3 : 1)));   // planes per batch
    Unroll<0, NC / CH>::run([&](auto C0) {
      constexpr int j0 = decltype(C0)::value * CH;
      double2 gg[CH];
#pragma unroll
      for (int j = 0; j < CH; j++) gg[j] = make_double2(dUs * xk[j0 + j].x, dUs * xk[j0 + j].y);
      if (ku >= 0) {                                                // Phi_s W^(n+e_s), CTA-uniform branch
        double2 v[CH];
        Unroll<0, CH>::run([&](auto J) { constexpr int j = decltype(J)::value; v[j] = ldg2o<(j0 + j) * PL2>(Xu, pol_u); });
#pragma unroll
        for (int j = 0; j < CH; j++) {
          const double psa = (s == 0) ? fma((double)(j0 + j), h1, p1_0) : (s == 1 ? p2 : p3a);
          const double psb = (s == 2) ? p3b : psa;
          gg[j] = fma2(cu, v[j], gg[j]);
          acc[j0 + j].x = fma(psa * pu, v[j].x, acc[j0 + j].x);
          acc[j0 + j].y = fma(psb * pu, v[j].y, acc[j0 + j].y);
        }
      }
      if (kd >= 0) {                                                // n_s Theta_s W^(n-e_s)
        double2 v[CH];
        Unroll<0, CH>::run([&](auto J) { constexpr int j = decltype(J)::value; v[j] = ldg2o<(j0 + j) * PL2>(Xd, pol_d); });
#pragma unroll
        for (int j = 0; j < CH; j++) {
          const double psa = (s == 0) ? fma((double)(j0 + j), h1, p1_0) : (s == 1 ? p2 : p3a);
          const double psb = (s == 2) ? p3b : psa;
          gg[j] = fma2(cd, v[j], gg[j]);
          acc[j0 + j].x = fma(psa * pd, v[j].x, acc[j0 + j].x);
          acc[j0 + j].y = fma(psb * pd, v[j].y, acc[j0 + j].y);
        }
      }
#pragma unroll
      for (int jj = 0; jj < CH; jj++) {
        const int j = j0 + jj;
        if (s == 0) {                                               // D_{p_1} G_1 in scatter form
          if (j >= 1) acc[j - 1] = fma2(wp8, gg[jj], acc[j - 1]);
          if (j + 1 < NC) acc[j + 1] = fma2(-wp8, gg[jj], acc[j + 1]);
          if (j >= 2) acc[j - 2] = fma2(-wp1, gg[jj], acc[j - 2]);
          if (j + 2 < NC) acc[j + 2] = fma2(wp1, gg[jj], acc[j + 2]);
          if (SPLIT > 1) {                                          // segment edges: hand G_1 to the neighbour segment
            if (j < 2) *reinterpret_cast<double2*>(xg + (seg * 4 + j) * PLANE + 2 * tid) = gg[jj];
            if (j >= NC - 2) *reinterpret_cast<double2*>(xg + (seg * 4 + 2 + j - (NC - 2)) * PLANE + 2 * tid) = gg[jj];
          }
        } else if (s == 1) {
          *reinterpret_cast<double2*>(g2 + (jbase + j) * G2_PLANE + (i2 + 2) * G2_ROW + i3) = gg[jj];
        } else if (SHFL3) {                                         // D_{p_3} G_3 from the neighbour lanes of the row
          constexpr int W = P3 / 2;
          const int c = tid % W;
          const double2 own = gg[jj];
          double ly = __shfl_up_sync(0xffffffffu, own.y, 1, W), rx = __shfl_down_sync(0xffffffffu, own.x, 1, W);
          if (c == 0) ly = 0.0;
          if (c == W - 1) rx = 0.0;
          double e3x = own.y - ly, e3y = rx - own.x;
          if (wide) {
            double lx = __shfl_up_sync(0xffffffffu, own.x, 1, W), ry = __shfl_down_sync(0xffffffffu, own.y, 1, W);
            if (c == 0) lx = 0.0;
            if (c == W - 1) ry = 0.0;
            e3x = fma(8.0, e3x, -(rx - lx));
            e3y = fma(8.0, e3y, -(ry - ly));
          }
          acc[j].x = fma(wp, e3x, acc[j].x);
          acc[j].y = fma(wp, e3y, acc[j].y);
        } else {
          *reinterpret_cast<double2*>(g3 + (jbase + j) * G3_PLANE + i2 * G3_ROW + i3 + 2) = gg[jj];
          if (KEEP_G3) g3own[KEEP_G3 ? j : 0] = gg[jj];
        }
      }
    });
    if (NPASS > 1 && s == 0) {                                      // G_1 on the two planes beyond a pass edge
      if (seg == SPLIT - 1 && pass + 1 < NPASS) {
#pragma unroll
        for (int hp = 0; hp < 2; hp++) {
          double2 gg = hp == 0 ? ldg2o<NC * PL2>(Xk, pol_own) : ldg2o<(NC + 1) * PL2>(Xk, pol_own);
          gg = make_double2(dUs * gg.x, dUs * gg.y);
          if (ku >= 0) gg = fma2(cu, hp == 0 ? ldg2o<NC * PL2>(Xu, pol_u) : ldg2o<(NC + 1) * PL2>(Xu, pol_u), gg);
          if (kd >= 0) gg = fma2(cd, hp == 0 ? ldg2o<NC * PL2>(Xd, pol_d) : ldg2o<(NC + 1) * PL2>(Xd, pol_d), gg);
          if (hp == 0) { acc[NC - 1] = fma2(wp8, gg, acc[NC - 1]); acc[NC - 2] = fma2(-wp1, gg, acc[NC - 2]); }
          else acc[NC - 1] = fma2(-wp1, gg, acc[NC - 1]);
        }
      }
      if (seg == 0 && pass > 0) {
        const double2* Xkm = Xk - 2 * PL2;
        const double2* Xum = Xu - 2 * PL2;
        const double2* Xdm = Xd - 2 * PL2;
#pragma unroll
        for (int hp = 0; hp < 2; hp++) {                            // hp = 0: plane -2, hp = 1: plane -1
          double2 gg = hp == 0 ? ldg2o<0>(Xkm, pol_own) : ldg2o<PL2>(Xkm, pol_own);
          gg = make_double2(dUs * gg.x, dUs * gg.y);
          if (ku >= 0) gg = fma2(cu, hp == 0 ? ldg2o<0>(Xum, pol_u) : ldg2o<PL2>(Xum, pol_u), gg);
          if (kd >= 0) gg = fma2(cd, hp == 0 ? ldg2o<0>(Xdm, pol_d) : ldg2o<PL2>(Xdm, pol_d), gg);
          if (hp == 1) { acc[0] = fma2(-wp8, gg, acc[0]); acc[1] = fma2(wp1, gg, acc[1]); }
          else acc[0] = fma2(wp1, gg, acc[0]);
        }
      }
    }
  }
  __syncthreads();
  if (SPLIT > 1) {
    const double wp = wide ? -op.c2[3] : op.c1[3];
    const double wp8 = wide ? 8.0 * wp : wp, wp1 = wide ? wp : 0.0;
    if (seg > 0) {                                                  // G_1 at planes jbase-2, jbase-1
      const double2 gm2 = *reinterpret_cast<const double2*>(xg + ((seg - 1) * 4 + 2) * PLANE + 2 * tid);
      const double2 gm1 = *reinterpret_cast<const double2*>(xg + ((seg - 1) * 4 + 3) * PLANE + 2 * tid);
      acc[0] = fma2(-wp8, gm1, acc[0]);
      acc[0] = fma2(wp1, gm2, acc[0]);
      acc[1] = fma2(wp1, gm1, acc[1]);
    }
    if (seg + 1 < SPLIT) {                                          // G_1 at planes jbase+NC, jbase+NC+1
      const double2 gp0 = *reinterpret_cast<const double2*>(xg + ((seg + 1) * 4 + 0) * PLANE + 2 * tid);
      const double2 gp1 = *reinterpret_cast<const double2*>(xg + ((seg + 1) * 4 + 1) * PLANE + 2 * tid);
      acc[NC - 1] = fma2(wp8, gp0, acc[NC - 1]);
      acc[NC - 1] = fma2(-wp1, gp1, acc[NC - 1]);
      acc[NC - 2] = fma2(-wp1, gp0, acc[NC - 2]);
    }
  }
  {
    const double* c2 = g2 + jbase * G2_PLANE + (i2 + 2) * G2_ROW + i3;
    const double* c3 = g3 + jbase * G3_PLANE + i2 * G3_ROW + i3 + 2;
#pragma unroll
    for (int j = 0; j < NC; j++) {
      const double* a2 = c2 + j * G2_PLANE;
      const double* a3 = c3 + j * G3_PLANE;
      double e2x = 0.0, e2y = 0.0;
      if (!SKIP1) {
        const double2 u1 = *reinterpret_cast<const double2*>(a2 + G2_ROW), d1 = *reinterpret_cast<const double2*>(a2 - G2_ROW);
        e2x = u1.x - d1.x; e2y = u1.y - d1.y;
      }
      double e3x = 0.0, e3y = 0.0;
      double2 lft = make_double2(0.0, 0.0), rgt = lft;
      if (!SHFL3) {
        lft = *reinterpret_cast<const double2*>(a3 - 2); rgt = *reinterpret_cast<const double2*>(a3 + 2);
        // pair (i3, i3+1): neighbours i3-2..i3+3 = lft.x lft.y [own.x own.y] rgt.x rgt.y
        const double2 own = KEEP_G3 ? g3own[KEEP_G3 ? j : 0] : *reinterpret_cast<const double2*>(a3);
        e3x = own.y - lft.y; e3y = rgt.x - own.x;
      }
      if (wide) {
        if (!SKIP1) {
          const double2 u2 = *reinterpret_cast<const double2*>(a2 + 2 * G2_ROW), d2 = *reinterpret_cast<const double2*>(a2 - 2 * G2_ROW);
          e2x = fma(8.0, e2x, -(u2.x - d2.x));
          e2y = fma(8.0, e2y, -(u2.y - d2.y));
        }
        if (!SHFL3) {
          e3x = fma(8.0, e3x, -(rgt.x - lft.x));
          e3y = fma(8.0, e3y, -(rgt.y - lft.y));
        }
      }
      if (!SKIP1) {
        acc[j].x = fma(w2, e2x, acc[j].x);
        acc[j].y = fma(w2, e2y, acc[j].y);
      }
      if (!SHFL3) {
        acc[j].x = fma(w3, e3x, acc[j].x);
        acc[j].y = fma(w3, e3y, acc[j].y);
      }
    }
  }

  // stage combine.  y may alias out (last stage, in place): a thread reads only the cells it writes, and all
  // its reads are issued before its first write.
  if (!y_is_in) {
    const double2* Y = reinterpret_cast<const double2*>(y + boff) + ((size_t)k * cells2 + brick2 + tpart);
    Unroll<0, NC>::run([&](auto J) { constexpr int j = decltype(J)::value; xk[j] = ld2o<j * PL2>(Y, pol_str); });
  }
#pragma unroll
  for (int j = 0; j < NC; j++) acc[j] = make_double2(fma(cc, acc[j].x, a * xk[j].x), fma(cc, acc[j].y, a * xk[j].y));
  double2* O = reinterpret_cast<double2*>(out + boff) + ((size_t)k * cells2 + brick2 + tpart);
  Unroll<0, NC>::run([&](auto J) { constexpr int j = decltype(J)::value; st2o<j * PL2>(O, acc[j], pol_str); });
  __syncthreads();                                                  // shared bricks free for the next pass / brick
  }  // pass
  }  // brick
}

template <int P1, int P2, int P3, int SPLIT, int NPASS>
constexpr int brick3_smem_bytes() {
  return (int)sizeof(double) * ((P2 == 1 ? 0 : (P1 / NPASS) * (P2 + 4) * P3) +
                                (brick3_shfl3(P2, P3, SPLIT) ? 0 : (P1 / NPASS) * P2 * (P3 + 4)) +
                                (SPLIT > 1 ? SPLIT * 4 * P2 * P3 : 0));
}

}  // namespace

#define BRICK3_SPECIALISATIONS(X) X(16, 16, 16, 4, 1, 1) X(16, 16, 16, 2, 2, 1) X(20, 20, 20, 2, 1, 1) X(20, 20, 20, 2, 1, 2) X(12, 12, 12, 2, 2, 1) X(8, 8, 8, 2, 2, 1) X(48, 1, 48, 8, 2, 1) X(48, 1, 48, 16, 2, 1) X(16, 1, 16, 4, 2, 1)

int brick_has_fixed(int M, int P1, int P2, int P3, int split, int minb, int npass) {   // M = 2 arrives as (P1, 1, P2)
  if (M != 3 && M != 2) return 0;
#define X(A, B, C, S, MB, NP) if (P1 == A && P2 == B && P3 == C && split == S && minb == MB && npass == NP) return 1;
  BRICK3_SPECIALISATIONS(X)
#undef X
  return 0;
}

int brick_configure(const BrickPlan& bp, int M) {
  cudaError_t e = cudaErrorInvalidValue;
  if (M != 3 && M != 2) return (int)e;
#define X(A, B, C, S, MB, NP)                                                                             \
  if (bp.P1 == A && bp.P2 == B && bp.P3 == C && bp.split == S && bp.minb == MB && bp.npass == NP)         \
    e = cudaFuncSetAttribute(k_stage_brick3<A, B, C, S, MB, NP>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                             brick3_smem_bytes<A, B, C, S, NP>());
  BRICK3_SPECIALISATIONS(X)
#undef X
  return (int)e;
}

int launch_stage_brick(const DevOp& op, const BrickPlan& bp, const double* in, const double* y, double* out, double a,
                       double c, int nb, size_t slot_stride, cudaStream_t s) {
  dim3 grid((unsigned)(((long long)op.K * op.nqc + bp.bpc - 1) / bp.bpc), nb);
  const int y_is_in = (y == in) ? 1 : 0;
#define X(A, B, C, S, MB, NP)                                                                              \
  if (bp.P1 == A && bp.P2 == B && bp.P3 == C && bp.split == S && bp.minb == MB && bp.npass == NP)          \
    k_stage_brick3<A, B, C, S, MB, NP><<<grid, S * B * C / 2, brick3_smem_bytes<A, B, C, S, NP>(), s>>>(   \
        op, bp, in, y, out, a, c, slot_stride, y_is_in);
  BRICK3_SPECIALISATIONS(X)
#undef X
  return 1;
}
