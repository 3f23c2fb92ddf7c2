// Bulk-copy ("TMA") fed RK-stage kernel (steps a1-a3 of DESIGN.md) for three modes on sm_100a.
//
// Same arithmetic as chfpe_brick.cu (Eq. (8)-(12); G_s combination, scatter-form p_1 stencil, warp
// shuffle p_3 stencil), different data movement.  A brick (all momenta of one (element, q-point)) is cut along p_1 into
// NPART parts of PP planes; one part of one brick is a contiguous run of PP*P2*P3 doubles ("chunk", 16 KB at 16^3 with
// two parts).  A CTA owns one q_3 line of one part.  Every chunk the line needs -- the part of the own brick, of the
// hierarchy neighbours, of the q_1 / q_2 neighbour bricks, of y -- is streamed with 1-D bulk async copies
// (cp.async.bulk, completion on an mbarrier) into a ring of shared-memory slots, in a fixed order that every thread
// can enumerate (one ring slot per chunk kind, so slot, barrier parity and shared address are compile-time constants);
// the warps take turns to refill a slot, one kind late, with the chunk SLOTS places ahead, so there is no producer
// warp (it would be the ninth warp of the CTA and cost 32 registers per thread: warps are allocated in fours).  All threads read each chunk exactly once with LDS.128 and fold it into their accumulators, so no load
// latency is exposed and no
// register is pinned by a load in flight.  Half of the q_3 derivative runs in scatter form along the line the CTA
// marches (RING): the own chunk of brick i_3 is added to the accumulators of bricks i_3+1 and i_3+2, which live in
// registers, so the neighbours i_3-1, i_3-2 are never loaded (14.7 instead of 16.7 chunk loads per brick).  Cutting bricks along p_1 halves the L2 window a lock-step group of elements needs,
// which pays for groups of four linked elements; the p_1 stencil needs G_1 on two planes beyond a part edge, and
// those planes (of the own brick and its up_1 / down_1 neighbours) arrive by three small bulk copies one brick ahead.
#include <type_traits>
#include "chfpe_internal.cuh"

namespace {

// compile-time loop (chunk kinds must be template arguments)
template <int J, int N> struct Unroll {
  template <typename F> __device__ __forceinline__ static void run(F&& f) { f(std::integral_constant<int, J>()); Unroll<J + 1, N>::run(f); }
};
template <int N> struct Unroll<N, N> {
  template <typename F> __device__ __forceinline__ static void run(F&&) {}
};


__device__ __forceinline__ unsigned t_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void t_mbar_init(void* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(t_smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void t_mbar_arrive(void* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(t_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void t_mbar_expect_tx(void* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(t_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void t_mbar_wait(void* bar, unsigned parity) {
  unsigned done;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.b32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(t_smem_u32(bar)), "r"(parity)
        : "memory");
  } while (!done);
}
__device__ __forceinline__ void t_bulk_g2s(void* dst, const void* src, unsigned bytes, void* bar, unsigned long long pol) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
          t_smem_u32(dst)),
      "l"(src), "r"(bytes), "r"(t_smem_u32(bar)), "l"(pol)
      : "memory");
}
// variants on precomputed 32-bit shared-window addresses (no address conversion per call)
__device__ __forceinline__ void a_mbar_arrive(unsigned bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void a_mbar_arrive_if(unsigned bar, bool on) {            // predicated, no branch
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.u32 p, %1, 0;\n\t"
      "@p mbarrier.arrive.shared::cta.b64 _, [%0];\n\t}" ::"r"(bar), "r"((unsigned)on)
      : "memory");
}
__device__ __forceinline__ void a_mbar_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ unsigned a_mbar_try(unsigned bar, unsigned parity) {   // may suspend briefly; 1 = phase complete
  unsigned done;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.b32 %0, 1, 0, p;\n\t}"
      : "=r"(done)
      : "r"(bar), "r"(parity)
      : "memory");
  return done;
}
__device__ __forceinline__ unsigned a_mbar_test(unsigned bar, unsigned parity) {  // never suspends
  unsigned done;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.b32 %0, 1, 0, p;\n\t}"
      : "=r"(done)
      : "r"(bar), "r"(parity)
      : "memory");
  return done;
}
__device__ __forceinline__ void a_mbar_wait(unsigned bar, unsigned parity) {
  while (!a_mbar_try(bar, parity)) {}
}
__device__ __forceinline__ void a_bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar, unsigned long long pol) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst),
      "l"(src), "r"(bytes), "r"(bar), "l"(pol)
      : "memory");
}
__device__ __forceinline__ double2 a_lds2(unsigned addr) {
  double2 v;
  asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
  return v;
}
__device__ __forceinline__ void t_prefetch_l2(const void* src, unsigned bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ unsigned long long t_policy(int kind) {   // 0 normal, 1 evict_first, 2 evict_last
  unsigned long long p;
  if (kind == 1) asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  else if (kind == 2) asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  else asm("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ double2 t_ldg2(const double2* p, unsigned long long pol) {
  double2 v;
  asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol));
  return v;
}
__device__ __forceinline__ void t_st2(double2* p, double2 v, unsigned long long pol) {
  asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}
__device__ __forceinline__ double2 t_fma2(double c, double2 a, double2 b) { return make_double2(fma(c, a.x, b.x), fma(c, a.y, b.y)); }
__device__ __forceinline__ double2 t_fma2(double2 c, double2 a, double2 b) { return make_double2(fma(c.x, a.x, b.x), fma(c.y, a.y, b.y)); }

__host__ __device__ constexpr bool tma_shfl3(int p2, int p3) {       // p_3 rows of P3/2 pairs tile a warp
  return (p3 % 2 == 0) && (32 % (p3 / 2) == 0) && ((p2 * p3 / 2) % 32 == 0);
}

template <int P1, int P2, int P3, int NPART, int NSEG, int SLOTS, bool RING>
struct TmaCfg {
  static_assert(P3 % 2 == 0 && P1 % (NPART * NSEG) == 0 && P1 / (NPART * NSEG) >= 2, "unsupported brick shape");
  static constexpr int PLANE = P2 * P3, PL2 = PLANE / 2, PP = P1 / NPART, NC = PP / NSEG;
  static constexpr int NACT = NSEG * PL2;                          // threads that own cells
  static constexpr int NT = (NACT + 31) / 32 * 32, NW = NT / 32;
  static constexpr unsigned CHUNK = PP * PLANE * (unsigned)sizeof(double);
  static constexpr bool SHFL3 = tma_shfl3(P2, P3);
  static constexpr int G2_ROW = P3, G2_PLANE = (P2 == 1) ? 0 : (P2 + 4) * P3;       // G_2[plane][i2+2][i3]
  // p_3 stencil: neighbour lanes (a thread owns a pair of p_3-adjacent cells).  SHFL3: the rows of P3/2 pairs tile a warp.
  // Otherwise a row may cross a warp boundary: lane 0 / 31 of every warp leave their G_3 pairs in a small edge buffer and
  // the thread on the other side adds the missing terms after the exchange barrier (the stencil is linear).
  static constexpr int EB = SHFL3 ? 0 : NW * 2 * NC * 2;                            // doubles: G_3 pair [warp][side][plane]
  static constexpr int XG = (NSEG > 1) ? (NSEG - 1) * 4 * PLANE : 0;                // G_1 planes next to a segment edge
  static_assert(NPART <= 2, "a part has at most one edge inside the brick (the halo planes share one ring slot)");
  // Chunk kinds of one step (= one brick of the line), consumed in this order; kind e always uses ring slot e % SLOTS,
  // so slots, barrier parities and shared addresses are compile-time constants.  A kind that does not exist for a brick
  // (ghost bricks R9, missing hierarchy neighbours, the q_3 kinds the ring replaces) moves no data but still flips
  // its barriers.
  //   0 own part | 1, 2 up / down neighbour element along mode 1 | 3 the two planes beyond the part edge of 0, 1, 2
  //   (three pieces in one slot; NPART = 2 only) | 4..7 up / down neighbour elements along modes 2, 3 |
  //   8+4s+d neighbour brick along q_s (s = 0, 1), d = 0..3: +1, -1, +2, -2 | 16+d neighbour brick along q_3 (with
  //   the ring only d = 0, 1 meaning +1, +2) | NK-1 y
  static constexpr int NK = RING ? 20 : 24, USES = NK / SLOTS;     // uses of a slot per step
  static_assert(3 * 2 * PLANE <= PP * PLANE, "halo pieces must fit a slot");
  static_assert(NK % SLOTS == 0, "the slot of a kind must not depend on the step");
  static constexpr int MAXQ3 = 64;                                 // longest q_3 line (dU/dq_s table of the line)
  static constexpr size_t SMEM = (size_t)SLOTS * CHUNK + sizeof(double) * (PP * G2_PLANE + EB + XG) +
                                 16 * SLOTS + 16 + 8 * NK + 8 * 3 * MAXQ3 + 16;
  static constexpr int MINB = (2 * (SMEM + 1024) <= 227 * 1024 && 2 * NT <= 1024) ? 2 : 1;
};

// one line of the sweep: {element, i_q1 | i_q2 << 10 | part << 20, own-mask (as BrickId::own), bit d: the q_2 neighbour
// d (+1, -1, +2, -2) lies outside the q_2 chunk of the sweep, i.e. outside the L2 window}
struct TmaLine { int k, iq1, iq2, part, own, q2out; };
__device__ __forceinline__ TmaLine decode_line(const int4* lines, long long L) {
  const int4 t = __ldg(lines + L);
  TmaLine l;
  l.k = t.x; l.iq1 = t.y & 1023; l.iq2 = (t.y >> 10) & 1023; l.part = t.y >> 20; l.own = t.z; l.q2out = t.w;
  return l;
}

template <int E> using KindC = std::integral_constant<int, E>;

template <int P1, int P2, int P3, int NPART, int NSEG, int SLOTS, bool RING>
__global__ void __launch_bounds__(TmaCfg<P1, P2, P3, NPART, NSEG, SLOTS, RING>::NT, TmaCfg<P1, P2, P3, NPART, NSEG, SLOTS, RING>::MINB)
k_stage_tma(DevOp op, BrickPlan bp, const double* __restrict__ in, const double* y, double* out, double a, double cc,
            size_t slot_stride) {
  using C = TmaCfg<P1, P2, P3, NPART, NSEG, SLOTS, RING>;
  constexpr int PLANE = C::PLANE, PL2 = C::PL2, PP = C::PP, NC = C::NC, NK = C::NK;
  constexpr bool SKIP1 = (P2 == 1);                                 // two-mode view: middle mode has one point
  constexpr size_t BRICK = (size_t)P1 * PLANE;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char* ring = smem_raw;
  double* g2 = reinterpret_cast<double*>(smem_raw + (size_t)SLOTS * C::CHUNK);
  double* eb = g2 + PP * C::G2_PLANE;
  double* xg = eb + C::EB;
  unsigned long long* full = reinterpret_cast<unsigned long long*>(xg + C::XG);       // data of a slot has landed
  unsigned long long* empty = full + SLOTS;                                           // all warps have released a slot
  unsigned long long* xbar = empty + SLOTS;                                           // exchange planes: [0] written, [1] read
  const double** ent = reinterpret_cast<const double**>(xbar + 2);                    // source of every kind at step 0
  double* sdu = reinterpret_cast<double*>(ent + NK);                                  // dU/dq_s at the q-points of the line
  const unsigned ring_a = t_smem_u32(ring), full_a = t_smem_u32(full), empty_a = t_smem_u32(empty), xbar_a = t_smem_u32(xbar);

  const int t = threadIdx.x;
  const TmaLine ln = decode_line(bp.lines, blockIdx.x);
  const int k = ln.k, part = ln.part;
  const int n1 = op.n[0], n2 = op.n[1], n3 = op.n[2];
  const size_t boff = (size_t)blockIdx.y * slot_stride;
  const double* X = in + boff;
  const long long ql0 = ((long long)ln.iq1 * n2 + ln.iq2) * n3;     // q index of i_q3 = 0
  const size_t pofs = (size_t)part * PP * PLANE;                    // first plane of this part inside a brick
  const int kup0 = __ldg(op.up + 3 * k + 0), kup1 = __ldg(op.up + 3 * k + 1), kup2 = __ldg(op.up + 3 * k + 2);
  const int kdn0 = __ldg(op.dn + 3 * k + 0), kdn1 = __ldg(op.dn + 3 * k + 1), kdn2 = __ldg(op.dn + 3 * k + 2);
  const int kupa[3] = {kup0, SKIP1 ? -1 : kup1, kup2};
  const int kdna[3] = {kdn0, SKIP1 ? -1 : kdn1, kdn2};

  // kind of the up (dir 0) / down (dir 1) neighbour element along mode s
  auto hk = [](int s, int dir) { return (s == 0 ? 1 : 2 + 2 * s) + dir; };
  unsigned mask_line = 1u | (1u << (NK - 1));                       // kinds that exist for every brick of the line
  if (NPART > 1) mask_line |= 1u << 3;
#pragma unroll
  for (int s = 0; s < 3; s++) {
    if (kupa[s] >= 0) mask_line |= 1u << hk(s, 0);
    if (kdna[s] >= 0) mask_line |= 1u << hk(s, 1);
  }
#pragma unroll
  for (int d = 0; d < 4; d++) {
    const int off = (d == 0) ? 1 : (d == 1 ? -1 : (d == 2 ? 2 : -2));
    if (ln.iq1 + off >= 0 && ln.iq1 + off < n1) mask_line |= 1u << (8 + d);
    if (!SKIP1 && ln.iq2 + off >= 0 && ln.iq2 + off < n2) mask_line |= 1u << (12 + d);
  }
  auto step_mask = [&](int m) -> unsigned {                         // RING: x_{m-1}, x_{m-2} reach brick m through registers
    unsigned mk = mask_line;
    if (RING) {
      if (m + 1 < n3) mk |= 1u << 16;
      if (m + 2 < n3) mk |= 1u << 17;
    } else {
      if (m + 1 < n3) mk |= 1u << 16;
      if (m >= 1) mk |= 1u << 17;
      if (m + 2 < n3) mk |= 1u << 18;
      if (m >= 2) mk |= 1u << 19;
    }
    return mk;
  };
  unsigned pol_bits = (1u << (NK - 1)) | (1u << 3);                 // kinds whose lines are touched once: evict_first
#pragma unroll
  for (int s = 0; s < 3; s++) {
    if (!((ln.own >> (2 * s)) & 1)) pol_bits |= 1u << hk(s, 0);
    if (!((ln.own >> (2 * s + 1)) & 1)) pol_bits |= 1u << hk(s, 1);
  }
  const unsigned long long pol_own = t_policy((bp.l2mode & 2) ? 2 : 0);
  const unsigned long long pol_str = t_policy((bp.l2mode & 1) ? 1 : 0);
  // load kind e of brick m into its slot, or (kind absent) complete the slot's barrier without data  (one thread)
  constexpr unsigned HB = 2 * PLANE * sizeof(double);               // one halo piece: two planes
  const long long hofs = (part > 0 ? -2 : PP) * (long long)PLANE;   // NPART = 2: part 1 looks below itself, part 0 above
  auto issue = [&](int m, int e, unsigned mk) {
    const unsigned fb = full_a + 8 * (e % SLOTS), dst = ring_a + (e % SLOTS) * C::CHUNK;
    if (!((mk >> e) & 1u)) {
      a_mbar_arrive(fb);
    } else if (NPART > 1 && e == 3) {                               // planes beyond the part edge: own, up_1, down_1
      a_mbar_expect_tx(fb, HB * (1 + ((mk >> 1) & 1u) + ((mk >> 2) & 1u)));
      a_bulk_g2s(dst, ent[0] + (size_t)m * BRICK + hofs, HB, fb, pol_str);
      if ((mk >> 1) & 1u) a_bulk_g2s(dst + HB, ent[1] + (size_t)m * BRICK + hofs, HB, fb, pol_str);
      if ((mk >> 2) & 1u) a_bulk_g2s(dst + 2 * HB, ent[2] + (size_t)m * BRICK + hofs, HB, fb, pol_str);
    } else {
      a_mbar_expect_tx(fb, C::CHUNK);
      a_bulk_g2s(dst, ent[e] + (size_t)m * BRICK, C::CHUNK, fb, ((pol_bits >> e) & 1u) ? pol_str : pol_own);
    }
  };

  if (t == 0) {
    for (int s = 0; s < SLOTS; s++) { t_mbar_init(full + s, 1); t_mbar_init(empty + s, C::NW); }
    t_mbar_init(xbar, C::NW); t_mbar_init(xbar + 1, C::NW);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    const double* Xk = X + (size_t)k * op.cells + pofs + (size_t)ql0 * BRICK;
    for (int e = 0; e < NK; e++) ent[e] = Xk;
    ent[NK - 1] = y + boff + (size_t)k * op.cells + pofs + (size_t)ql0 * BRICK;
#pragma unroll
    for (int s = 0; s < 3; s++) {
      ent[hk(s, 0)] = X + (size_t)(kupa[s] >= 0 ? kupa[s] : k) * op.cells + pofs + (size_t)ql0 * BRICK;
      ent[hk(s, 1)] = X + (size_t)(kdna[s] >= 0 ? kdna[s] : k) * op.cells + pofs + (size_t)ql0 * BRICK;
    }
#pragma unroll
    for (int d = 0; d < 4; d++) {
      const int off = (d == 0) ? 1 : (d == 1 ? -1 : (d == 2 ? 2 : -2));
      ent[8 + d] = Xk + off * op.st[0];
      ent[12 + d] = Xk + off * op.st[1];
      if (!RING) ent[16 + d] = Xk + off * op.st[2];
    }
    if (RING) { ent[16] = Xk + op.st[2]; ent[17] = Xk + 2 * op.st[2]; }
    const unsigned mk0 = step_mask(0);
    for (int e = 0; e < SLOTS; e++) issue(0, e, mk0);               // fill the ring
  }
  for (int i = t; i < 3 * n3; i += C::NT) {
    const int s = i / n3, m = i - s * n3;
    sdu[s * C::MAXQ3 + m] = __ldg(op.dU[s] + ql0 + m);
  }
  // ghost rows / columns of the exchange planes stay zero for the whole kernel
  for (int i = t; i < (SKIP1 ? 0 : PP * 4 * P3); i += C::NT) {
    const int pl = i / (4 * P3), rr = i - pl * (4 * P3), row = rr / P3, col = rr - row * P3;
    g2[pl * C::G2_PLANE + (row < 2 ? row : P2 + row) * C::G2_ROW + col] = 0.0;
  }
  __syncthreads();

  const bool active = t < C::NACT;
  const int tt = active ? t : 0;
  const int seg = (NSEG == 1) ? 0 : tt / PL2;
  const int tid = tt - seg * PL2;                                   // pair index inside the plane
  const int jbase = seg * NC;                                       // first plane (inside the part) of this thread
  const int i2 = tid / (P3 / 2), i3 = 2 * (tid - i2 * (P3 / 2));
  const int lane = t & 31, warp = __shfl_sync(0xffffffffu, t >> 5, 0);   // (warp-uniform by construction)
  unsigned my_a = ring_a + (unsigned)(jbase * PL2 + tid) * 16;         // this thread's first pair inside slot 0
  asm volatile("" : "+r"(my_a));                                     // (kept in a register: not rematerialised per chunk)
  const double h1 = op.h[3];
  const double p1_0 = op.x0[3] + (part * PP + jbase) * h1;
  const double p2 = op.x0[4] + i2 * op.h[4];
  const double p3a = op.x0[5] + i3 * op.h[5], p3b = op.x0[5] + (i3 + 1) * op.h[5];
  // CENTRAL4 weights: D f_i = [8 (f_{i+1} - f_{i-1}) - (f_{i+2} - f_{i-2})] / (12 h)
  const double w1p = -op.c2[3], w2p = -op.c2[4], w3p = -op.c2[5];   // 1 / (12 h) of p_1, p_2, p_3
  const double wp8 = 8.0 * w1p, wp1 = w1p;
  const double Gam = __ldg(op.Gamma + k);
  double Vp[3], cdf[3];
#pragma unroll
  for (int s = 0; s < 2; s++) {
    const double qs = op.x0[s] + (s == 0 ? ln.iq1 : ln.iq2) * op.h[s];
    Vp[s] = fma(op.VSL[s], qs, op.VLL[s]);
  }
#pragma unroll
  for (int s = 0; s < 3; s++) cdf[s] = __ldg(op.nvec + 3 * k + s) * op.cdn[s];
  const bool do_lo = NPART > 1 && seg == 0 && part > 0;             // this thread adds G_1 of the planes below / above the part
  const bool do_hi = NPART > 1 && seg == NSEG - 1 && part + 1 < NPART;

  int m = 0;
  // (masks are the same in every thread; the shuffle tells the compiler so: uniform branches, no reconvergence code)
  unsigned mask = __shfl_sync(0xffffffffu, step_mask(0), 0), maskn = __shfl_sync(0xffffffffu, step_mask(1), 0), mpar = 0;
  // barrier parity of use (step parity mp, kind E) of slot E % SLOTS
  auto parity = [&](int E, unsigned mp) -> unsigned { return ((unsigned)(E / SLOTS) & 1u) ^ ((C::USES & 1) ? mp : 0u); };
  // Refill duty for use (mm, EP): wait until every warp has let go of the slot, then load its next user -- kind
  // EP + SLOTS of the same brick, or kind EP + SLOTS - NK of the next one.  Called one kind late (the slot is almost
  // always free by then) by warp EP % NW, so a warp can block on every NW-th kind only.  (Letting the last arriver
  // refill -- mbarrier.pending_count of its own arrive -- was measured slower, 4.5 vs 3.2 ms: the last warp is the
  // slowest one and gets the extra work.)
  auto duty = [&](auto KEP, int mm, unsigned mp, unsigned mk_same, unsigned mk_next) {
    constexpr int EP = decltype(KEP)::value;
    constexpr int E2 = (EP + SLOTS < NK) ? EP + SLOTS : EP + SLOTS - NK;
    const int m2 = (EP + SLOTS < NK) ? mm : mm + 1;
    if (mm < 0 || m2 >= n3) return;
    a_mbar_wait(empty_a + 8 * (EP % SLOTS), parity(EP, mp));
    if (lane == 0) issue(m2, E2, (EP + SLOTS < NK) ? mk_same : mk_next);
  };
  // consume kind E of the current brick: body(address of this thread's first pair in the slot) if the kind exists
  auto chunk = [&](auto KE, auto&& body) {
    constexpr int E = decltype(KE)::value;
    // (an absent kind is waited for as well: its barrier is completed, without data, only after every warp has
    // released the slot's previous user, which keeps a fast warp from arriving twice in one phase of `empty`)
    a_mbar_wait(full_a + 8 * (E % SLOTS), parity(E, mpar));
    if ((mask >> E) & 1u) body(my_a + (E % SLOTS) * C::CHUNK);
    __syncwarp();
    a_mbar_arrive_if(empty_a + 8 * (E % SLOTS), lane == 0);
    constexpr int EP = (E + NK - 1) % NK;                           // the kind before this one: its slot gets its next user now
    if (warp == EP % C::NW) {
      if (E == 0) duty(KindC<EP>(), m - 1, mpar ^ 1u, 0u, mask);    // last kind of the previous brick
      else duty(KindC<EP>(), m, mpar, mask, maskn);
    }
  };

  // RING: accumulators of bricks m, m+1, m+2 (the last one only while brick m is processed)
  constexpr int NA = RING ? 3 : 1;
  double2 A[NA][NC];
#pragma unroll
  for (int r = 0; r < NA; r++)
#pragma unroll
    for (int j = 0; j < NC; j++) A[r][j] = make_double2(0.0, 0.0);
  double2(&acc)[NC] = A[0];

  double2* Ob = reinterpret_cast<double2*>(out + boff + (size_t)k * op.cells + pofs + (size_t)ql0 * BRICK + (size_t)jbase * PLANE + 2 * tid);

#pragma unroll 1
  for (; m < n3; m++) {
    if (t == 0 && m + 1 < n3) {                                     // HBM-sourced data of brick m+1 -> L2
      const size_t bn = (size_t)(m + 1) * BRICK;
      if ((mask_line >> 10) & 1u) t_prefetch_l2(ent[10] + bn, C::CHUNK);       // first touch of the brick two q_1 planes ahead
#pragma unroll
      for (int e = 1; e < 8; e++)
        if (e != 3 && ((mask_line >> e) & (pol_bits >> e) & 1u)) t_prefetch_l2(ent[e] + bn, C::CHUNK);
#pragma unroll
      for (int d = 0; d < 4; d++)
        if ((mask_line >> (12 + d)) & (ln.q2out >> d) & 1u) t_prefetch_l2(ent[12 + d] + bn, C::CHUNK);
      t_prefetch_l2(ent[NK - 1] + bn, C::CHUNK);
      if (NPART > 1) {
#pragma unroll
        for (int e = 0; e < 3; e++)
          if ((mask_line >> e) & 1u) t_prefetch_l2(ent[e] + bn + hofs, HB);
      }
    }
    double2 x[NC];
    chunk(KindC<0>(), [&](unsigned S) {
#pragma unroll
      for (int j = 0; j < NC; j++) x[j] = a_lds2(S + j * (PL2 * 16));
    });
    const double c3q = op.c2[2] * op.inv_mass[2];                   // -(1/m_3) / (12 h_q3)
    if (RING) {                                                     // -(p_3/m_3) dW/dq_3: brick m+1 sees x_m at -1 (weight -8),
      const double2 c3 = make_double2(c3q * p3a, c3q * p3b);       // brick m+2 at -2 (weight +1)
      const double2 c3m8 = make_double2(-8.0 * c3.x, -8.0 * c3.y);
#pragma unroll
      for (int j = 0; j < NC; j++) {
        A[1][j] = t_fma2(c3m8, x[j], A[1][j]);
        A[2][j] = make_double2(c3.x * x[j].x, c3.y * x[j].y);
      }
    }
#pragma unroll
    for (int j = 0; j < NC; j++) acc[j] = t_fma2(-Gam, x[j], acc[j]);
    Vp[2] = fma(op.VSL[2], op.x0[2] + m * op.h[2], op.VLL[2]);
#pragma unroll
    for (int s = 0; s < 3; s++) {
      const double dUs = sdu[s * C::MAXQ3 + m];
      const double cu = Vp[s], cd = cdf[s] * Vp[s];
      const double pu = cu * op.kup[s], pd = cd * op.kdn[s];
      double2 g[NC];
#pragma unroll
      for (int j = 0; j < NC; j++) g[j] = make_double2(dUs * x[j].x, dUs * x[j].y);
      Unroll<0, 2>::run([&](auto DIR) {                             // Phi_s W^(n+e_s) (Eq. 11), then n_s Theta_s W^(n-e_s) (Eq. 12, R1)
        constexpr int dir = decltype(DIR)::value;
        const double cg = dir ? cd : cu, pg = dir ? pd : pu;
        auto body = [&](unsigned S) {
#pragma unroll
          for (int j = 0; j < NC; j++) {
            const double2 v = a_lds2(S + j * (PL2 * 16));
            const double psa = (s == 0) ? fma((double)j, h1, p1_0) : (s == 1 ? p2 : p3a);
            const double psb = (s == 2) ? p3b : psa;
            g[j] = t_fma2(cg, v, g[j]);
            acc[j].x = fma(psa * pg, v.x, acc[j].x);
            acc[j].y = fma(psb * pg, v.y, acc[j].y);
          }
        };
        if (s == 0) chunk(KindC<1 + dir>(), body);
        else if (s == 1) chunk(KindC<4 + dir>(), body);
        else chunk(KindC<6 + dir>(), body);
      });
      if (SKIP1 && s == 1) continue;
      if (s == 0) {                                                 // D_{p_1} G_1 in scatter form
#pragma unroll
        for (int j = 0; j < NC; j++) {
          if (j >= 1) acc[j - 1] = t_fma2(wp8, g[j], acc[j - 1]);
          if (j + 1 < NC) acc[j + 1] = t_fma2(-wp8, g[j], acc[j + 1]);
          if (j >= 2) acc[j - 2] = t_fma2(-wp1, g[j], acc[j - 2]);
          if (j + 2 < NC) acc[j + 2] = t_fma2(wp1, g[j], acc[j + 2]);
        }
        chunk(KindC<3>(), [&](unsigned S) {                         // G_1 on the two planes beyond the part edge
          if (!(do_lo || do_hi)) return;
          const unsigned H = ring_a + (3 % SLOTS) * C::CHUNK + tid * 16;
          double2 gh[2];
#pragma unroll
          for (int e = 0; e < 2; e++) {
            const double2 hx = a_lds2(H + e * (PL2 * 16));
            gh[e] = make_double2(dUs * hx.x, dUs * hx.y);
            if (kupa[0] >= 0) gh[e] = t_fma2(cu, a_lds2(H + HB + e * (PL2 * 16)), gh[e]);
            if (kdna[0] >= 0) gh[e] = t_fma2(cd, a_lds2(H + 2 * HB + e * (PL2 * 16)), gh[e]);
          }
          if (do_lo) {                                              // planes -2, -1 below the part
            acc[0] = t_fma2(wp1, gh[0], acc[0]);
            acc[0] = t_fma2(-wp8, gh[1], acc[0]);
            acc[1] = t_fma2(wp1, gh[1], acc[1]);
          } else {                                                  // planes PP, PP+1 above the part
            acc[NC - 1] = t_fma2(wp8, gh[0], acc[NC - 1]);
            acc[NC - 2] = t_fma2(-wp1, gh[0], acc[NC - 2]);
            acc[NC - 1] = t_fma2(-wp1, gh[1], acc[NC - 1]);
          }
        });
        // exchange planes of the previous brick are free: split-phase barrier, every warp arrived on it when it had read
        // them (end of the previous brick), four chunk kinds ago
        if (m > 0) a_mbar_wait(xbar_a + 8, (unsigned)(m - 1) & 1u);
        if (NSEG > 1 && active) {                                   // planes next to a segment edge -> neighbour segment
#pragma unroll
          for (int j = 0; j < NC; j++) {
            if (j >= NC - 2 && seg + 1 < NSEG) *reinterpret_cast<double2*>(xg + (seg * 4 + j - (NC - 2)) * PLANE + 2 * tid) = g[j];
            if (j < 2 && seg > 0) *reinterpret_cast<double2*>(xg + ((seg - 1) * 4 + 2 + j) * PLANE + 2 * tid) = g[j];
          }
        }
      } else if (s == 1) {
        if (active) {
#pragma unroll
          for (int j = 0; j < NC; j++)
            *reinterpret_cast<double2*>(g2 + (jbase + j) * C::G2_PLANE + (i2 + 2) * C::G2_ROW + i3) = g[j];
        }
      } else {                                                      // D_{p_3} G_3 from the neighbour lanes of the row
        constexpr int W = P3 / 2, SW = C::SHFL3 ? W : 32;
        const int c = tid % W;
        const bool nol = c == 0 || (!C::SHFL3 && lane == 0), nor = c == W - 1 || (!C::SHFL3 && lane == 31);
#pragma unroll
        for (int j = 0; j < NC; j++) {
          const double2 own = g[j];
          double ly = __shfl_up_sync(0xffffffffu, own.y, 1, SW), rx = __shfl_down_sync(0xffffffffu, own.x, 1, SW);
          double lx = __shfl_up_sync(0xffffffffu, own.x, 1, SW), ry = __shfl_down_sync(0xffffffffu, own.y, 1, SW);
          if (nol) { ly = 0.0; lx = 0.0; }
          if (nor) { rx = 0.0; ry = 0.0; }
          const double e3x = fma(8.0, own.y - ly, -(rx - lx));
          const double e3y = fma(8.0, rx - own.x, -(ry - ly));
          acc[j].x = fma(w3p, e3x, acc[j].x);
          acc[j].y = fma(w3p, e3y, acc[j].y);
          if (!C::SHFL3 && active && (lane == 0 || lane == 31))     // for the neighbour in the next / previous warp
            *reinterpret_cast<double2*>(eb + ((warp * 2 + (lane == 31)) * NC + j) * 2) = own;
        }
      }
    }
    __syncwarp();
    a_mbar_arrive_if(xbar_a, lane == 0);                            // this warp's G_2 / G_3 / segment-edge G_1 are written
    // ---- -(p_s/m_s) dW/dq_s: one chunk per existing neighbour brick (q_3: only x_{m+1}, x_{m+2} with the ring) ----
    Unroll<0, (RING ? 10 : 12)>::run([&](auto SD) {
      constexpr int sd = decltype(SD)::value, s = sd / 4;
      constexpr int d = (RING && s == 2) ? 2 * (sd % 4) : sd % 4;   // ring: kinds 16, 17 are the +1 and +2 neighbours
      const double wd = op.cqw[s][d];                               // host-tabulated: one multiply per coefficient here
      chunk(KindC<8 + sd>(), [&](unsigned S) {
#pragma unroll
        for (int j = 0; j < NC; j++) {
          const double2 v = a_lds2(S + j * (PL2 * 16));
          const double ca = (s == 0) ? wd * fma((double)j, h1, p1_0) : (s == 1 ? wd * p2 : wd * p3a);
          const double cb = (s == 2) ? wd * p3b : ca;
          acc[j].x = fma(ca, v.x, acc[j].x);
          acc[j].y = fma(cb, v.y, acc[j].y);
        }
      });
    });
    if (RING) { chunk(KindC<18>(), [&](unsigned) {}); }             // (unused kind: keeps NK a multiple of SLOTS)
    else { chunk(KindC<20>(), [&](unsigned) {}); chunk(KindC<21>(), [&](unsigned) {}); chunk(KindC<22>(), [&](unsigned) {}); }
    a_mbar_wait(xbar_a, (unsigned)m & 1u);                          // G_2 / G_3 / segment-edge G_1 of every warp complete
    if (NSEG > 1) {
      if (seg > 0) {                                                // G_1 at planes jbase-2, jbase-1
        const double2 gm2 = *reinterpret_cast<const double2*>(xg + ((seg - 1) * 4 + 0) * PLANE + 2 * tid);
        const double2 gm1 = *reinterpret_cast<const double2*>(xg + ((seg - 1) * 4 + 1) * PLANE + 2 * tid);
        acc[0] = t_fma2(-wp8, gm1, acc[0]);
        acc[0] = t_fma2(wp1, gm2, acc[0]);
        acc[1] = t_fma2(wp1, gm1, acc[1]);
      }
      if (seg + 1 < NSEG) {                                         // G_1 at planes jbase+NC, jbase+NC+1
        const double2 gp0 = *reinterpret_cast<const double2*>(xg + (seg * 4 + 2) * PLANE + 2 * tid);
        const double2 gp1 = *reinterpret_cast<const double2*>(xg + (seg * 4 + 3) * PLANE + 2 * tid);
        acc[NC - 1] = t_fma2(wp8, gp0, acc[NC - 1]);
        acc[NC - 1] = t_fma2(-wp1, gp1, acc[NC - 1]);
        acc[NC - 2] = t_fma2(-wp1, gp0, acc[NC - 2]);
      }
    }
    {
      const double* c2 = g2 + jbase * C::G2_PLANE + (i2 + 2) * C::G2_ROW + i3;
#pragma unroll
      for (int j = 0; j < NC; j++) {
        if (!SKIP1) {
          const double* a2 = c2 + j * C::G2_PLANE;
          const double2 u1 = *reinterpret_cast<const double2*>(a2 + C::G2_ROW), d1 = *reinterpret_cast<const double2*>(a2 - C::G2_ROW);
          const double2 u2 = *reinterpret_cast<const double2*>(a2 + 2 * C::G2_ROW), d2 = *reinterpret_cast<const double2*>(a2 - 2 * C::G2_ROW);
          acc[j].x = fma(w2p, fma(8.0, u1.x - d1.x, -(u2.x - d2.x)), acc[j].x);
          acc[j].y = fma(w2p, fma(8.0, u1.y - d1.y, -(u2.y - d2.y)), acc[j].y);
        }
      }
      if (!C::SHFL3 && active) {                                    // the row continues in the previous / next warp
        constexpr int W = P3 / 2;
        const int c = tid % W;
        if (lane == 0 && c != 0) {                                  // pair (i3-2, i3-1): -8 ly + lx on x, + ly on y
#pragma unroll
          for (int j = 0; j < NC; j++) {
            const double2 l = *reinterpret_cast<const double2*>(eb + (((warp - 1) * 2 + 1) * NC + j) * 2);
            acc[j].x = fma(w3p, fma(-8.0, l.y, l.x), acc[j].x);
            acc[j].y = fma(w3p, l.y, acc[j].y);
          }
        }
        if (lane == 31 && c != W - 1) {                             // pair (i3+2, i3+3): - rx on x, 8 rx - ry on y
#pragma unroll
          for (int j = 0; j < NC; j++) {
            const double2 r = *reinterpret_cast<const double2*>(eb + (((warp + 1) * 2 + 0) * NC + j) * 2);
            acc[j].x = fma(w3p, -r.x, acc[j].x);
            acc[j].y = fma(w3p, fma(8.0, r.x, -r.y), acc[j].y);
          }
        }
      }
    }
    __syncwarp();
    a_mbar_arrive_if(xbar_a + 8, lane == 0);                        // this warp has read the exchange planes
    chunk(KindC<NK - 1>(), [&](unsigned S) {                        // stage combine: out = a y + c F
      double2* O = Ob + (size_t)m * (BRICK / 2);
#pragma unroll
      for (int j = 0; j < NC; j++) {
        const double2 yv = a_lds2(S + j * (PL2 * 16));
        if (active) t_st2(O + j * PL2, make_double2(fma(cc, acc[j].x, a * yv.x), fma(cc, acc[j].y, a * yv.y)), pol_str);
      }
    });
#pragma unroll
    for (int j = 0; j < NC; j++) {                                  // the line advances by one brick
      if (RING) { A[0][j] = A[1][j]; A[1][j] = A[2][j]; }
      else A[0][j] = make_double2(0.0, 0.0);
    }
    mask = maskn;
    maskn = __shfl_sync(0xffffffffu, step_mask(m + 2), 0);
    mpar ^= 1u;
  }
}

}  // namespace

// (P1, P2, P3, NPART, NSEG, SLOTS, RING)
#define TMA_SPECIALISATIONS(X) \
  X(16, 16, 16, 2, 2, 5, true) X(16, 16, 16, 2, 2, 4, true) X(16, 16, 16, 2, 2, 4, false) X(16, 16, 16, 1, 4, 5, true) X(16, 16, 16, 1, 4, 4, true) \
  X(8, 8, 8, 1, 2, 5, true) X(8, 8, 8, 1, 2, 4, true) X(8, 8, 8, 1, 2, 4, false) X(12, 12, 12, 2, 3, 5, true) X(12, 12, 12, 2, 3, 4, true) \
  X(20, 20, 20, 2, 2, 5, true) X(20, 20, 20, 2, 2, 4, true) X(20, 20, 20, 2, 2, 4, false)

int tma_has_fixed(int M, int P1, int P2, int P3, int npart, int nseg, int slots, int ring) {
  if (M != 3) return 0;
#define X(A, B, C, NP, NS, SL, R) if (P1 == A && P2 == B && P3 == C && npart == NP && nseg == NS && slots == SL && (ring != 0) == R) return 1;
  TMA_SPECIALISATIONS(X)
#undef X
  return 0;
}

int tma_configure(const BrickPlan& bp) {
  cudaError_t e = cudaErrorInvalidValue;
#define X(A, B, C, NP, NS, SL, R)                                                                                  \
  if (bp.P1 == A && bp.P2 == B && bp.P3 == C && bp.tma_npart == NP && bp.tma_nseg == NS && bp.tma_slots == SL &&   \
      (bp.tma_ring != 0) == R)                                                                                     \
    e = cudaFuncSetAttribute(k_stage_tma<A, B, C, NP, NS, SL, R>, cudaFuncAttributeMaxDynamicSharedMemorySize,     \
                             (int)TmaCfg<A, B, C, NP, NS, SL, R>::SMEM);
  TMA_SPECIALISATIONS(X)
#undef X
  return (int)e;
}

int launch_stage_tma(const DevOp& op, const BrickPlan& bp, const double* in, const double* y, double* out, double a,
                     double c, int nb, size_t slot_stride, cudaStream_t s) {
  dim3 grid((unsigned)bp.n_lines, nb);
#define X(A, B, C, NP, NS, SL, R)                                                                                  \
  if (bp.P1 == A && bp.P2 == B && bp.P3 == C && bp.tma_npart == NP && bp.tma_nseg == NS && bp.tma_slots == SL &&   \
      (bp.tma_ring != 0) == R)                                                                                     \
    k_stage_tma<A, B, C, NP, NS, SL, R><<<grid, TmaCfg<A, B, C, NP, NS, SL, R>::NT,                                \
                                          TmaCfg<A, B, C, NP, NS, SL, R>::SMEM, s>>>(op, bp, in, y, out, a, c, slot_stride);
  TMA_SPECIALISATIONS(X)
#undef X
  return 1;
}
