// Bulk-copy ("TMA") fed RK-stage kernel (steps a1-a3 of DESIGN.md) for three modes on sm_100a.
//
// Same arithmetic as chfpe_brick.cu (Eq. (8)-(12); G_s combination, scatter-form p_1 stencil, warp
// shuffle p_3 stencil), different data movement.  A brick (all momenta of one (element, q-point)) is cut along p_1 into
// NPART parts of PP planes; one part of one brick is a contiguous run of PP*P2*P3 doubles ("chunk", 16 KB at 16^3 with
// two parts).  A CTA owns one q_3 line of one part.  Every chunk the line needs -- the part of the own brick, of the
// hierarchy neighbours, of the q_1 / q_2 neighbour bricks, of y -- is streamed with 1-D bulk async copies
// (cp.async.bulk, completion on an mbarrier) into a ring of shared-memory slots, in a fixed order that every thread
// can enumerate; the LAST warp to release a slot refills it at once with the chunk SLOTS places ahead, so there is no
// producer warp (it would be the ninth warp of the CTA and cost 32 registers per thread: warps are allocated in
// fours).  All threads read each chunk exactly once with LDS.128 and fold it into their accumulators, so no load
// latency is exposed and no
// register is pinned by a load in flight (measured: the bulk-copy engine delivers 71 B/clk/SM = 20 TB/s from L2 while
// the consumers read and use everything, profiles/r02_probe_bulk_copy.md).  The q_3 derivative runs in scatter form
// along the line the CTA marches (RING): the own chunk of brick i_3 is added to the accumulators of bricks i_3-2,
// i_3-1, i_3+1, i_3+2, which live in registers, so no q_3 neighbour is ever loaded (12.7 instead of 16.7 chunk loads per
// brick).  Cutting bricks along p_1 halves the L2 window a lock-step group of elements needs,
// which pays for groups of four linked elements; the p_1 stencil needs G_1 on two planes beyond a part edge, and
// those planes (of the own brick and its up_1 / down_1 neighbours) arrive by three small bulk copies one brick ahead.
#include "chfpe_internal.cuh"

namespace {

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
  static constexpr int G3_ROW = P3 + 4, G3_PLANE = SHFL3 ? 0 : P2 * (P3 + 4);       // G_3[plane][i2][i3+2]
  static constexpr int XG = (NSEG > 1) ? (NSEG - 1) * 4 * PLANE : 0;                // G_1 planes next to a segment edge
  static constexpr int HSIDES = (NPART == 1) ? 0 : (NPART == 2 ? 1 : 2);            // part edges inside the brick
  static constexpr int HALO = HSIDES * 3 * 2 * PLANE;                               // [side][own, up_1, down_1][2 planes]
  static constexpr int NE = 21;                                    // chunk kinds per step
  static constexpr int MAXQ3 = 64;                                 // longest q_3 line (dU/dq_s table of the line)
  static constexpr size_t SMEM = (size_t)SLOTS * CHUNK + sizeof(double) * (PP * G2_PLANE + PP * G3_PLANE + XG + HALO) +
                                 16 * SLOTS + 8 + 8 * NE + 8 * 3 * MAXQ3 + 16;
  static constexpr int MINB = (2 * (SMEM + 1024) <= 227 * 1024 && 2 * NT <= 1024) ? 2 : 1;
};

// one line of the sweep: {element, i_q1 | i_q2 << 10 | part << 20, own-mask (as BrickId::own), unused}
struct TmaLine { int k, iq1, iq2, part, own; };
__device__ __forceinline__ TmaLine decode_line(const int4* lines, long long L) {
  const int4 t = __ldg(lines + L);
  TmaLine l;
  l.k = t.x; l.iq1 = t.y & 1023; l.iq2 = (t.y >> 10) & 1023; l.part = t.y >> 20; l.own = t.z;
  return l;
}

template <int P1, int P2, int P3, int NPART, int NSEG, int SLOTS, bool RING>
__global__ void __launch_bounds__(TmaCfg<P1, P2, P3, NPART, NSEG, SLOTS, RING>::NT, TmaCfg<P1, P2, P3, NPART, NSEG, SLOTS, RING>::MINB)
k_stage_tma(DevOp op, BrickPlan bp, const double* __restrict__ in, const double* y, double* out, double a, double cc,
            size_t slot_stride) {
  using C = TmaCfg<P1, P2, P3, NPART, NSEG, SLOTS, RING>;
  constexpr int PLANE = C::PLANE, PL2 = C::PL2, PP = C::PP, NC = C::NC;
  constexpr bool SKIP1 = (P2 == 1);                                 // two-mode view: middle mode has one point
  constexpr size_t BRICK = (size_t)P1 * PLANE;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char* ring = smem_raw;
  double* g2 = reinterpret_cast<double*>(smem_raw + (size_t)SLOTS * C::CHUNK);
  double* g3 = g2 + PP * C::G2_PLANE;
  double* xg = g3 + PP * C::G3_PLANE;
  double* halo = xg + C::XG;
  unsigned long long* full = reinterpret_cast<unsigned long long*>(halo + C::HALO);   // data of a slot has landed
  unsigned long long* hbar = full + SLOTS;                                            // halo planes have landed
  unsigned long long* empty = hbar + 1;                                               // all warps have released a slot
  const double** ent = reinterpret_cast<const double**>(empty + SLOTS);               // source of every chunk kind at step 0
  double* sdu = reinterpret_cast<double*>(ent + C::NE);                               // dU/dq_s at the q-points of the line
  const unsigned ring_a = t_smem_u32(ring), full_a = t_smem_u32(full), empty_a = t_smem_u32(empty), hbar_a = t_smem_u32(hbar);

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
  const int nsteps = RING ? n3 + 2 : n3;

  // ---- the chunk stream.  Kinds per step m (bit e of a step's mask; existence is uniform over the CTA):
  //   0 own part of brick m | 1 y of brick m-2 (RING) | 2+2s, 3+2s up / down neighbour element along s |
  //   8+4s+d q_s neighbour brick, d = 0..3: +1, -1, +2, -2 (s = 2 only without RING; R9: ghost bricks are skipped) |
  //   20 y of brick m (no RING).  Chunks are consumed in ascending (m, e); ent[e] + m * BRICK is the source.
  unsigned mask_line = 0;                                           // kinds 2..15, the same for every brick of the line
#pragma unroll
  for (int s = 0; s < 3; s++) {
    if (kupa[s] >= 0) mask_line |= 1u << (2 + 2 * s);
    if (kdna[s] >= 0) mask_line |= 1u << (3 + 2 * s);
  }
#pragma unroll
  for (int d = 0; d < 4; d++) {
    const int off = (d == 0) ? 1 : (d == 1 ? -1 : (d == 2 ? 2 : -2));
    if (ln.iq1 + off >= 0 && ln.iq1 + off < n1) mask_line |= 1u << (8 + d);
    if (!SKIP1 && ln.iq2 + off >= 0 && ln.iq2 + off < n2) mask_line |= 1u << (12 + d);
  }
  auto step_mask = [&](int m) -> unsigned {
    unsigned mk = 0;
    if (m < n3) {
      mk = mask_line | 1u;
      if (!RING) {
        mk |= 1u << 20;
        if (m + 1 < n3) mk |= 1u << 16;
        if (m >= 1) mk |= 1u << 17;
        if (m + 2 < n3) mk |= 1u << 18;
        if (m >= 2) mk |= 1u << 19;
      }
    }
    if (RING && m >= 2) mk |= 2u;
    return mk;
  };
  unsigned pol_bits = (1u << 1) | (1u << 20);                       // kinds whose lines are touched once: evict_first
#pragma unroll
  for (int s = 0; s < 3; s++) {
    if (!((ln.own >> (2 * s)) & 1)) pol_bits |= 1u << (2 + 2 * s);
    if (!((ln.own >> (2 * s + 1)) & 1)) pol_bits |= 1u << (3 + 2 * s);
  }
  const unsigned long long pol_own = t_policy((bp.l2mode & 2) ? 2 : 0);
  const unsigned long long pol_str = t_policy((bp.l2mode & 1) ? 1 : 0);
  // issue chunk (m, e) into ring slot sl (one thread)
  auto issue = [&](int m, int e, int sl) {
    a_mbar_expect_tx(full_a + 8 * sl, C::CHUNK);
    a_bulk_g2s(ring_a + sl * C::CHUNK, ent[e] + (size_t)m * BRICK, C::CHUNK, full_a + 8 * sl,
               ((pol_bits >> e) & 1u) ? pol_str : pol_own);
  };
  // halo planes of brick m (the two planes beyond each part edge of the own part and of its up_1 / down_1 neighbours)
  constexpr unsigned HB = 2 * PLANE * sizeof(double);
  auto issue_halo = [&](int m) {
    unsigned bytes = 0;
#pragma unroll
    for (int sd = 0; sd < C::HSIDES; sd++) {
      const bool lo = (C::HSIDES == 2) ? (sd == 0) : (part > 0);    // which edge this buffer side serves
      if (C::HSIDES == 2 && ((lo && part == 0) || (!lo && part + 1 == NPART))) continue;
      bytes += HB * (1 + (kupa[0] >= 0) + (kdna[0] >= 0));
    }
    if (bytes == 0) return;
    a_mbar_expect_tx(hbar_a, bytes);
#pragma unroll
    for (int sd = 0; sd < C::HSIDES; sd++) {
      const bool lo = (C::HSIDES == 2) ? (sd == 0) : (part > 0);
      if (C::HSIDES == 2 && ((lo && part == 0) || (!lo && part + 1 == NPART))) continue;
      const long long po = (lo ? -2 : PP) * (long long)PLANE + (long long)m * (long long)BRICK;
      const unsigned dst = t_smem_u32(halo + sd * 3 * 2 * PLANE);
      a_bulk_g2s(dst, ent[0] + po, HB, hbar_a, pol_str);
      if (kupa[0] >= 0) a_bulk_g2s(dst + 2 * PLANE * 8, ent[2] + po, HB, hbar_a, pol_str);
      if (kdna[0] >= 0) a_bulk_g2s(dst + 4 * PLANE * 8, ent[3] + po, HB, hbar_a, pol_str);
    }
  };

  if (t == 0) {
    for (int s = 0; s < SLOTS; s++) { t_mbar_init(full + s, 1); t_mbar_init(empty + s, C::NW); }
    t_mbar_init(hbar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    const double* Xk = X + (size_t)k * op.cells + pofs + (size_t)ql0 * BRICK;
    const double* Yk = y + boff + (size_t)k * op.cells + pofs + (size_t)ql0 * BRICK;
    ent[0] = Xk;
    ent[1] = Yk - 2 * BRICK;
    ent[20] = Yk;
#pragma unroll
    for (int s = 0; s < 3; s++) {
      ent[2 + 2 * s] = X + (size_t)(kupa[s] >= 0 ? kupa[s] : k) * op.cells + pofs + (size_t)ql0 * BRICK;
      ent[3 + 2 * s] = X + (size_t)(kdna[s] >= 0 ? kdna[s] : k) * op.cells + pofs + (size_t)ql0 * BRICK;
#pragma unroll
      for (int d = 0; d < 4; d++) {
        const int off = (d == 0) ? 1 : (d == 1 ? -1 : (d == 2 ? 2 : -2));
        ent[8 + 4 * s + d] = Xk + off * op.st[s];
      }
    }
  }
  // cursor of the chunk SLOTS places ahead of the one being consumed (the same in every thread): step, kinds left in it
  int f_m = 0;
  unsigned f_rest = step_mask(0);
  auto f_next = [&]() {                                             // drop the lowest kind, move on to the next non-empty step
    f_rest &= f_rest - 1u;
    while (f_rest == 0 && f_m < nsteps) { f_m++; f_rest = (f_m < nsteps) ? step_mask(f_m) : 0u; }
  };
  __syncthreads();                                                  // barriers initialised, ent[] written
  for (int sl = 0; sl < SLOTS; sl++) {                              // fill the ring: the first SLOTS chunks of the stream
    if (t == 0 && f_m < nsteps) issue(f_m, __ffs(f_rest) - 1, sl);
    f_next();
  }
  if (NPART > 1 && t == 0) issue_halo(0);
  for (int i = t; i < 3 * n3; i += C::NT) {
    const int s = i / n3, m = i - s * n3;
    sdu[s * C::MAXQ3 + m] = __ldg(op.dU[s] + ql0 + m);
  }
  // ghost rows / columns of the exchange planes stay zero for the whole kernel
  for (int i = t; i < (SKIP1 ? 0 : PP * 4 * P3); i += C::NT) {
    const int pl = i / (4 * P3), rr = i - pl * (4 * P3), row = rr / P3, col = rr - row * P3;
    g2[pl * C::G2_PLANE + (row < 2 ? row : P2 + row) * C::G2_ROW + col] = 0.0;
  }
  for (int i = t; i < (C::SHFL3 ? 0 : PP * P2 * 4); i += C::NT) {
    const int rw = i >> 2, c4 = i & 3;
    g3[rw * C::G3_ROW + (c4 < 2 ? c4 : P3 + c4)] = 0.0;
  }
  __syncthreads();

  const bool active = t < C::NACT;
  const int tt = active ? t : 0;
  const int seg = (NSEG == 1) ? 0 : tt / PL2;
  const int tid = tt - seg * PL2;                                   // pair index inside the plane
  const int jbase = seg * NC;                                       // first plane (inside the part) of this thread
  const int i2 = tid / (P3 / 2), i3 = 2 * (tid - i2 * (P3 / 2));
  const int lane = t & 31;
  const unsigned tpart = (unsigned)(jbase * PL2 + tid);             // first own pair inside a chunk
  const double h1 = op.h[3];
  const double p1_0 = op.x0[3] + (part * PP + jbase) * h1;
  const double p2 = op.x0[4] + i2 * op.h[4];
  const double p3a = op.x0[5] + i3 * op.h[5], p3b = op.x0[5] + (i3 + 1) * op.h[5];
  // CENTRAL4 weights: D f_i = [8 (f_{i+1} - f_{i-1}) - (f_{i+2} - f_{i-2})] / (12 h)
  const double w1p = -op.c2[3], w2p = -op.c2[4], w3p = -op.c2[5];   // 1 / (12 h) of p_1, p_2, p_3
  const double wp8 = 8.0 * w1p, wp1 = w1p;
  double cq[3];                                                     // -(1/m_s) / (12 h_qs)
#pragma unroll
  for (int s = 0; s < 3; s++) cq[s] = op.c2[s] * op.inv_mass[s];
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

  int slot = 0, turn = 0;                                           // ring slot of the current chunk; warp whose turn it is to refill
  unsigned ph = 0, hph = 0;
  const int warp = t >> 5;
  const unsigned my_a = ring_a + tpart * 16;                        // this thread's first pair inside slot 0
  unsigned pre = 0;                                                 // early (non-blocking) look at the current slot's barrier
  auto acquire = [&]() -> unsigned {
    if (!pre) a_mbar_wait(full_a + 8 * slot, ph);
    return my_a + slot * C::CHUNK;
  };
  // Release the current chunk n.  The refill lags one chunk: the warp whose turn it is waits until every warp has let
  // go of the slot of chunk n-1 (almost always the case by now) and loads the chunk SLOTS places after n-1 into it.
  // Turns rotate, so a warp can block on every NW-th chunk only.
  int pslot = -1;                                                   // slot of chunk n-1
  unsigned pph = 0;
  auto release = [&]() {
    __syncwarp();
    if (lane == 0) a_mbar_arrive(empty_a + 8 * slot);
    if (pslot >= 0) {
      if (warp == turn && f_m < nsteps) {
        a_mbar_wait(empty_a + 8 * pslot, pph);
        if (lane == 0) issue(f_m, __ffs(f_rest) - 1, pslot);
      }
      f_next();
    }
    if (++turn == C::NW) turn = 0;
    pslot = slot; pph = ph;
    if (++slot == SLOTS) { slot = 0; ph ^= 1u; }
    pre = a_mbar_test(full_a + 8 * slot, ph);                       // consumed at the next acquire
  };

  // accumulators of the bricks m-1, m, m+1, m+2 of the line (RING; brick m-2 is finished inside a step and its
  // registers take the new brick m+2), or of the current brick only
  constexpr int NA = RING ? 4 : 1;
  double2 A[NA][NC];
#pragma unroll
  for (int r = 0; r < NA; r++)
#pragma unroll
    for (int j = 0; j < NC; j++) A[r][j] = make_double2(0.0, 0.0);
  // RING roles at the start of step m: A[0] = brick m-2, A[1] = m-1, A[2] = m, A[3] = m+1

  const size_t ebase = (size_t)k * op.cells + pofs + (size_t)jbase * PLANE + 2 * tid;   // own cells inside brick 0 of an element
  double2* Ob = reinterpret_cast<double2*>(out + boff + ebase);

#pragma unroll 1
  for (int m = 0; m < nsteps; m++) {
    const size_t bq = (size_t)(ql0 + m) * BRICK;
    const bool have = m < n3;                                       // brick m exists (RING: the last two steps only finish)
    if (t == 0 && m + 1 < n3) {                                     // HBM-sourced data of brick m+1 -> L2
      const size_t bn = (size_t)(m + 1) * BRICK;
      if ((mask_line >> 10) & 1u) t_prefetch_l2(ent[10] + bn, C::CHUNK);
#pragma unroll
      for (int e = 2; e < 8; e++)
        if ((mask_line >> e) & (pol_bits >> e) & 1u) t_prefetch_l2(ent[e] + bn, C::CHUNK);
      t_prefetch_l2(ent[20] + bn, C::CHUNK);
    }
    double2 x[NC];
    if (have) {
      const unsigned S = acquire();                                 // kind 0: own part
#pragma unroll
      for (int j = 0; j < NC; j++) x[j] = a_lds2(S + j * (PL2 * 16));
      release();
    }
    if (RING) {
      const double2 c3 = make_double2(cq[2] * p3a, cq[2] * p3b);   // -(p_3/m_3)/(12 h): dW/dq_3 in scatter form along the line
      if (have) {
#pragma unroll
        for (int j = 0; j < NC; j++) A[0][j] = t_fma2(make_double2(-c3.x, -c3.y), x[j], A[0][j]);   // brick m-2 sees x_m at +2: weight -1
      }
      if (m >= 2) {                                                 // finish brick m-2: out = a y + c F
        const unsigned S = acquire();                               // kind 1: y of brick m-2
        double2* O = Ob + (bq - 2 * BRICK) / 2;
#pragma unroll
        for (int j = 0; j < NC; j++) {
          const double2 yv = a_lds2(S + j * (PL2 * 16));
          if (active) t_st2(O + j * PL2, make_double2(fma(cc, A[0][j].x, a * yv.x), fma(cc, A[0][j].y, a * yv.y)), pol_str);
        }
        release();
      }
      if (have) {
        const double2 c38 = make_double2(8.0 * c3.x, 8.0 * c3.y);
#pragma unroll
        for (int j = 0; j < NC; j++) {
          A[1][j] = t_fma2(c38, x[j], A[1][j]);                                     // brick m-1 sees x_m at +1: weight +8
          A[3][j] = t_fma2(make_double2(-c38.x, -c38.y), x[j], A[3][j]);            // brick m+1 sees x_m at -1: weight -8
          A[0][j] = make_double2(c3.x * x[j].x, c3.y * x[j].y);                     // brick m+2 sees x_m at -2: weight +1
        }
      } else {
#pragma unroll
        for (int j = 0; j < NC; j++) A[0][j] = make_double2(0.0, 0.0);
      }
    }
    if (have) {
      double2(&acc)[NC] = A[RING ? 2 : 0];
#pragma unroll
      for (int j = 0; j < NC; j++) acc[j] = t_fma2(-Gam, x[j], acc[j]);
      Vp[2] = fma(op.VSL[2], op.x0[2] + m * op.h[2], op.VLL[2]);
#pragma unroll
      for (int s = 0; s < 3; s++) {
        if (SKIP1 && s == 1) continue;
        const double dUs = sdu[s * C::MAXQ3 + m];
        const double cu = Vp[s], cd = cdf[s] * Vp[s];
        const double pu = cu * op.kup[s], pd = cd * op.kdn[s];
        double2 g[NC];
#pragma unroll
        for (int j = 0; j < NC; j++) g[j] = make_double2(dUs * x[j].x, dUs * x[j].y);
        if (kupa[s] >= 0) {                                         // Phi_s W^(n+e_s), Eq. (11)
          const unsigned S = acquire();
#pragma unroll
          for (int j = 0; j < NC; j++) {
            const double2 v = a_lds2(S + j * (PL2 * 16));
            const double psa = (s == 0) ? fma((double)j, h1, p1_0) : (s == 1 ? p2 : p3a);
            const double psb = (s == 2) ? p3b : psa;
            g[j] = t_fma2(cu, v, g[j]);
            acc[j].x = fma(psa * pu, v.x, acc[j].x);
            acc[j].y = fma(psb * pu, v.y, acc[j].y);
          }
          release();
        }
        if (kdna[s] >= 0) {                                         // n_s Theta_s W^(n-e_s), Eq. (12) with R1
          const unsigned S = acquire();
#pragma unroll
          for (int j = 0; j < NC; j++) {
            const double2 v = a_lds2(S + j * (PL2 * 16));
            const double psa = (s == 0) ? fma((double)j, h1, p1_0) : (s == 1 ? p2 : p3a);
            const double psb = (s == 2) ? p3b : psa;
            g[j] = t_fma2(cd, v, g[j]);
            acc[j].x = fma(psa * pd, v.x, acc[j].x);
            acc[j].y = fma(psb * pd, v.y, acc[j].y);
          }
          release();
        }
        if (s == 0) {                                               // D_{p_1} G_1 in scatter form
#pragma unroll
          for (int j = 0; j < NC; j++) {
            if (j >= 1) acc[j - 1] = t_fma2(wp8, g[j], acc[j - 1]);
            if (j + 1 < NC) acc[j + 1] = t_fma2(-wp8, g[j], acc[j + 1]);
            if (j >= 2) acc[j - 2] = t_fma2(-wp1, g[j], acc[j - 2]);
            if (j + 2 < NC) acc[j + 2] = t_fma2(wp1, g[j], acc[j + 2]);
          }
          if (NPART > 1 && (do_lo || do_hi)) {                      // G_1 on the two planes beyond a part edge
            a_mbar_wait(hbar_a, hph);
#pragma unroll
            for (int sd = 0; sd < C::HSIDES; sd++) {
              const bool lo = (C::HSIDES == 2) ? (sd == 0) : (part > 0);
              if (lo ? !do_lo : !do_hi) continue;
              const double* H = halo + sd * 3 * 2 * PLANE + 2 * tid;
              double2 gh[2];
#pragma unroll
              for (int e = 0; e < 2; e++) {
                const double2 hx = *reinterpret_cast<const double2*>(H + e * PLANE);
                gh[e] = make_double2(dUs * hx.x, dUs * hx.y);
                if (kupa[0] >= 0) gh[e] = t_fma2(cu, *reinterpret_cast<const double2*>(H + (2 + e) * PLANE), gh[e]);
                if (kdna[0] >= 0) gh[e] = t_fma2(cd, *reinterpret_cast<const double2*>(H + (4 + e) * PLANE), gh[e]);
              }
              if (lo) {                                             // planes -2, -1 below the part
                acc[0] = t_fma2(wp1, gh[0], acc[0]);
                acc[0] = t_fma2(-wp8, gh[1], acc[0]);
                acc[1] = t_fma2(wp1, gh[1], acc[1]);
              } else {                                              // planes PP, PP+1 above the part
                acc[NC - 1] = t_fma2(wp8, gh[0], acc[NC - 1]);
                acc[NC - 2] = t_fma2(-wp1, gh[0], acc[NC - 2]);
                acc[NC - 1] = t_fma2(-wp1, gh[1], acc[NC - 1]);
              }
            }
          }
          hph ^= 1u;
          asm volatile("bar.sync 1, %0;" ::"r"(C::NT) : "memory");  // exchange planes of the previous brick are free
          if (NSEG > 1 && active) {                                 // planes next to a segment edge -> neighbour segment
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
        } else if (C::SHFL3) {                                      // D_{p_3} G_3 from the neighbour lanes of the row
          constexpr int W = P3 / 2;
          const int c = tid % W;
#pragma unroll
          for (int j = 0; j < NC; j++) {
            const double2 own = g[j];
            double ly = __shfl_up_sync(0xffffffffu, own.y, 1, W), rx = __shfl_down_sync(0xffffffffu, own.x, 1, W);
            double lx = __shfl_up_sync(0xffffffffu, own.x, 1, W), ry = __shfl_down_sync(0xffffffffu, own.y, 1, W);
            if (c == 0) { ly = 0.0; lx = 0.0; }
            if (c == W - 1) { rx = 0.0; ry = 0.0; }
            const double e3x = fma(8.0, own.y - ly, -(rx - lx));
            const double e3y = fma(8.0, rx - own.x, -(ry - ly));
            acc[j].x = fma(w3p, e3x, acc[j].x);
            acc[j].y = fma(w3p, e3y, acc[j].y);
          }
        } else if (active) {
#pragma unroll
          for (int j = 0; j < NC; j++)
            *reinterpret_cast<double2*>(g3 + (jbase + j) * C::G3_PLANE + i2 * C::G3_ROW + i3 + 2) = g[j];
        }
      }
      // ---- -(p_s/m_s) dW/dq_s, s = 1, 2 (and 3 without the ring): one chunk per existing neighbour brick ----
#pragma unroll
      for (int s = 0; s < (RING ? 2 : 3); s++) {
        if (SKIP1 && s == 1) continue;
#pragma unroll
        for (int d = 0; d < 4; d++) {
          const int off = (d == 0) ? 1 : (d == 1 ? -1 : (d == 2 ? 2 : -2));
          const bool ex = (s < 2) ? ((mask_line >> (8 + 4 * s + d)) & 1u) != 0 : (m + off >= 0 && m + off < n3);
          if (!ex) continue;
          const double wd = cq[s] * ((d == 0) ? 8.0 : (d == 1 ? -8.0 : (d == 2 ? -1.0 : 1.0)));
          const unsigned S = acquire();
#pragma unroll
          for (int j = 0; j < NC; j++) {
            const double2 v = a_lds2(S + j * (PL2 * 16));
            const double ca = (s == 0) ? wd * fma((double)j, h1, p1_0) : (s == 1 ? wd * p2 : wd * p3a);
            const double cb = (s == 2) ? wd * p3b : ca;
            acc[j].x = fma(ca, v.x, acc[j].x);
            acc[j].y = fma(cb, v.y, acc[j].y);
          }
          release();
        }
      }
      asm volatile("bar.sync 1, %0;" ::"r"(C::NT) : "memory");      // G_2 / G_3 / segment-edge G_1 complete, halo planes read
      if (NPART > 1 && t == 0 && m + 1 < n3) issue_halo(m + 1);
      if (NSEG > 1) {
        if (seg > 0) {                                              // G_1 at planes jbase-2, jbase-1
          const double2 gm2 = *reinterpret_cast<const double2*>(xg + ((seg - 1) * 4 + 0) * PLANE + 2 * tid);
          const double2 gm1 = *reinterpret_cast<const double2*>(xg + ((seg - 1) * 4 + 1) * PLANE + 2 * tid);
          acc[0] = t_fma2(-wp8, gm1, acc[0]);
          acc[0] = t_fma2(wp1, gm2, acc[0]);
          acc[1] = t_fma2(wp1, gm1, acc[1]);
        }
        if (seg + 1 < NSEG) {                                       // G_1 at planes jbase+NC, jbase+NC+1
          const double2 gp0 = *reinterpret_cast<const double2*>(xg + (seg * 4 + 2) * PLANE + 2 * tid);
          const double2 gp1 = *reinterpret_cast<const double2*>(xg + (seg * 4 + 3) * PLANE + 2 * tid);
          acc[NC - 1] = t_fma2(wp8, gp0, acc[NC - 1]);
          acc[NC - 1] = t_fma2(-wp1, gp1, acc[NC - 1]);
          acc[NC - 2] = t_fma2(-wp1, gp0, acc[NC - 2]);
        }
      }
      {
        const double* c2 = g2 + jbase * C::G2_PLANE + (i2 + 2) * C::G2_ROW + i3;
        const double* c3p = g3 + jbase * C::G3_PLANE + i2 * C::G3_ROW + i3 + 2;
#pragma unroll
        for (int j = 0; j < NC; j++) {
          if (!SKIP1) {
            const double* a2 = c2 + j * C::G2_PLANE;
            const double2 u1 = *reinterpret_cast<const double2*>(a2 + C::G2_ROW), d1 = *reinterpret_cast<const double2*>(a2 - C::G2_ROW);
            const double2 u2 = *reinterpret_cast<const double2*>(a2 + 2 * C::G2_ROW), d2 = *reinterpret_cast<const double2*>(a2 - 2 * C::G2_ROW);
            acc[j].x = fma(w2p, fma(8.0, u1.x - d1.x, -(u2.x - d2.x)), acc[j].x);
            acc[j].y = fma(w2p, fma(8.0, u1.y - d1.y, -(u2.y - d2.y)), acc[j].y);
          }
          if (!C::SHFL3) {
            const double* a3 = c3p + j * C::G3_PLANE;
            const double2 lft = *reinterpret_cast<const double2*>(a3 - 2), rgt = *reinterpret_cast<const double2*>(a3 + 2);
            const double2 own = *reinterpret_cast<const double2*>(a3);
            // pair (i3, i3+1): neighbours i3-2..i3+3 = lft.x lft.y [own.x own.y] rgt.x rgt.y
            acc[j].x = fma(w3p, fma(8.0, own.y - lft.y, -(rgt.x - lft.x)), acc[j].x);
            acc[j].y = fma(w3p, fma(8.0, rgt.x - own.x, -(rgt.y - lft.y)), acc[j].y);
          }
        }
      }
      if (!RING) {                                                  // stage combine of this brick
        const unsigned S = acquire();                               // kind 20: y
        double2* O = Ob + bq / 2;
#pragma unroll
        for (int j = 0; j < NC; j++) {
          const double2 yv = a_lds2(S + j * (PL2 * 16));
          if (active) t_st2(O + j * PL2, make_double2(fma(cc, acc[j].x, a * yv.x), fma(cc, acc[j].y, a * yv.y)), pol_str);
          acc[j] = make_double2(0.0, 0.0);
        }
        release();
      }
    }
    if (RING) {                                                     // the line advances by one brick
#pragma unroll
      for (int j = 0; j < NC; j++) {
        const double2 nw = A[0][j];
        A[0][j] = A[1][j]; A[1][j] = A[2][j]; A[2][j] = A[3][j]; A[3][j] = nw;
      }
    }
  }
}

}  // namespace

// (P1, P2, P3, NPART, NSEG, SLOTS, RING)
#define TMA_SPECIALISATIONS(X) \
  X(16, 16, 16, 2, 2, 4, true) X(16, 16, 16, 2, 2, 4, false) X(16, 16, 16, 1, 4, 4, true) X(16, 16, 16, 1, 4, 4, false) \
  X(16, 16, 16, 2, 2, 3, false) X(16, 16, 16, 2, 2, 8, false) X(16, 16, 16, 2, 2, 3, true) X(16, 16, 16, 2, 2, 8, true) X(16, 16, 16, 1, 4, 5, false) \
  X(8, 8, 8, 2, 2, 4, true) X(8, 8, 8, 1, 2, 4, true) X(8, 8, 8, 1, 2, 4, false) X(12, 12, 12, 2, 3, 4, true)

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
