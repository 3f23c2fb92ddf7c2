// Bulk-copy fed RK-stage kernel of the Hermite representation (row f1; included by chfpe_hermite.cu inside its anonymous
// namespace, after HOp / HSlab).  Same arithmetic as hermite_patch_body (de-garbled Eq. A1-A4, reading
// R19), the data movement of k_stage_tma (chfpe_tma.cu): three modes on an n_1 x 32 x 32 mesh, explicit stencils.
//
// A CTA owns one slab (element n, Hermite multi-index k) and marches along q_1 in bands of two planes: a band of a slab
// is a contiguous 16 KB chunk, so every operand arrives by a 1-D bulk copy (cp.async.bulk + mbarrier) into a ring of
// shared-memory slots and is read exactly once with LDS.128.  Chunk kinds per band, consumed in this order (kind e always
// uses slot e mod SLOTS; a kind that is absent moves no data but still flips its barriers):
//   0 own slab | per mode s = 1..3: up (n, k+e_s), down (n, k-e_s), dU/dq_s on the band | six hierarchy neighbours
//   (n-e_s, k+e_s), (n+e_s, k-e_s) | y of the PREVIOUS band | three unused kinds (20 kinds = 4 x 5 slots).
// A thread owns four pairs of q_3-adjacent points: both planes of the band on rows r and r + 16.  Per mode the ladder
// combination P_s = sqrt(k_s+1) c_up + sqrt(k_s) c_dn is formed in registers; its derivative runs along q_3 on warp
// shuffles (a row is 16 lanes), along q_2 through one shared plane pair (ghost rows by predicate), and along q_1 in scatter form over
// the march: P_1 of band m is added to the accumulators of bands m-1, m and m+1, which live in registers (the halo of
// two planes is exactly one band), so band m-1 is finished, combined with y and written while band m is in flight.
// No q_1 halo is ever loaded: 13 chunks per band on average against 16.5 slab-units per value in the patch kernel.
// COMPACT6 (template flag CMP): the compact (Pade) derivative along q_2 and q_3 is solved inside the kernel on shared
// memory (Eq. 25-31 :177-201 with a = 7/9, R4; Thomas as in k_hermite_compact_line); only the q_1 lines, which run along
// the march, keep their line pass, so a stage is 2 launches instead of 4.

__device__ __forceinline__ unsigned ht_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void ht_mbar_init(unsigned bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void ht_arrive(unsigned bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void ht_arrive_if(unsigned bar, bool on) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.u32 p, %1, 0;\n\t"
      "@p mbarrier.arrive.shared::cta.b64 _, [%0];\n\t}" ::"r"(bar), "r"((unsigned)on)
      : "memory");
}
__device__ __forceinline__ void ht_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void ht_wait(unsigned bar, unsigned parity) {
  unsigned done;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.b32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
  } while (!done);
}
__device__ __forceinline__ void ht_bulk(unsigned dst, const void* src, unsigned bytes, unsigned bar, unsigned long long pol) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst),
      "l"(src), "r"(bytes), "r"(bar), "l"(pol)
      : "memory");
}
__device__ __forceinline__ void ht_prefetch(const void* src, unsigned bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ double2 ht_lds2(unsigned addr) {
  double2 v;
  asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
  return v;
}
__device__ __forceinline__ unsigned long long ht_policy(int kind) {   // 0 normal, 1 evict_first
  unsigned long long p;
  if (kind == 1) asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  else asm("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ void ht_st2(double2* p, double2 v, unsigned long long pol) {
  asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}
__device__ __forceinline__ double2 ht_fma2(double c, double2 a, double2 b) { return make_double2(fma(c, a.x, b.x), fma(c, a.y, b.y)); }

template <int J, int N> struct HtUnroll {
  template <typename F> __device__ __forceinline__ static void run(F&& f) { f(std::integral_constant<int, J>()); HtUnroll<J + 1, N>::run(f); }
};
template <int N> struct HtUnroll<N, N> {
  template <typename F> __device__ __forceinline__ static void run(F&&) {}
};
template <int E> using HtKind = std::integral_constant<int, E>;

// One compact-derivative line of 32 points in shared memory, in place: point i holds P_i on entry and d_i on exit, where
// tridiag(1/3, 1, 1/3) d = r, r_i = ca (P_{i+1} - P_{i-1}) + cb (P_{i+2} - P_{i-2}), zero ghosts.  tab: reciprocal pivots
// [0, 32) and elimination factors [32, 64) (read-only after the kernel's setup: loaded through asm the compiler may hoist).
// ST is a compile-time stride so that the window loads are provably distinct from the stores and leave the dependency chain,
// which is one FMA per point in either sweep.
__device__ __forceinline__ double ht_lds_const(unsigned addr) {
  double v;
  asm("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
  return v;
}
template <int ST, bool SWZ>
__device__ __forceinline__ void ht_thomas32(double* __restrict__ B0, const int l, const unsigned tab_a, const double ca, const double cb) {
  // point i of line l lives at B0[i * ST + (SWZ ? l ^ (i >> 1) : l)]
  auto at = [&](int i) -> double& { return B0[i * ST + (SWZ ? (l ^ (i >> 1)) : l)]; };
  double Pm2 = 0.0, Pm1 = 0.0, P0 = at(0), P1 = at(1), prev = 0.0;
#pragma unroll
  for (int i = 0; i < 32; i++) {
    const double P2 = (i + 2 < 32) ? at(i + 2) : 0.0;
    const double r = ca * (P1 - Pm1) + cb * (P2 - Pm2);
    const double ib = ht_lds_const(tab_a + 8 * i);
    prev = fma((-1.0 / 3.0) * ib, prev, r * ib);
    at(i) = prev;                                                   // P_i is not read again: the window holds P_{i-2} .. P_{i+2}
    Pm2 = Pm1; Pm1 = P0; P0 = P1; P1 = P2;
  }
  double x = prev;
#pragma unroll
  for (int i = 30; i >= 0; i--) { x = fma(-ht_lds_const(tab_a + 8 * (32 + i + 1)), x, at(i)); at(i) = x; }
}

// CMP = false: explicit stencils (CENTRAL4 / CENTRAL2).  CMP = true: COMPACT6, the Pade derivative along q_2 and q_3 is solved
// inside the kernel (one Thomas solve per line of the band, 128 lines of 32 points: 16 lanes of every warp own one line each,
// the recurrence of k_hermite_compact_line on shared memory); the q_1 lines run along the march and keep their own line pass.
template <bool CMP> struct HtCfgT {
  static constexpr int NROW = 32, NCOL = 32, PLANE = NROW * NCOL, BAND = 2 * PLANE;   // two q_1 planes per band
  static constexpr unsigned CHUNK = BAND * sizeof(double);                            // 16 KB
  // ring depth: 2 CTAs x (SLOTS x 16 KB + planes) must fit the SM's 228 KB; the kernel waits for data, so depth is speed
  // (explicit scheme at cfg4h: 4 slots 3.92 ms, 5 slots 3.15 ms); NK = kinds per band, padded to a multiple of SLOTS
  static constexpr int SLOTS = CMP ? 5 : 6, NK = CMP ? 20 : 18, NT = 256, NW = NT / 32, NI = 4;   // NI pairs per thread
  static constexpr int G2_PLANE = NROW * NCOL;                                        // P_2[plane][row][col]
  // CMP: P_3[plane][col][row ^ (col >> 1)]: transposed, so that the q_3 solve walks the same stride as the q_2 solve, and
  // swizzled, so that both the solver (16 consecutive rows per warp) and the owners (16 pair columns of a row) are conflict-free
  static constexpr int G3_PLANE = NROW * NCOL;
  static constexpr size_t SMEM = (size_t)SLOTS * CHUNK + sizeof(double) * 2 * (G2_PLANE + (CMP ? G3_PLANE : 0)) + 16 * SLOTS + 32 +
                                 8 * NK + (CMP ? 512 : 0) + 16;
};
using HtCfg = HtCfgT<false>;

template <bool CMP>
__global__ void __launch_bounds__(HtCfgT<CMP>::NT, 2) k_hermite_stage_tma(const HOp op, const double* __restrict__ in, const double* y,
                                                                         double* out, const double a, const double c,
                                                                         const size_t slot_stride) {
  using C = HtCfgT<CMP>;
  constexpr int NK = C::NK, SLOTS = C::SLOTS, NI = C::NI;
  extern __shared__ __align__(128) unsigned char ht_smem[];
  double* g2 = reinterpret_cast<double*>(ht_smem + (size_t)SLOTS * C::CHUNK);
  double* g3 = g2 + 2 * C::G2_PLANE;                                // CMP only
  unsigned long long* full = reinterpret_cast<unsigned long long*>(g3 + (CMP ? 2 * C::G3_PLANE : 0));
  unsigned long long* empty = full + SLOTS;
  unsigned long long* xbar = empty + SLOTS;                         // [0]: P planes written, [1]: read, [2]: solved (CMP)
  const double** ent = reinterpret_cast<const double**>(xbar + 4);  // source of every kind at band 0
  double* tab = reinterpret_cast<double*>(ent + NK);                // CMP: reciprocal pivots [0, 32) and elimination factors [32, 64)
  const unsigned tab_a = ht_smem_u32(tab);
  const unsigned ring_a = ht_smem_u32(ht_smem), full_a = ht_smem_u32(full), empty_a = ht_smem_u32(empty), xbar_a = ht_smem_u32(xbar);

  const int t = threadIdx.x, lane = t & 31, warp = __shfl_sync(0xffffffffu, t >> 5, 0);
  const int slab = blockIdx.x;
  const size_t soff = (size_t)blockIdx.y * slot_stride, Q = (size_t)op.Q;
  const HSlab* __restrict__ S = op.slabs + slab;
  const int nbands = op.nq[0] / 2;
  int up[3], dn[3], hdn[3], hup[3];
#pragma unroll
  for (int s = 0; s < 3; s++) { up[s] = S->up[s]; dn[s] = S->dn[s]; hdn[s] = S->hdn[s]; hup[s] = S->hup[s]; }
  // kinds: 0 self | 1+3s up_s, 2+3s dn_s, 3+3s dU_s | 10+2s hdn_s, 11+2s hup_s | 16 y of the previous band
  unsigned mask_line = 1u;
#pragma unroll
  for (int s = 0; s < 3; s++) {
    if (up[s] >= 0) mask_line |= 1u << (1 + 3 * s);
    if (dn[s] >= 0) mask_line |= 1u << (2 + 3 * s);
    if (up[s] >= 0 || dn[s] >= 0) mask_line |= 1u << (3 + 3 * s);
    if (hdn[s] >= 0) mask_line |= 1u << (10 + 2 * s);
    if (hup[s] >= 0) mask_line |= 1u << (11 + 2 * s);
  }
  auto step_mask = [&](int m) -> unsigned { return (m < nbands ? mask_line : 0u) | ((m >= 1 && m <= nbands) ? (1u << 16) : 0u); };
  // own slab, Hermite neighbours, dU: re-read by the CTAs of the neighbouring slabs -> normal L2 policy; hierarchy neighbours
  // (other elements: 512 slabs away in launch order) and y are used once per launch -> evict_first, as are the stores
  const unsigned long long pol_in = ht_policy(0), pol_str = ht_policy(1);
  auto issue = [&](int m, int e, unsigned mk) {                      // one thread: load kind e of band m, or just flip its barrier
    const unsigned fb = full_a + 8 * (e % SLOTS);
    if ((mk >> e) & 1u) {
      ht_expect_tx(fb, C::CHUNK);
      ht_bulk(ring_a + (e % SLOTS) * C::CHUNK, ent[e] + (size_t)m * C::BAND, C::CHUNK, fb, e >= 10 ? pol_str : pol_in);
    } else {
      ht_arrive(fb);
    }
  };
  if (t == 0) {
    for (int s = 0; s < SLOTS; s++) { ht_mbar_init(full_a + 8 * s, 1); ht_mbar_init(empty_a + 8 * s, C::NW); }
    ht_mbar_init(xbar_a, C::NW); ht_mbar_init(xbar_a + 8, C::NW); ht_mbar_init(xbar_a + 16, C::NW);
    if (CMP)                                                        // both axes have 32 points: one table (it depends on n only)
      for (int i = 0; i < 32; i++) { tab[i] = op.ibet[1][i]; tab[32 + i] = op.cfac[1][i]; }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    const double* X = in + soff;
    for (int e = 0; e < NK; e++) ent[e] = X + (size_t)slab * Q;
#pragma unroll
    for (int s = 0; s < 3; s++) {
      ent[1 + 3 * s] = X + (size_t)(up[s] >= 0 ? up[s] : slab) * Q;
      ent[2 + 3 * s] = X + (size_t)(dn[s] >= 0 ? dn[s] : slab) * Q;
      ent[3 + 3 * s] = op.dU[s];
      ent[10 + 2 * s] = X + (size_t)(hdn[s] >= 0 ? hdn[s] : slab) * Q;
      ent[11 + 2 * s] = X + (size_t)(hup[s] >= 0 ? hup[s] : slab) * Q;
    }
    ent[16] = (a != 0.0 ? y + soff : X) + (size_t)slab * Q - C::BAND;   // (band m - 1 at step m; a = 0: y is not to be read)
    const unsigned mk0 = step_mask(0);
    for (int e = 0; e < SLOTS; e++) issue(0, e, mk0);
  }
  __syncthreads();

  const int cp = t & 15, r0 = t >> 4;                               // pair column, first row (the second one is r0 + 16)
  // item j = 0..3: plane j >> 1, row r0 + 16 (j & 1); byte offset of the pair inside a chunk
  unsigned my_a = ring_a + (unsigned)(r0 * C::NCOL + 2 * cp) * 8;
  asm volatile("" : "+r"(my_a));
  auto item_off = [](int j) { return (unsigned)(((j >> 1) * C::PLANE + (j & 1) * 16 * C::NCOL) * 8); };
  const double gam = S->gam;
  int m = 0;
  unsigned mask = __shfl_sync(0xffffffffu, step_mask(0), 0), maskn = __shfl_sync(0xffffffffu, step_mask(1), 0), mpar = 0;
  auto parity = [&](int E, unsigned mp) -> unsigned { return ((unsigned)(E / SLOTS) & 1u) ^ (((NK / SLOTS) & 1) ? mp : 0u); };
  auto duty = [&](auto KEP, int mm, unsigned mp, unsigned mk_same, unsigned mk_next) {
    constexpr int EP = decltype(KEP)::value;
    constexpr int E2 = (EP + SLOTS < NK) ? EP + SLOTS : EP + SLOTS - NK;
    const int m2 = (EP + SLOTS < NK) ? mm : mm + 1;
    if (mm < 0 || m2 > nbands) return;
    ht_wait(empty_a + 8 * (EP % SLOTS), parity(EP, mp));
    if (lane == 0) issue(m2, E2, (EP + SLOTS < NK) ? mk_same : mk_next);
  };
  auto chunk = [&](auto KE, auto&& body) {
    constexpr int E = decltype(KE)::value;
    ht_wait(full_a + 8 * (E % SLOTS), parity(E, mpar));
    if ((mask >> E) & 1u) body(my_a + (E % SLOTS) * C::CHUNK);
    __syncwarp();
    ht_arrive_if(empty_a + 8 * (E % SLOTS), lane == 0);
    constexpr int EP = (E + NK - 1) % NK;
    if (warp == EP % C::NW) {
      if (E == 0) duty(HtKind<EP>(), m - 1, mpar ^ 1u, 0u, mask);
      else duty(HtKind<EP>(), m, mpar, mask, maskn);
    }
  };
  // accumulators: A[0] band m-1 (complete after this step), A[1] band m, A[2] band m+1
  double2 A[3][NI];
#pragma unroll
  for (int q = 0; q < 3; q++)
#pragma unroll
    for (int j = 0; j < NI; j++) A[q][j] = make_double2(0.0, 0.0);
  double2* Ob = reinterpret_cast<double2*>(out + soff + (size_t)slab * Q) + (r0 * C::NCOL + 2 * cp) / 2;
  const double q3a = op.q0[2] + op.h[2] * (double)(2 * cp), q3b = q3a + op.h[2];

#pragma unroll 1
  for (; m <= nbands; m++) {
    const bool have = m < nbands;
    if (t == 0 && m + 1 < nbands) {                                  // hierarchy neighbours and y come from HBM: ask L2 one band
      const size_t bn = (size_t)(m + 1) * C::BAND;                   // early (two bands early measured slower: 3.43 vs 3.15 ms)
#pragma unroll
      for (int e = 10; e < 16; e++)
        if ((mask_line >> e) & 1u) ht_prefetch(ent[e] + bn, C::CHUNK);
      ht_prefetch(ent[16] + bn + C::BAND, C::CHUNK);
    }
    double2(&acc)[NI] = A[1];
    chunk(HtKind<0>(), [&](unsigned Sa) {                           // -Gamma_n c
#pragma unroll
      for (int j = 0; j < NI; j++) acc[j] = ht_fma2(-gam, ht_lds2(Sa + item_off(j)), acc[j]);
    });
    HtUnroll<0, 3>::run([&](auto SS) {
      constexpr int s = decltype(SS)::value;
      const double su = (up[s] >= 0) ? S->su[s] : 0.0, sd = (dn[s] >= 0) ? S->sd[s] : 0.0;
      double2 P[NI], Lc[NI];                                        // su c_up + sd c_dn,  su c_up - sd c_dn
#pragma unroll
      for (int j = 0; j < NI; j++) { P[j] = make_double2(0.0, 0.0); Lc[j] = make_double2(0.0, 0.0); }
      chunk(HtKind<1 + 3 * s>(), [&](unsigned Sa) {
#pragma unroll
        for (int j = 0; j < NI; j++) { const double2 v = ht_lds2(Sa + item_off(j)); P[j] = ht_fma2(su, v, P[j]); Lc[j] = ht_fma2(su, v, Lc[j]); }
      });
      chunk(HtKind<2 + 3 * s>(), [&](unsigned Sa) {
#pragma unroll
        for (int j = 0; j < NI; j++) { const double2 v = ht_lds2(Sa + item_off(j)); P[j] = ht_fma2(sd, v, P[j]); Lc[j] = ht_fma2(-sd, v, Lc[j]); }
      });
      const double a1f = op.a1f[s];
      chunk(HtKind<3 + 3 * s>(), [&](unsigned Sa) {                 // a1f dU/dq_s (su c_up - sd c_dn)
#pragma unroll
        for (int j = 0; j < NI; j++) {
          const double2 v = ht_lds2(Sa + item_off(j));
          acc[j].x = fma(a1f * v.x, Lc[j].x, acc[j].x);
          acc[j].y = fma(a1f * v.y, Lc[j].y, acc[j].y);
        }
      });
      const double w1 = -op.a2[s] * op.c1[s], w2 = -op.a2[s] * op.c2[s];   // -a2 D_q P, D f = c1 (f+1 - f-1) + c2 (f+2 - f-2)
      if (CMP) {                                                    // P_2, P_3 go to shared memory for the line solves
        if (have && s == 1) {
          if (m > 0) ht_wait(xbar_a + 8, (unsigned)(m - 1) & 1u);   // the results of the previous band have been read
#pragma unroll
          for (int j = 0; j < NI; j++)
            *reinterpret_cast<double2*>(g2 + (j >> 1) * C::G2_PLANE + (r0 + 16 * (j & 1)) * C::NCOL + 2 * cp) = P[j];
        }
        if (have && s == 2) {
#pragma unroll
          for (int j = 0; j < NI; j++) {
            double* g = g3 + (j >> 1) * C::G3_PLANE + 2 * cp * C::NROW + ((r0 + 16 * (j & 1)) ^ cp);
            g[0] = P[j].x; g[C::NROW] = P[j].y;
          }
          __syncwarp();
          ht_arrive_if(xbar_a, lane == 0);                          // this warp's P_2 and P_3 values are written
        }
      } else
      if (have && ((mask_line >> (3 + 3 * s)) & 1u)) {
        if (s == 0) {                                               // q_1: planes i0 = 2m (items 0, 1) and i0 + 1 (items 2, 3)
#pragma unroll
          for (int rr = 0; rr < 2; rr++) {
            const double2 f0 = P[rr], f1 = P[2 + rr];
            A[0][rr] = ht_fma2(w2, f0, A[0][rr]);                                   // row 2m-2 sees f(2m) at +2
            A[0][2 + rr] = ht_fma2(w1, f0, ht_fma2(w2, f1, A[0][2 + rr]));          // row 2m-1: +1 and +2
            A[1][rr] = ht_fma2(w1, f1, A[1][rr]);                                   // row 2m sees f(2m+1) at +1
            A[1][2 + rr] = ht_fma2(-w1, f0, A[1][2 + rr]);                          // row 2m+1 sees f(2m) at -1
            A[2][rr] = ht_fma2(-w1, f1, ht_fma2(-w2, f0, A[2][rr]));                // row 2m+2: -1 and -2
            A[2][2 + rr] = ht_fma2(-w2, f1, A[2][2 + rr]);                          // row 2m+3 sees f(2m+1) at -2
          }
        } else if (s == 1) {                                        // q_2: through the shared plane pair
          if (m > 0) ht_wait(xbar_a + 8, (unsigned)(m - 1) & 1u);   // the planes of the previous band have been read
#pragma unroll
          for (int j = 0; j < NI; j++)
            *reinterpret_cast<double2*>(g2 + (j >> 1) * C::G2_PLANE + (r0 + 16 * (j & 1)) * C::NCOL + 2 * cp) = P[j];
        } else {                                                    // q_3: the 16 lanes of a row
#pragma unroll
          for (int j = 0; j < NI; j++) {
            const double2 own = P[j];
            double ly = __shfl_up_sync(0xffffffffu, own.y, 1, 16), rx = __shfl_down_sync(0xffffffffu, own.x, 1, 16);
            double lx = __shfl_up_sync(0xffffffffu, own.x, 1, 16), ry = __shfl_down_sync(0xffffffffu, own.y, 1, 16);
            if (cp == 0) { ly = 0.0; lx = 0.0; }
            if (cp == 15) { rx = 0.0; ry = 0.0; }
            // pair (i, i+1): neighbours i-2 .. i+3 = lx ly [own.x own.y] rx ry
            acc[j].x = fma(w1, own.y - ly, fma(w2, rx - lx, acc[j].x));
            acc[j].y = fma(w1, rx - own.x, fma(w2, ry - ly, acc[j].y));
          }
        }
      } else if (!CMP && s == 1 && have) {                          // nothing to exchange for this slab: keep the barriers in step
        if (m > 0) ht_wait(xbar_a + 8, (unsigned)(m - 1) & 1u);
#pragma unroll
        for (int j = 0; j < NI; j++)
          *reinterpret_cast<double2*>(g2 + (j >> 1) * C::G2_PLANE + (r0 + 16 * (j & 1)) * C::NCOL + 2 * cp) = make_double2(0.0, 0.0);
      }
      if (!CMP && s == 1 && have) { __syncwarp(); ht_arrive_if(xbar_a, lane == 0); }     // this warp's P_2 values are written
    });
    HtUnroll<0, 6>::run([&](auto HH) {                              // V'_s (hd c(n-e_s, k+e_s) + hu c(n+e_s, k-e_s))
      constexpr int hh = decltype(HH)::value, s = hh / 2;
      const double hc = (hh & 1) ? S->hu[s] : S->hd[s];
      chunk(HtKind<10 + hh>(), [&](unsigned Sa) {
#pragma unroll
        for (int j = 0; j < NI; j++) {
          const double2 v = ht_lds2(Sa + item_off(j));
          const double qa = (s == 0) ? op.q0[0] + op.h[0] * (double)(2 * m + (j >> 1))
                          : (s == 1 ? op.q0[1] + op.h[1] * (double)(r0 + 16 * (j & 1)) : q3a);
          const double qb = (s == 2) ? q3b : qa;
          acc[j].x = fma(hc * fma(op.VSL[s], qa, op.VLL[s]), v.x, acc[j].x);
          acc[j].y = fma(hc * fma(op.VSL[s], qb, op.VLL[s]), v.y, acc[j].y);
        }
      });
    });
    if (CMP && have) {
      // 128 lines per band (2 planes x 32 columns along q_2, 2 planes x 32 rows along q_3), 16 per warp.  T d = r, T = tridiag(1/3, 1, 1/3), r_i = ca (P_{i+1} - P_{i-1}) + cb (P_{i+2} - P_{i-2}) with zero
      // ghosts (R9), by the Thomas recurrence with the host-tabulated reciprocal pivots of k_hermite_compact_line, in place.
      ht_wait(xbar_a, (unsigned)m & 1u);
      if (lane < 16) {                                              // warps 0-3: q_2 lines (plane, column); warps 4-7: q_3 lines (plane, row)
        const int ln = (warp & 3) * 16 + lane, pl = ln >> 5, i0 = ln & 31;
        if (warp < 4) ht_thomas32<C::NCOL, false>(g2 + pl * C::G2_PLANE, i0, tab_a, op.ca[1], op.cb[1]);
        else ht_thomas32<C::NROW, true>(g3 + pl * C::G3_PLANE, i0, tab_a, op.ca[2], op.cb[2]);
      }
      __syncwarp();
      ht_arrive_if(xbar_a + 16, lane == 0);
      ht_wait(xbar_a + 16, (unsigned)m & 1u);
      const double f2 = -op.a2[1], f3 = -op.a2[2];
#pragma unroll
      for (int j = 0; j < NI; j++) {
        const double2 d2 = *reinterpret_cast<const double2*>(g2 + (j >> 1) * C::G2_PLANE + (r0 + 16 * (j & 1)) * C::NCOL + 2 * cp);
        const double* g = g3 + (j >> 1) * C::G3_PLANE + 2 * cp * C::NROW + ((r0 + 16 * (j & 1)) ^ cp);
        acc[j].x = fma(f2, d2.x, fma(f3, g[0], acc[j].x));
        acc[j].y = fma(f2, d2.y, fma(f3, g[C::NROW], acc[j].y));
      }
      __syncwarp();
      ht_arrive_if(xbar_a + 8, lane == 0);
    }
    if (!CMP && have) {                                             // q_2 stencil of P_2
      ht_wait(xbar_a, (unsigned)m & 1u);
      const double w1 = -op.a2[1] * op.c1[1], w2 = -op.a2[1] * op.c2[1];
#pragma unroll
      for (int j = 0; j < NI; j++) {
        // rows r0 (j even) and r0 + 16 (j odd): the lower neighbours of the first and the upper ones of the second may be ghosts
        const double* g = g2 + (j >> 1) * C::G2_PLANE + (r0 + 16 * (j & 1)) * C::NCOL + 2 * cp;
        const bool v1 = (j & 1) ? r0 <= 14 : r0 >= 1, v2 = (j & 1) ? r0 <= 13 : r0 >= 2;   // the +-1 / +-2 neighbour on the ghost side exists
        const int o1 = (j & 1) ? C::NCOL : -C::NCOL;
        const double2 z = make_double2(0.0, 0.0);
        const double2 e1 = v1 ? *reinterpret_cast<const double2*>(g + o1) : z, e2 = v2 ? *reinterpret_cast<const double2*>(g + 2 * o1) : z;
        const double2 i1 = *reinterpret_cast<const double2*>(g - o1), i2 = *reinterpret_cast<const double2*>(g - 2 * o1);
        const double2 u1 = (j & 1) ? e1 : i1, d1 = (j & 1) ? i1 : e1, u2 = (j & 1) ? e2 : i2, d2 = (j & 1) ? i2 : e2;
        acc[j].x = fma(w1, u1.x - d1.x, fma(w2, u2.x - d2.x, acc[j].x));
        acc[j].y = fma(w1, u1.y - d1.y, fma(w2, u2.y - d2.y, acc[j].y));
      }
      __syncwarp();
      ht_arrive_if(xbar_a + 8, lane == 0);
    }
    chunk(HtKind<16>(), [&](unsigned Sa) {                          // band m-1 is complete: out = a y + c F
      double2* O = Ob + (size_t)(m - 1) * (C::BAND / 2);
#pragma unroll
      for (int j = 0; j < NI; j++) {
        const double2 yv = ht_lds2(Sa + item_off(j));
        ht_st2(O + item_off(j) / 16, make_double2(fma(c, A[0][j].x, a * yv.x), fma(c, A[0][j].y, a * yv.y)), pol_str);
      }
    });
    HtUnroll<17, NK>::run([&](auto KP) { chunk(KP, [&](unsigned) {}); });   // padding kinds: barriers only
#pragma unroll
    for (int j = 0; j < NI; j++) { A[0][j] = A[1][j]; A[1][j] = A[2][j]; A[2][j] = make_double2(0.0, 0.0); }
    mask = maskn;
    maskn = __shfl_sync(0xffffffffu, step_mask(m + 2), 0);
    mpar ^= 1u;
  }
}
