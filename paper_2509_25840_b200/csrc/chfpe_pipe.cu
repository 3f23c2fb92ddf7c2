// Plane-pipelined RK-stage kernel (steps a1-a3 of DESIGN.md) for three modes on sm_100a.
//
// Same arithmetic as chfpe_brick.cu (Eq. (8)-(12)), different data movement.  A persistent CTA walks
// a list of p-bricks (element k, q-point) in the q_1-plane / element-group order and cuts every brick into its P1
// momentum planes (P2*P3 contiguous doubles per array).  A producer warp streams, for every plane, the rows the
// plane needs -- own stage input, the up/down hierarchy neighbours, the 12 q-neighbour planes, y -- into a ring of
// shared-memory stages with 1-D bulk async copies (cp.async.bulk, the TMA engine; completion on an mbarrier), so
// the number of bytes in flight is set by shared memory, not by registers.  The consumer warps (one thread per cell
// of the plane) march along p_1: the p_1 stencil of G_1 lives in a register ring (scatter form), G_2 / G_3 are
// exchanged through a small zero-padded shared plane, and plane j-2 is written as soon as plane j has been added.
#include "chfpe_internal.cuh"

namespace {

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(void* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(void* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(void* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(void* bar, unsigned parity) {
  unsigned done;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.b32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  } while (!done);
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, void* bar, unsigned long long pol) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
          smem_u32(dst)),
      "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol)
      : "memory");
}
__device__ __forceinline__ void bulk_prefetch_l2(const void* src, unsigned bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ unsigned long long pipe_policy(int kind) {
  unsigned long long p;
  if (kind == 1) asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  else if (kind == 2) asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  else asm("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ void st_stream(double* p, double v, unsigned long long pol) {
  asm volatile("st.global.L2::cache_hint.f64 [%0], %1, %2;" ::"l"(p), "d"(v), "l"(pol) : "memory");
}

// rows of one stage
enum { ROW_XK = 0, ROW_NB = 1 /* +2s (up), +2s+1 (down) */, ROW_Q = 7 /* +4s: -2,-1,+1,+2 */, ROW_Y = 19, NROWS = 20 };

// what every thread of the CTA needs to know about a brick (CTA-uniform)
struct BrickInfo {
  int k, G, own;
  long long ql;
  int iq[3];
  size_t elem_off;       // k*cells + ql*pb (doubles, inside one replica)
  size_t slot_off;       // replica offset
};

__device__ __forceinline__ BrickInfo decode_brick(const DevOp& op, const BrickPlan& bp, long long Lt, size_t slot_stride) {
  BrickInfo b;
  const long long per_slot = (long long)op.K * op.nqc;
  const long long slot = Lt / per_slot;
  long long L = Lt - slot * per_slot;
  const BrickId id = decode_brick_id(op, bp, L);
  b.G = id.G; b.k = id.k; b.ql = id.ql; b.own = id.own;
  b.iq[0] = id.iq[0]; b.iq[1] = id.iq[1]; b.iq[2] = id.iq[2];
  b.elem_off = (size_t)b.k * op.cells + (size_t)b.ql * op.pb;
  b.slot_off = (size_t)slot * slot_stride;
  return b;
}

template <int P1, int P2, int P3, int STAGES>
struct PipeCfg {
  static constexpr int PLANE = P2 * P3;                          // cells per momentum plane
  static constexpr int NCONS = ((PLANE + 31) / 32) * 32;         // consumer threads
  static constexpr int NT = NCONS + 32;                          // + one producer warp
  static constexpr int X2 = (P2 + 4) * P3, X3 = P2 * (P3 + 4);   // exchange planes of G_2, G_3
  static constexpr int XCH = X2 + X3;
  static constexpr size_t SMEM = sizeof(double) * ((size_t)STAGES * NROWS * PLANE + 2 * XCH) + 16 * STAGES + 8 * NROWS + 16;
  static constexpr int MIN_CTAS = (SMEM <= 110 * 1024) ? 2 : 1;
};

template <int P1, int P2, int P3, int STAGES>
__global__ void __launch_bounds__(PipeCfg<P1, P2, P3, STAGES>::NT, PipeCfg<P1, P2, P3, STAGES>::MIN_CTAS)
k_stage_pipe(DevOp op, BrickPlan bp, const double* __restrict__ in, const double* y, double* out, double a, double cc,
             size_t slot_stride, int y_is_in, long long n_bricks) {
  using C = PipeCfg<P1, P2, P3, STAGES>;
  constexpr int PLANE = C::PLANE;
  constexpr unsigned ROW_BYTES = PLANE * sizeof(double);
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double* stages = reinterpret_cast<double*>(smem_raw);
  double* xch = stages + (size_t)STAGES * NROWS * PLANE;
  unsigned long long* full = reinterpret_cast<unsigned long long*>(xch + 2 * C::XCH);
  unsigned long long* empty = full + STAGES;

  const int tid = threadIdx.x;
  if (tid == 0) {
    for (int s = 0; s < STAGES; s++) { mbar_init(full + s, 1); mbar_init(empty + s, C::NCONS / 32); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  for (int i = tid; i < 2 * C::XCH; i += C::NT) xch[i] = 0.0;       // ghost rows / columns stay zero for ever
  __syncthreads();

  const bool wide = (op.scheme == CHFPE_CENTRAL4);

  if (tid >= C::NCONS) {
    // ======================= producer warp: lane r owns row r of every stage =======================
    const int lane = tid - C::NCONS;
    const unsigned long long pol_own = pipe_policy((bp.l2mode & 2) ? 2 : 0);
    const unsigned long long pol_str = pipe_policy((bp.l2mode & 1) ? 1 : 0);
    long long it = 0;
    for (long long Lt = blockIdx.x; Lt < n_bricks; Lt += gridDim.x) {
      const BrickInfo b = decode_brick(op, bp, Lt, slot_stride);
      const double* X = in + b.slot_off;
      const double* src = nullptr;                                    // this lane's row of plane 0, or absent
      bool own = true;                                                // L2 lines belong to the q_1-plane window
      if (lane == ROW_XK) {
        src = X + b.elem_off;
      } else if (lane < ROW_Q) {
        const int s = (lane - ROW_NB) >> 1;
        const int kn = ((lane - ROW_NB) & 1) ? __ldg(op.dn + 3 * b.k + s) : __ldg(op.up + 3 * b.k + s);
        if (kn >= 0) {
          src = X + (size_t)kn * op.cells + (size_t)b.ql * op.pb;
          own = ((b.own >> (lane - ROW_NB)) & 1) != 0;
        }
      } else if (lane < ROW_Y) {
        const int s = (lane - ROW_Q) >> 2, r = (lane - ROW_Q) & 3;
        const int off = (r < 2) ? r - 2 : r - 1;                      // -2, -1, +1, +2
        const int i = (s == 0 ? b.iq[0] : (s == 1 ? b.iq[1] : b.iq[2])) + off;
        const int n = (s == 0 ? op.n[0] : (s == 1 ? op.n[1] : op.n[2]));
        const long long st = (s == 0 ? op.st[0] : (s == 1 ? op.st[1] : op.st[2]));
        if (i >= 0 && i < n && (wide || off == 1 || off == -1)) src = X + b.elem_off + off * st;
      } else if (lane == ROW_Y) {
        if (!y_is_in) { src = y + b.slot_off + b.elem_off; own = false; }
      }
      const unsigned n_present = __popc(__ballot_sync(0xffffffffu, src != nullptr));
      const unsigned long long pol = own ? pol_own : pol_str;
      // ask L2 for the HBM-sourced bricks of the NEXT brick of this CTA while this one is streamed
      {
        const long long Ln = Lt + gridDim.x;
        if (Ln < n_bricks && (lane < ROW_Q || lane == ROW_Y)) {
          const BrickInfo nb = decode_brick(op, bp, Ln, slot_stride);
          const double* Xn = in + nb.slot_off;
          constexpr unsigned BB = P1 * ROW_BYTES;
          const double* pf = nullptr;
          if (lane == ROW_XK) pf = Xn + nb.elem_off;
          else if (lane == ROW_Y) pf = y_is_in ? nullptr : y + nb.slot_off + nb.elem_off;
          else {
            const int s = (lane - ROW_NB) >> 1;
            const int kn = ((lane - ROW_NB) & 1) ? __ldg(op.dn + 3 * nb.k + s) : __ldg(op.up + 3 * nb.k + s);
            if (kn >= 0) pf = Xn + (size_t)kn * op.cells + (size_t)nb.ql * op.pb;
          }
          if (pf) bulk_prefetch_l2(pf, BB);
        }
      }
      for (int j = 0; j < P1; j++, it++) {
        const int sg = (int)(it % STAGES);
        const unsigned ph = (unsigned)((it / STAGES) & 1);
        if (lane == 0) {
          mbar_wait(empty + sg, ph ^ 1u);
          mbar_expect_tx(full + sg, n_present * ROW_BYTES);
        }
        __syncwarp();
        if (src && lane < NROWS)
          bulk_g2s(stages + ((size_t)sg * NROWS + lane) * PLANE, src + (size_t)j * PLANE, ROW_BYTES, full + sg, pol);
      }
    }
    return;
  }

  // =================================== consumer warps ===================================
  const unsigned long long pol_out = pipe_policy((bp.l2mode & 1) ? 1 : 0);
  const bool active = tid < PLANE;
  const int cell = active ? tid : 0;
  const int i2 = cell / P3, i3 = cell - i2 * P3;
  const int x2 = (i2 + 2) * P3 + i3;                                 // own position in the G_2 exchange plane
  const int x3 = C::X2 + i2 * (P3 + 4) + i3 + 2;                     // and in the G_3 exchange plane
  const double p1_0 = op.x0[3], h1 = op.h[3];
  const double p2 = op.x0[4] + i2 * op.h[4], p3 = op.x0[5] + i3 * op.h[5];
  const double w1p = wide ? -op.c2[3] : op.c1[3], w2p = wide ? -op.c2[4] : op.c1[4], w3p = wide ? -op.c2[5] : op.c1[5];
  const double w8 = wide ? 8.0 * w1p : w1p, w1 = wide ? w1p : 0.0;
  double cq[3];
#pragma unroll
  for (int s = 0; s < 3; s++) cq[s] = -(wide ? -op.c2[s] : op.c1[s]) * op.inv_mass[s];
  cq[1] *= p2; cq[2] *= p3;

  long long it = 0;
  for (long long Lt = blockIdx.x; Lt < n_bricks; Lt += gridDim.x) {
    const BrickInfo b = decode_brick(op, bp, Lt, slot_stride);
    const double Gam = __ldg(op.Gamma + b.k);
    double dU[3], cu[3], cd[3], pu[3], pd[3];
    bool hu[3], hd[3], qm2[3], qm1[3], qp1[3], qp2[3];
#pragma unroll
    for (int s = 0; s < 3; s++) {
      const double qs = op.x0[s] + b.iq[s] * op.h[s];
      const double Vp = fma(op.VSL[s], qs, op.VLL[s]);
      dU[s] = __ldg(op.dU[s] + b.ql);
      hu[s] = __ldg(op.up + 3 * b.k + s) >= 0;
      hd[s] = __ldg(op.dn + 3 * b.k + s) >= 0;
      cu[s] = hu[s] ? Vp : 0.0;
      cd[s] = hd[s] ? __ldg(op.nvec + 3 * b.k + s) * op.cdn[s] * Vp : 0.0;
      pu[s] = cu[s] * op.kup[s]; pd[s] = cd[s] * op.kdn[s];
      const int i = b.iq[s], n = op.n[s];
      qm2[s] = wide && i >= 2; qm1[s] = i >= 1; qp1[s] = i + 1 < n; qp2[s] = wide && i + 2 < n;
    }
    double* obase = out + b.slot_off + b.elem_off + cell;

    double acc[P1], yv[P1];
#pragma unroll
    for (int j = 0; j < P1; j++) acc[j] = 0.0;

#pragma unroll
    for (int j = 0; j < P1; j++, it++) {
      const int sg = (int)(it % STAGES);
      const unsigned ph = (unsigned)((it / STAGES) & 1);
      mbar_wait(full + sg, ph);
      const double* S = stages + (size_t)sg * NROWS * PLANE + cell;
      const double xk = S[ROW_XK * PLANE];
      double g[3], pw = -Gam * xk;
#pragma unroll
      for (int s = 0; s < 3; s++) {
        const double xu = hu[s] ? S[(ROW_NB + 2 * s) * PLANE] : 0.0;
        const double xd = hd[s] ? S[(ROW_NB + 2 * s + 1) * PLANE] : 0.0;
        double gg = dU[s] * xk;
        gg = fma(cu[s], xu, gg);
        g[s] = fma(cd[s], xd, gg);
        const double ps = (s == 0) ? fma((double)j, h1, p1_0) : (s == 1 ? p2 : p3);
        pw = fma(ps, fma(pd[s], xd, pu[s] * xu), pw);
      }
#pragma unroll
      for (int s = 0; s < 3; s++) {
        const double fm2 = qm2[s] ? S[(ROW_Q + 4 * s + 0) * PLANE] : 0.0;
        const double fm1 = qm1[s] ? S[(ROW_Q + 4 * s + 1) * PLANE] : 0.0;
        const double fp1 = qp1[s] ? S[(ROW_Q + 4 * s + 2) * PLANE] : 0.0;
        const double fp2 = qp2[s] ? S[(ROW_Q + 4 * s + 3) * PLANE] : 0.0;
        const double d1 = fp1 - fm1;
        const double e = wide ? fma(8.0, d1, -(fp2 - fm2)) : d1;
        const double c = (s == 0) ? cq[0] * fma((double)j, h1, p1_0) : cq[s];
        pw = fma(c, e, pw);
      }
      yv[j] = y_is_in ? xk : S[ROW_Y * PLANE];
      // G_2, G_3 -> exchange plane (ping-pong), release the stage, then one consumer barrier
      double* xb = xch + (j & 1) * C::XCH;
      if (active) { xb[x2] = g[1]; xb[x3] = g[2]; }
      __syncwarp();
      if ((tid & 31) == 0) mbar_arrive(empty + sg);
      asm volatile("bar.sync 1, %0;" ::"r"(C::NCONS) : "memory");
      {
        const double* a2 = xb + x2;
        const double* a3 = xb + x3;
        const double d2 = a2[P3] - a2[-P3];
        const double d3 = a3[1] - a3[-1];
        double e2 = d2, e3 = d3;
        if (wide) {
          e2 = fma(8.0, d2, -(a2[2 * P3] - a2[-2 * P3]));
          e3 = fma(8.0, d3, -(a3[2] - a3[-2]));
        }
        pw = fma(w2p, e2, pw);
        pw = fma(w3p, e3, pw);
      }
      acc[j] += pw;
      if (j >= 1) acc[j - 1] = fma(w8, g[0], acc[j - 1]);             // D_{p_1} G_1 in scatter form
      if (j + 1 < P1) acc[j + 1] = fma(-w8, g[0], acc[j + 1]);
      if (j >= 2) acc[j - 2] = fma(-w1, g[0], acc[j - 2]);
      if (j + 2 < P1) acc[j + 2] = fma(w1, g[0], acc[j + 2]);
      if (j >= 2 && active) st_stream(obase + (size_t)(j - 2) * PLANE, fma(cc, acc[j - 2], a * yv[j - 2]), pol_out);
    }
    if (active) {
      st_stream(obase + (size_t)(P1 - 2) * PLANE, fma(cc, acc[P1 - 2], a * yv[P1 - 2]), pol_out);
      st_stream(obase + (size_t)(P1 - 1) * PLANE, fma(cc, acc[P1 - 1], a * yv[P1 - 1]), pol_out);
    }
  }
}

}  // namespace

#define PIPE_SPECIALISATIONS(X) X(16, 16, 16, 2) X(16, 16, 16, 4) X(8, 8, 8, 2)

int pipe_has_fixed(int M, int P1, int P2, int P3, int stages) {
  if (M != 3) return 0;
#define X(A, B, C, S) if (P1 == A && P2 == B && P3 == C && stages == S) return 1;
  PIPE_SPECIALISATIONS(X)
#undef X
  return 0;
}

size_t pipe_smem_bytes(const BrickPlan& bp) {
#define X(A, B, C, S) \
  if (bp.P1 == A && bp.P2 == B && bp.P3 == C && bp.pipe_stages == S) return PipeCfg<A, B, C, S>::SMEM;
  PIPE_SPECIALISATIONS(X)
#undef X
  return 0;
}

int pipe_configure(const BrickPlan& bp) {
  cudaError_t e = cudaErrorInvalidValue;
#define X(A, B, C, S)                                                                                          \
  if (bp.P1 == A && bp.P2 == B && bp.P3 == C && bp.pipe_stages == S)                                           \
    e = cudaFuncSetAttribute(k_stage_pipe<A, B, C, S>, cudaFuncAttributeMaxDynamicSharedMemorySize,            \
                             (int)PipeCfg<A, B, C, S>::SMEM);
  PIPE_SPECIALISATIONS(X)
#undef X
  return (int)e;
}

int launch_stage_pipe(const DevOp& op, const BrickPlan& bp, const double* in, const double* y, double* out, double a,
                      double c, int nb, size_t slot_stride, cudaStream_t s) {
  const long long n_bricks = (long long)nb * op.K * op.nqc;
  const int y_is_in = (y == in) ? 1 : 0;
  long long grid = (long long)bp.pipe_ctas;
  if (grid > n_bricks) grid = n_bricks;
#define X(A, B, C, S)                                                                                          \
  if (bp.P1 == A && bp.P2 == B && bp.P3 == C && bp.pipe_stages == S)                                           \
    k_stage_pipe<A, B, C, S><<<(unsigned)grid, PipeCfg<A, B, C, S>::NT, PipeCfg<A, B, C, S>::SMEM, s>>>(       \
        op, bp, in, y, out, a, c, slot_stride, y_is_in, n_bricks);
  PIPE_SPECIALISATIONS(X)
#undef X
  return 1;
}
