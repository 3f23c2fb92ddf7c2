// Internal declarations shared by the host API (chfpe_api.cu) and the kernels (chfpe_kernels.cu).
// Not part of the C-ABI; nothing here is used by the oracle.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>
#include "../../include/chfpe.h"

#define CHFPE_MAXAX 6

// Device-side view of the operator: passed BY VALUE to every kernel (< 1 KB of kernel parameter space).
// Internal axis order ("q-major / p-minor bricks"): a = 0..M-1 are q_1..q_M, a = M..2M-1 are p_1..p_M,
// last axis fastest, so all momenta of one q-point form one contiguous "p-brick" of pb cells.
struct DevOp {
  int M, nax, K, scheme, gauge;
  int closure, depth;                 // CHFPE_CLOSURE_*; N (elements with sum n = N are the top level)
  int expect_pbrick;                  // expectation values by k_expect_pbrick (CHFPE_EXPECT_PBRICK=0: generic reduction)
  int n[CHFPE_MAXAX];                 // points per internal axis
  long long st[CHFPE_MAXAX];          // internal strides (doubles)
  long long cells, nqc, pb;           // cells per element, q-points, p-brick size
  double x0[CHFPE_MAXAX], h[CHFPE_MAXAX];
  double c1[CHFPE_MAXAX], c2[CHFPE_MAXAX];   // pre-multiplied stencil coefficients (+-1, +-2 neighbours)
  double inv_mass[3], kup[3], kdn[3], cdn[3], VLL[3], VSL[3], beta;
  double gam[3];                      // gamma_s (terminator closure: Gamma_{n+e_s} = Gamma_n + gamma_s)
  double cqw[3][4];                   // CENTRAL4: -(1/m_s)/(12 h_qs) x stencil weight of the q_s neighbour +1, -1, +2, -2
  double dV;
  const double* dU[3];                // dU/dq_s on the q-subgrid, q_1 slowest   (device)
  const double* eU;                   // exp(-beta U/2) (sqrt gauge) or exp(-beta U) (W gauge) on the q-subgrid
  const double* ep[3];                // exp(-beta p^2/(4m)) resp. exp(-beta p^2/(2m)) per p-axis
  const int* up;                      // [K][3] element index of n + e_s or -1
  const int* dn;                      // [K][3] element index of n - e_s or -1
  const int* nvec;                    // [K][3]
  const double* Gamma;                // [K] sum_s n_s gamma_s
};

// Launch plan of the brick kernels (chfpe_brick.cu, chfpe_tma.cu): bricks = all momenta of one (element, q-point).
struct BrickPlan {
  int enabled;
  int P1, P2, P3, PB2;                // p-extents, PB2 = P2*P3 (two modes: P2 = 1)
  int vn[3];                          // q-extents as the three-mode kernels see them (two modes: vn[1] = 1)
  int g;                              // elements per lock-step group (L2 window)
  int n_groups;
  long long blocks_per_full_group;    // g * nqc
  long long rest;                     // q-points per q1 plane
  int bpc;                            // consecutive bricks per CTA of the brick kernel
  int q2chunk;                        // q_2 rows per sweep chunk (= n_q2 unless five q_1 planes exceed the L2 budget)
  const int* order;                   // [K] element order, groups contiguous (device)
  const int* pos;                     // [K] position of element k in `order`
  const int4* table;                  // [K * n_q] brick order (device), see decode_brick_id
  int l2mode;                         // bit 0: once-touched data evict_first, bit 1: window data evict_last
  int minb;                           // CTAs per SM the specialised kernel is compiled for (register budget)
  int npass;                          // passes over blocks of P1/npass planes per brick (large bricks)
  int split;                          // p_1 segments (thread groups) per brick in the specialised kernel
  int fixed;                          // a compile-time specialisation (k_stage_brick3<P1,P2,P3,...>) exists
  // bulk-copy fed kernel (chfpe_tma.cu): a CTA owns one q_3 line of one p_1 part of the bricks
  int tma;                            // use it (CENTRAL4, three-mode view, a compile-time specialisation exists)
  int tma_npart, tma_nseg, tma_slots, tma_ring;
  int n_lines;                        // K * n_q1 * n_q2 * tma_npart
  const int4* lines;                  // [n_lines] sweep order, see decode_line
};

#ifdef __CUDACC__
// Brick order of the three-mode kernels: element group -> q_2 chunk -> q_1 plane -> element in group -> (q_2, q_3).
// The five q_1 planes (of one chunk of q_2 rows) of the group's stage input are the L2 reuse window.
struct BrickId { int k, G, iq[3], own; long long ql; };
// The order is tabulated once per handle by the host (make_brick_plan): one int4 per brick,
// {k, linear q index, iq_1 | iq_2 << 10 | iq_3 << 20, group | own-mask << 16}; own-mask bit 2s (+1) says that the
// up (down) neighbour along s belongs to the same group, i.e. its bricks are part of the L2 window.
__device__ __forceinline__ BrickId decode_brick_id(const DevOp&, const BrickPlan& bp, long long L) {
  const int4 t = __ldg(bp.table + L);
  BrickId b;
  b.k = t.x;
  b.ql = t.y;
  b.iq[0] = t.z & 1023; b.iq[1] = (t.z >> 10) & 1023; b.iq[2] = (t.z >> 20) & 1023;
  b.G = t.w & 0xffff;
  b.own = t.w >> 16;
  return b;
}
#endif

struct DevObs {                       // observable polynomial, Eq. (13)-(14)
  double c0, lin_q[3], quad[3][3], lin_p[3];
};

// COMPACT6 (step a9): per-axis elimination factors of tridiag(1/3, 1, 1/3) (device), see chfpe_compact.cu
struct CompactTables {
  const double* bet[CHFPE_MAXAX];
  const double* cfac[CHFPE_MAXAX];
  const double* ibet[CHFPE_MAXAX];    // 1 / bet (recurrence as two FMAs in k_compact_pbrick)
};

enum ReduceMode { RED_EXPECT = 0, RED_SUMSQ = 1, RED_SUM = 2 };

struct chfpe_handle {
  chfpe_desc desc;
  std::vector<chfpe_monomial> U;
  DevOp op;
  DevOp op3;                          // the same operator as a three-mode one (identical for M = 3), brick kernels
  BrickPlan bp;
  CompactTables ct;
  double* scratch;                    // COMPACT6 only: three element-sized arrays (G, D, F)
  cudaStream_t stream;
  int K, batch, n_arrays;
  long long cells;
  size_t state_doubles;               // K * cells
  double* arrays;                     // n_arrays * state_doubles, carved from the workspace
  // slot b uses arrays[3b] (state y), arrays[3b+1], arrays[3b+2] (stage buffers); optional spare array last
  double* partial;                    // reduction scratch
  double* results;                    // batch doubles (device)
  int red_blocks;
  std::vector<int> elem;              // host copy [K][3]
  bool initialised;
  bool norm_ref_valid;                // norm guard of chfpe_step: reference taken since the last non-propagating change
  std::vector<double> norm_ref;       // per slot: sum of squares of the state at that point
  int64_t launches;
  int coop_mode;                      // CHFPE_COOP: 0 off, 1 tiny states only, 2 every L2-resident state
  bool coop;                          // persistent cooperative kernel allowed for L2-resident states
  bool prof;                          // bracket every stage launch with CUDA events (chfpe_profile_*)
  std::vector<cudaEvent_t> prof_ev;   // pairs (start, stop); prof_used of them are pending
  size_t prof_used;
  std::string err;
  double* y(int b) const { return arrays + (size_t)(3 * b) * state_doubles; }
  double* va(int b) const { return arrays + (size_t)(3 * b + 1) * state_doubles; }
  double* vb(int b) const { return arrays + (size_t)(3 * b + 2) * state_doubles; }
  double* spare() const { return arrays + (size_t)(3 * batch) * state_doubles; }
};

// ---- launchers implemented in chfpe_kernels.cu (all asynchronous on `s`; return the launch count) ----
// out = a*y + c*F(in) for slots [b0, b0+nb); slot stride = 3*state_doubles for all three pointers.
int launch_stage(const DevOp& op, const double* in, const double* y, double* out, double a, double c,
                 int nb, size_t slot_stride, cudaStream_t s);
// COMPACT6 path (chfpe_compact.cu): element-by-element assembly from whole-array Pade derivatives
int launch_stage_compact(const DevOp& op, const CompactTables& ct, const double* in, const double* y, double* out, double a,
                         double c, int nb, size_t slot_stride, double* scratch, cudaStream_t s);
int launch_kick_compact(const DevOp& op, const CompactTables& ct, const DevObs& o, const double* in, double* out, int nb,
                        size_t slot_stride, double* scratch, cudaStream_t s);
// persistent cooperative kernel for L2-resident states (one replica): n_samples x (stride steps [+ <O> sample]);
// returns 0 if a cooperative launch is not possible
int launch_steps_coop(const DevOp& op, const DevObs& o, double* y, double* va, double* vb, double dt,
                      long long n_samples, long long stride, int do_expect, double* partial, int max_blocks,
                      double* results, cudaStream_t s);
// same operation by the brick kernel (chfpe_brick.cu); requires bp.enabled
int launch_stage_brick(const DevOp& op, const BrickPlan& bp, const double* in, const double* y, double* out,
                       double a, double c, int nb, size_t slot_stride, cudaStream_t s);
// bulk-copy fed variant (chfpe_tma.cu): one CTA per q_3 line and p_1 part, producer thread + consumer warps
int tma_has_fixed(int M, int P1, int P2, int P3, int npart, int nseg, int slots, int ring);
int tma_configure(const BrickPlan& bp);
int launch_stage_tma(const DevOp& op, const BrickPlan& bp, const double* in, const double* y, double* out, double a,
                     double c, int nb, size_t slot_stride, cudaStream_t s);
// one-off opt-in to > 48 KB dynamic shared memory for the brick kernels; returns a cudaError_t as int
int brick_configure(const BrickPlan& bp, int M);
int brick_has_fixed(int M, int P1, int P2, int P3, int split, int minb, int npass);
// terminator closure on top of a stage kernel that does not know it (brick / bulk-copy kernels):
// out += c * (slaved-element coupling of every top-level element), see terminator_value in chfpe_kernels.cu
int launch_terminator_add(const DevOp& op, const double* in, double* out, double c, int nb, size_t slot_stride,
                          cudaStream_t s);
// x <- Kick_obs(x) in place, one CTA per p-brick (M >= 2, explicit schemes); returns 0 if it does not apply
int launch_kick_brick(const DevOp& op, const DevObs& o, double* x, int nb, size_t slot_stride, cudaStream_t s);
// out = Kick_obs(in) on every element, slots [b0, b0+nb)
int launch_kick(const DevOp& op, const DevObs& o, const double* in, double* out, int nb, size_t slot_stride,
                cudaStream_t s);
// results[b*res_stride] = scale * sum over ncells cells starting at element k of slot b of the integrand;
// deterministic two-pass reduction (fixed block partition, fixed-order final pass)
int launch_reduce(const DevOp& op, const DevObs& o, int mode, const double* x, int k, long long ncells,
                  int nb, size_t slot_stride, double scale, double* partial, int red_blocks, double* results,
                  long long res_stride, cudaStream_t s);
// element 0 <- unnormalised equilibrium profile, other elements <- 0 (one slot)
int launch_init_eq(const DevOp& op, double* x, cudaStream_t s);
int launch_scale(double* x, long long n, const double* denom_dev, double mult, cudaStream_t s);
// layout conversion between canonical (q1,p1,...,qM,pM) and internal (q..., p...) for all K elements
int launch_permute(const DevOp& op, const double* src, double* dst, int to_internal, cudaStream_t s);
