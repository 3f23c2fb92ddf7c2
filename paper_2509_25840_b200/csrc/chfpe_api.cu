// Host side of the C-ABI (include/chfpe.h): validation, setup tables (step a0), workspace carving and the
// drivers that sequence kernel launches (equilibrate a6, step a1-a3, kick a4, expect a5, R1 a7, R2 a8).
// No arithmetic of the method runs on the host beyond the one-off tables of `create`.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include "chfpe_internal.cuh"
#include "chfpe_poly.h"

static thread_local std::string g_create_err;

#define FAIL(h, code, msg)                  \
  do {                                      \
    (h)->err = (msg);                       \
    return (code);                          \
  } while (0)

#define CU(h, call)                                              \
  do {                                                           \
    cudaError_t e_ = (call);                                     \
    if (e_ != cudaSuccess) {                                     \
      (h)->err = std::string(#call) + ": " + cudaGetErrorString(e_); \
      return CHFPE_ERR_CUDA;                                     \
    }                                                            \
  } while (0)

static size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

static int enumerate_elements(int M, int depth, std::vector<int>* out) {
  int K = 0;
  for (int lev = 0; lev <= depth; lev++) {
    for (int a = lev; a >= 0; a--) {
      if (M == 1) { if (a != lev) break; if (out) { out->push_back(a); out->push_back(0); out->push_back(0); } K++; continue; }
      for (int b = lev - a; b >= 0; b--) {
        if (M == 2) { if (b != lev - a) break; if (out) { out->push_back(a); out->push_back(b); out->push_back(0); } K++; continue; }
        if (out) { out->push_back(a); out->push_back(b); out->push_back(lev - a - b); }
        K++;
      }
    }
  }
  return K;
}

static int validate(const chfpe_desc* d, std::string* why) {
  if (!d) { *why = "null descriptor"; return CHFPE_ERR_INVALID; }
  if (d->n_modes < 1 || d->n_modes > 3) { *why = "n_modes must be 1..3"; return CHFPE_ERR_INVALID; }
  if (d->depth < 0 || d->depth > 64) { *why = "depth out of range"; return CHFPE_ERR_INVALID; }
  if (!(d->beta > 0)) { *why = "beta must be > 0"; return CHFPE_ERR_INVALID; }
  if (d->scheme != CHFPE_CENTRAL4 && d->scheme != CHFPE_CENTRAL2 && d->scheme != CHFPE_COMPACT6) { *why = "unknown scheme"; return CHFPE_ERR_INVALID; }
  if (d->gauge != CHFPE_GAUGE_SQRT_EQ && d->gauge != CHFPE_GAUGE_W) { *why = "unknown gauge"; return CHFPE_ERR_INVALID; }
  if (d->batch < 1 || d->batch > 4096) { *why = "batch must be 1..4096"; return CHFPE_ERR_INVALID; }
  if (d->closure != CHFPE_CLOSURE_TRUNCATE && d->closure != CHFPE_CLOSURE_TERMINATOR) { *why = "unknown closure"; return CHFPE_ERR_INVALID; }
  if (d->closure == CHFPE_CLOSURE_TERMINATOR && d->scheme == CHFPE_COMPACT6) { *why = "the terminator closure needs an explicit scheme"; return CHFPE_ERR_INVALID; }
  if (d->n_terms < 0 || (d->n_terms > 0 && !d->U)) { *why = "bad potential term list"; return CHFPE_ERR_INVALID; }
  for (int t = 0; t < d->n_terms; t++) {
    int deg = 0;
    for (int s = 0; s < 3; s++) {
      if (d->U[t].expo[s] < 0) { *why = "negative exponent"; return CHFPE_ERR_INVALID; }
      if (s < d->n_modes) deg += d->U[t].expo[s];
    }
    if (deg > 4) { *why = "potential degree > 4"; return CHFPE_ERR_INVALID; }
  }
  for (int s = 0; s < d->n_modes; s++) {
    if (d->nq[s] < 5 || d->np[s] < 5) { *why = "need >= 5 grid points per axis"; return CHFPE_ERR_INVALID; }
    if (d->scheme == CHFPE_COMPACT6 && (d->nq[s] > 4096 || d->np[s] > 4096)) { *why = "COMPACT6: at most 4096 points per axis"; return CHFPE_ERR_INVALID; }
    if (!(d->mass[s] > 0) || !(d->gamma[s] > 0) || d->zeta[s] < 0) { *why = "mass, gamma must be > 0 and zeta >= 0"; return CHFPE_ERR_INVALID; }
    if (!(d->qmax[s] > d->qmin[s]) || !(d->pmax[s] > d->pmin[s])) { *why = "empty coordinate range"; return CHFPE_ERR_INVALID; }
  }
  double cells = 1.0;
  for (int s = 0; s < d->n_modes; s++) cells *= (double)d->nq[s] * d->np[s];
  if (cells >= 2147483648.0) { *why = "grid of 2^31 cells or more"; return CHFPE_ERR_INVALID; }
  return CHFPE_OK;
}

struct Plan {
  int M, K, batch, n_arrays, red_blocks;
  long long cells, nqc;
  size_t off_tables, tables_bytes, off_partial, off_results, off_arrays, off_scratch, total;
  static const long long RESULTS = 1 << 16;
};

static Plan make_plan(const chfpe_desc* d) {
  Plan p;
  p.M = d->n_modes; p.batch = d->batch;
  p.K = enumerate_elements(p.M, d->depth, nullptr);
  p.cells = 1; p.nqc = 1;
  long long sum_n = 0;
  for (int s = 0; s < p.M; s++) { p.cells *= (long long)d->nq[s] * d->np[s]; p.nqc *= d->nq[s]; sum_n += d->np[s]; }
  p.n_arrays = 3 * p.batch + (p.batch == 1 ? 1 : 0);
  p.red_blocks = 592;
  size_t o = 0;
  p.off_tables = o;
  size_t tb = 0;
  tb += align256(sizeof(double) * p.nqc) * (p.M + 1);          // dU[s], eU
  tb += align256(sizeof(double) * sum_n);                      // ep
  tb += align256(sizeof(int) * 3 * p.K) * 6;                   // up, dn, nvec (+ their three-mode view for M = 2)
  tb += align256(sizeof(double) * p.K);                        // Gamma
  if (d->scheme == CHFPE_COMPACT6) tb += 2 * p.M * 3 * align256(sizeof(double) * 4096);   // Thomas factors per axis
  tb += align256(sizeof(int) * p.K) * 2;                       // brick-kernel element order and its inverse
  tb += align256(sizeof(int) * 4 * (size_t)p.K * p.nqc);       // brick-order table of the three-mode kernels
  if (p.M == 3) tb += align256(sizeof(int) * 4 * 4 * (size_t)p.K * d->nq[0] * d->nq[1]);   // line table (chfpe_tma.cu), <= 4 parts
  p.tables_bytes = tb; o += tb;
  p.off_partial = o; o += align256(sizeof(double) * p.red_blocks * (size_t)p.batch);
  p.off_results = o; o += align256(sizeof(double) * Plan::RESULTS);
  p.off_arrays = o; o += align256(sizeof(double) * (size_t)p.n_arrays * p.K * p.cells);
  p.off_scratch = o;
  if (d->scheme == CHFPE_COMPACT6) o += align256(sizeof(double) * 3 * (size_t)p.cells);   // G, D, F of chfpe_compact.cu
  p.total = o;
  return p;
}

static int env_int(const char* name, int dflt) {
  const char* v = getenv(name);
  return (v && *v) ? atoi(v) : dflt;
}

// Choose the stage-kernel family (chfpe_brick.cu, chfpe_tma.cu) and the element groups that sweep q_1 in lock-step.
// order_out: elements with the groups contiguous.  The CHFPE_* environment variables read here are debugging and
// measurement tunables, documented in include/chfpe.h ("Tunables"); none of them changes a result.
static BrickPlan make_brick_plan(const chfpe_desc* d, const Plan& pl, const std::vector<int>& up, const std::vector<int>& dn,
                                 std::vector<int>* order_out) {
  BrickPlan bp;
  memset(&bp, 0, sizeof(bp));
  const int M = pl.M, K = pl.K;
  order_out->resize(K);
  for (int k = 0; k < K; k++) (*order_out)[k] = k;
  bp.g = 1; bp.n_groups = K;
  if (M < 2 || d->scheme == CHFPE_COMPACT6 || !env_int("CHFPE_BRICK", 1)) return bp;
  // two modes run as three with a one-point, uncoupled middle mode (same memory layout)
  const int vnq[3] = {d->nq[0], M == 3 ? d->nq[1] : 1, M == 3 ? d->nq[2] : d->nq[1]};
  const int vnp[3] = {d->np[0], M == 3 ? d->np[1] : 1, M == 3 ? d->np[2] : d->np[1]};
  if (vnq[0] > 1023 || vnq[1] > 1023 || vnq[2] > 1023 || (long long)pl.K * pl.nqc > 0x7fffffffLL) return bp;
  bp.P1 = vnp[0]; bp.P2 = vnp[1]; bp.P3 = vnp[2];
  bp.PB2 = bp.P2 * bp.P3;
  // threads per CTA = split * P2*P3/2 (128-bit accesses); aim at ~512 threads (one CTA per SM at 128 registers)
  // with >= 4 planes per thread: at 16^3 the 256-thread / 2-CTA variant times the same but its register allocation
  // sits on the spill edge (a few more live scalars cost 15 %)
  int split_default = 1;
  while (split_default < bp.P1 && bp.P1 % (2 * split_default) == 0 && bp.P1 / (2 * split_default) >= 4 &&
         split_default * bp.PB2 / 2 < 384)
    split_default *= 2;
  if (bp.P1 == 12) split_default = 2;
  // the instantiated two-mode shapes; 48 x 48: 16 segments of 3 planes (384 threads, 2 CTAs per SM) measured 0.82 ms per
  // stage at config 3 against 1.01 ms with 8 segments of 6 planes (192 threads): the kernel is L2-latency bound there
  if (M == 2) split_default = (bp.P1 == 48) ? 16 : 4;
  bp.split = env_int("CHFPE_BRICK_SPLIT", split_default);
  bp.minb = env_int("CHFPE_BRICK_MINB", (M == 2 || bp.PB2 * bp.split / 2 <= 256) ? 2 : 1);
  bp.vn[0] = vnq[0]; bp.vn[1] = vnq[1]; bp.vn[2] = vnq[2];
  // bricks with more than 16 planes are swept in two passes of P1/2 planes: 5 instead of 10 planes of state per
  // thread at 20^3 (no register spills; measured 25.4 -> 21.6 ms per stage at config 5)
  bp.npass = env_int("CHFPE_BRICK_NPASS", (bp.P1 > 16 && bp.P1 % (2 * bp.split) == 0) ? 2 : 1);
  bp.fixed = brick_has_fixed(M, bp.P1, bp.P2, bp.P3, bp.split, bp.minb, bp.npass);
  if (!bp.fixed && bp.npass > 1 && brick_has_fixed(M, bp.P1, bp.P2, bp.P3, bp.split, bp.minb, 1)) {
    bp.npass = 1; bp.fixed = 1;                                      // shapes instantiated single-pass only (48 x 48)
  }
  // bulk-copy fed kernel (chfpe_tma.cu): CENTRAL4, three modes, bricks cut into tma_npart parts along p_1
  bp.tma_npart = env_int("CHFPE_TMA_NPART", bp.P1 >= 12 ? 2 : 1);   // (the halo planes of a part must fit one slot)
  bp.tma_nseg = env_int("CHFPE_TMA_NSEG", bp.P1 == 8 ? 2 : (bp.tma_npart == 1 ? 4 : (bp.P1 == 12 ? 3 : 2)));
  bp.tma_slots = env_int("CHFPE_TMA_SLOTS", 5);                        // (20^3: 32 KB chunks, five fit beside the exchange planes: 216 KB)
  bp.tma_ring = env_int("CHFPE_TMA_RING", 1);
  bp.tma = (M == 3 && d->scheme == CHFPE_CENTRAL4 && vnq[2] <= 64 && env_int("CHFPE_TMA", 1))   // (q_3 lines of <= 64 bricks: TmaCfg::MAXQ3)
               ? tma_has_fixed(M, bp.P1, bp.P2, bp.P3, bp.tma_npart, bp.tma_nseg, bp.tma_slots, bp.tma_ring) : 0;
  if (!bp.fixed && !bp.tma) return bp;
  // L2 reuse window = five q_1 planes x (q_2 chunk + 2+2 halo rows) x g elements of the stage input; budget 64 MiB
  // of the 126 MB L2 (the rest serves the once-touched streams).  Pairs of linked elements (g = 2) save one
  // neighbour-brick read per pair if at least 6 q_2 rows per chunk still fit, else one element at a time.
  // (a sweep of the bulk-copy kernel covers one p_1 part of the bricks: its window is 1/tma_npart of that)
  const double plane_bytes = 8.0 * (double)pl.cells / vnq[0] / (bp.tma ? bp.tma_npart : 1);
  const double row_bytes = plane_bytes / vnq[1];                 // one q_2 row of one q_1 plane
  const double budget = env_int("CHFPE_L2_WINDOW_MB", 64) * 1024.0 * 1024.0;
  auto rows_that_fit = [&](int gg) { return (int)(budget / (5.0 * row_bytes * gg)) - 4; };
  int g = (K >= 2 && rows_that_fit(2) >= 6) ? 2 : 1;
  if (bp.tma && K >= 4 && rows_that_fit(4) >= 6) g = 4;           // squares n, n+e_a, n+e_b, n+e_a+e_b: 4 links inside
  if (vnq[1] == 1) {                                                 // no q_2 rows to chunk: as many whole planes as fit
    g = (int)(budget / (5.0 * plane_bytes));
    if (g < 1) g = 1;
    if (g > K) g = K;
  }
  g = env_int("CHFPE_GROUP", g);
  if (g < 1) g = 1;
  if (g > K) g = K;
  int cs = rows_that_fit(g);
  if (cs >= vnq[1]) cs = vnq[1];
  else {
    if (cs < 4) cs = 4;
    const int nch = (vnq[1] + cs - 1) / cs;                      // equalise the chunks
    cs = (vnq[1] + nch - 1) / nch;
  }
  cs = env_int("CHFPE_Q2CHUNK", cs);
  if (cs < 1) cs = 1;
  if (cs > vnq[1]) cs = vnq[1];
  bp.q2chunk = cs;
  // greedy grouping: grow each group by the unassigned element with most hierarchy links into it
  std::vector<int> assigned(K, 0), order;
  for (int k0 = 0; k0 < K; k0++) {
    if (assigned[k0]) continue;
    std::vector<int> grp(1, k0);
    assigned[k0] = 1;
    while ((int)grp.size() < g) {
      int best = -1, best_links = -1;
      for (int c = 0; c < K; c++) {
        if (assigned[c]) continue;
        int links = 0;
        for (int e : grp)
          for (int s = 0; s < M; s++) links += (up[3 * e + s] == c) + (dn[3 * e + s] == c);
        if (links > best_links) { best_links = links; best = c; }
      }
      if (best < 0) break;
      assigned[best] = 1; grp.push_back(best);
    }
    for (int e : grp) order.push_back(e);
  }
  *order_out = order;
  bp.g = g; bp.n_groups = (K + g - 1) / g;
  bp.blocks_per_full_group = (long long)g * pl.nqc;
  bp.rest = pl.nqc / vnq[0];
  bp.enabled = 1;
  {                                                                  // bricks per CTA: amortises the per-CTA setup
    int bpc = 1;                                                     // (16^6: 4.47 -> 4.17 ms); a divisor of n_q3 so
    for (int c = 2; c <= 16; c++) if (vnq[2] % c == 0) bpc = c;    // that a run never straddles two q_3 lines
    bp.bpc = env_int("CHFPE_BPC", bpc);
  }
  if (bp.bpc < 1) bp.bpc = 1;
  return bp;
}

extern "C" int chfpe_workspace_bytes(const chfpe_desc* desc, size_t* bytes) {
  std::string why;
  int rc = validate(desc, &why);
  if (rc != CHFPE_OK || !bytes) { g_create_err = why.empty() ? "null output" : why; return CHFPE_ERR_INVALID; }
  *bytes = make_plan(desc).total;
  return CHFPE_OK;
}

extern "C" int chfpe_create(const chfpe_desc* desc, void* ws, size_t bytes, void* cuda_stream, chfpe_handle** out) {
  std::string why;
  int rc = validate(desc, &why);
  if (rc != CHFPE_OK) { g_create_err = why; return rc; }
  if (!out) { g_create_err = "null output"; return CHFPE_ERR_INVALID; }
  Plan pl = make_plan(desc);
  if (!ws || bytes < pl.total || ((uintptr_t)ws & 255)) { g_create_err = "workspace too small or misaligned"; return CHFPE_ERR_WORKSPACE; }
  int ndev = 0;
  cudaError_t ce = cudaGetDeviceCount(&ndev);
  if (ce != cudaSuccess || ndev == 0) { g_create_err = std::string("no CUDA device: ") + cudaGetErrorString(ce); return CHFPE_ERR_CUDA; }

  chfpe_handle* h = new chfpe_handle();
  h->desc = *desc;
  h->U.assign(desc->U, desc->U + desc->n_terms);
  h->desc.U = h->U.data();
  h->stream = (cudaStream_t)cuda_stream;
  h->K = pl.K; h->batch = pl.batch; h->n_arrays = pl.n_arrays; h->cells = pl.cells;
  h->state_doubles = (size_t)pl.K * pl.cells;
  h->red_blocks = pl.red_blocks;
  h->initialised = false; h->launches = 0; h->prof = false; h->prof_used = 0; h->norm_ref_valid = false;
  h->coop_mode = env_int("CHFPE_COOP", 1);
  h->coop = h->coop_mode != 0;
  const int M = pl.M;
  enumerate_elements(M, desc->depth, &h->elem);

  DevOp& op = h->op;
  memset(&op, 0, sizeof(op));
  op.M = M; op.nax = 2 * M; op.K = pl.K; op.scheme = desc->scheme; op.gauge = desc->gauge; op.beta = desc->beta;
  op.closure = desc->closure; op.depth = desc->depth;
  op.expect_pbrick = env_int("CHFPE_EXPECT_PBRICK", 1);
  for (int s = 0; s < M; s++) {
    op.n[s] = desc->nq[s]; op.n[M + s] = desc->np[s];
    op.x0[s] = desc->qmin[s]; op.x0[M + s] = desc->pmin[s];
    op.h[s] = (desc->qmax[s] - desc->qmin[s]) / (desc->nq[s] - 1);
    op.h[M + s] = (desc->pmax[s] - desc->pmin[s]) / (desc->np[s] - 1);
    op.inv_mass[s] = 1.0 / desc->mass[s];
    op.cdn[s] = desc->zeta[s] * desc->gamma[s] * desc->mass[s] / desc->beta;
    if (desc->gauge == CHFPE_GAUGE_W) { op.kup[s] = 0.0; op.kdn[s] = desc->beta / desc->mass[s]; }
    else { op.kup[s] = -desc->beta / (2 * desc->mass[s]); op.kdn[s] = desc->beta / (2 * desc->mass[s]); }
    op.VLL[s] = desc->V_LL[s]; op.VSL[s] = desc->V_SL[s];
    op.gam[s] = desc->gamma[s];
  }
  op.cells = pl.cells; op.nqc = pl.nqc; op.pb = pl.cells / pl.nqc;
  op.dV = 1.0;
  long long st = 1;
  for (int a = 2 * M - 1; a >= 0; a--) {
    op.st[a] = st; st *= op.n[a]; op.dV *= op.h[a];
    if (desc->scheme == CHFPE_CENTRAL4) { op.c1[a] = 8.0 / (12.0 * op.h[a]); op.c2[a] = -1.0 / (12.0 * op.h[a]); }
    else { op.c1[a] = 1.0 / (2.0 * op.h[a]); op.c2[a] = 0.0; }
  }

  for (int s = 0; s < M; s++) {
    const double w[4] = {8.0, -8.0, -1.0, 1.0};
    for (int dd = 0; dd < 4; dd++) op.cqw[s][dd] = op.c2[s] * op.inv_mass[s] * w[dd];
  }
  // ---- host tables (setup step a0) ----
  std::vector<double> dU[3], eU(pl.nqc);
  for (int s = 0; s < M; s++) dU[s].resize(pl.nqc);
  const double wfac = (desc->gauge == CHFPE_GAUGE_W) ? 1.0 : 0.5;     // weight exponent: e^{-beta H} or e^{-beta H/2}
  ChfpePoly poly;
  poly.build(h->U.data(), (int)h->U.size(), M);
  for (long long l = 0; l < pl.nqc; l++) {
    int iq[3] = {0, 0, 0}; long long r = l;
    for (int s = M - 1; s >= 0; s--) { iq[s] = (int)(r % op.n[s]); r /= op.n[s]; }
    double q[3] = {0, 0, 0};
    for (int s = 0; s < M; s++) q[s] = op.x0[s] + iq[s] * op.h[s];
    eU[l] = exp(-wfac * desc->beta * poly.value(q));
    for (int s = 0; s < M; s++) dU[s][l] = poly.grad(s, q);
  }
  std::vector<double> ep;
  size_t ep_off[3] = {0, 0, 0};
  for (int s = 0; s < M; s++) {
    ep_off[s] = ep.size();
    for (int i = 0; i < op.n[M + s]; i++) {
      double p = op.x0[M + s] + i * op.h[M + s];
      ep.push_back(exp(-wfac * desc->beta * p * p / (2.0 * desc->mass[s])));
    }
  }
  std::vector<int> up(3 * pl.K, -1), dn(3 * pl.K, -1), nv(3 * pl.K, 0);
  std::vector<double> Gam(pl.K, 0.0);
  auto find = [&](const int n[3]) {
    for (int k = 0; k < pl.K; k++)
      if (h->elem[3 * k] == n[0] && h->elem[3 * k + 1] == n[1] && h->elem[3 * k + 2] == n[2]) return k;
    return -1;
  };
  for (int k = 0; k < pl.K; k++)
    for (int s = 0; s < M; s++) {
      int n[3] = {h->elem[3 * k], h->elem[3 * k + 1], h->elem[3 * k + 2]};
      nv[3 * k + s] = n[s];
      Gam[k] += n[s] * desc->gamma[s];
      n[s] += 1; up[3 * k + s] = find(n);
      n[s] -= 2; if (n[s] >= 0) dn[3 * k + s] = find(n);
    }

  // ---- carve and upload ----
  char* base = (char*)ws;
  char* tp = base + pl.off_tables;
  auto put = [&](const void* src, size_t nbytes) -> void* {
    void* dst = tp;
    cudaMemcpyAsync(dst, src, nbytes, cudaMemcpyHostToDevice, h->stream);
    tp += align256(nbytes);
    return dst;
  };
  for (int s = 0; s < M; s++) op.dU[s] = (const double*)put(dU[s].data(), sizeof(double) * pl.nqc);
  op.eU = (const double*)put(eU.data(), sizeof(double) * pl.nqc);
  const double* epd = (const double*)put(ep.data(), sizeof(double) * ep.size());
  for (int s = 0; s < M; s++) op.ep[s] = epd + ep_off[s];
  op.up = (const int*)put(up.data(), sizeof(int) * up.size());
  op.dn = (const int*)put(dn.data(), sizeof(int) * dn.size());
  op.nvec = (const int*)put(nv.data(), sizeof(int) * nv.size());
  op.Gamma = (const double*)put(Gam.data(), sizeof(double) * Gam.size());
  std::vector<int> order;
  h->bp = make_brick_plan(desc, pl, up, dn, &order);
  h->bp.order = (const int*)put(order.data(), sizeof(int) * order.size());
  std::vector<int> pos(order.size());
  for (size_t i = 0; i < order.size(); i++) pos[order[i]] = (int)i;
  h->bp.pos = (const int*)put(pos.data(), sizeof(int) * pos.size());
  h->bp.l2mode = env_int("CHFPE_L2MODE", h->bp.tma ? 3 : 1);
  if (h->bp.enabled) {                                                 // tabulate the brick order (decode_brick_id)
    const BrickPlan& b = h->bp;
    const int n1 = b.vn[0], n2 = b.vn[1], n3 = b.vn[2], cs = b.q2chunk;
    const int nch = (n2 + cs - 1) / cs;
    std::vector<int> tab;
    tab.reserve((size_t)4 * pl.K * pl.nqc);
    for (int G = 0; G < b.n_groups; G++) {
      const int gs = std::min(b.g, pl.K - G * b.g);
      for (int ch = 0; ch < nch; ch++) {
        const int w = std::min(cs, n2 - ch * cs);
        for (int i1 = 0; i1 < n1; i1++)
          for (int kk = 0; kk < gs; kk++) {
            const int k = order[G * b.g + kk];
            int own = 0;
            for (int s = 0; s < M; s++) {
              const int vs = (M == 2 && s == 1) ? 2 : s;                // mode index in the three-mode view
              if (up[3 * k + s] >= 0 && pos[up[3 * k + s]] / b.g == G) own |= 1 << (2 * vs);
              if (dn[3 * k + s] >= 0 && pos[dn[3 * k + s]] / b.g == G) own |= 1 << (2 * vs + 1);
            }
            for (int r2 = 0; r2 < w; r2++)
              for (int i3 = 0; i3 < n3; i3++) {
                const int i2 = ch * cs + r2;
                tab.push_back(k);
                tab.push_back((i1 * n2 + i2) * n3 + i3);
                tab.push_back(i1 | (i2 << 10) | (i3 << 20));
                tab.push_back(G | (own << 16));
              }
          }
      }
    }
    h->bp.table = (const int4*)put(tab.data(), sizeof(int) * tab.size());
    cudaStreamSynchronize(h->stream);                                  // `tab` goes out of scope
    if (b.tma) {   // sweep order of the bulk-copy kernel: group -> q_2 chunk -> p_1 part -> q_1 plane -> element -> q_2 row
      std::vector<int> lt;
      lt.reserve((size_t)4 * pl.K * n1 * n2 * b.tma_npart);
      for (int G = 0; G < b.n_groups; G++) {
        const int gs = std::min(b.g, pl.K - G * b.g);
        for (int ch = 0; ch < nch; ch++) {
          const int w = std::min(cs, n2 - ch * cs);
          for (int part = 0; part < b.tma_npart; part++)
            for (int i1 = 0; i1 < n1; i1++)
              for (int kk = 0; kk < gs; kk++) {
                const int k = order[G * b.g + kk];
                int own = 0;
                for (int s = 0; s < M; s++) {
                  if (up[3 * k + s] >= 0 && pos[up[3 * k + s]] / b.g == G) own |= 1 << (2 * s);
                  if (dn[3 * k + s] >= 0 && pos[dn[3 * k + s]] / b.g == G) own |= 1 << (2 * s + 1);
                }
                for (int r2 = 0; r2 < w; r2++) {
                  const int offs[4] = {1, -1, 2, -2};
                  int q2out = 0;                                         // q_2 neighbours outside this chunk's rows
                  for (int dd = 0; dd < 4; dd++)
                    if (r2 + offs[dd] < 0 || r2 + offs[dd] >= w) q2out |= 1 << dd;
                  lt.push_back(k);
                  lt.push_back(i1 | ((ch * cs + r2) << 10) | (part << 20));
                  lt.push_back(own);
                  lt.push_back(q2out);
                }
              }
        }
      }
      h->bp.n_lines = (int)(lt.size() / 4);
      h->bp.lines = (const int4*)put(lt.data(), sizeof(int) * lt.size());
      cudaStreamSynchronize(h->stream);
    }
    // operator as the three-mode kernels see it
    h->op3 = op;
    if (M == 2) {
      DevOp& v = h->op3;
      v.M = 3; v.nax = 6;
      const int map[3] = {0, -1, 1};                                   // view mode -> real mode
      for (int vs = 0; vs < 3; vs++) {
        const int r = map[vs];
        v.n[vs] = r < 0 ? 1 : op.n[r];          v.n[3 + vs] = r < 0 ? 1 : op.n[M + r];
        v.x0[vs] = r < 0 ? 0.0 : op.x0[r];      v.x0[3 + vs] = r < 0 ? 0.0 : op.x0[M + r];
        v.h[vs] = r < 0 ? 1.0 : op.h[r];        v.h[3 + vs] = r < 0 ? 1.0 : op.h[M + r];
        v.c1[vs] = r < 0 ? 0.0 : op.c1[r];      v.c1[3 + vs] = r < 0 ? 0.0 : op.c1[M + r];
        v.c2[vs] = r < 0 ? 0.0 : op.c2[r];      v.c2[3 + vs] = r < 0 ? 0.0 : op.c2[M + r];
        v.inv_mass[vs] = r < 0 ? 0.0 : op.inv_mass[r];
        v.kup[vs] = r < 0 ? 0.0 : op.kup[r];    v.kdn[vs] = r < 0 ? 0.0 : op.kdn[r];
        v.cdn[vs] = r < 0 ? 0.0 : op.cdn[r];
        for (int dd = 0; dd < 4; dd++) v.cqw[vs][dd] = r < 0 ? 0.0 : op.cqw[r][dd];
        v.VLL[vs] = r < 0 ? 0.0 : op.VLL[r];    v.VSL[vs] = r < 0 ? 0.0 : op.VSL[r];
        v.dU[vs] = op.dU[r < 0 ? 0 : r];
      }
      long long st = 1;
      for (int a2 = 5; a2 >= 0; a2--) { v.st[a2] = st; st *= v.n[a2]; }
      std::vector<int> up3(3 * pl.K, -1), dn3(3 * pl.K, -1), nv3(3 * pl.K, 0);
      for (int k = 0; k < pl.K; k++)
        for (int vs = 0; vs < 3; vs++)
          if (map[vs] >= 0) {
            up3[3 * k + vs] = up[3 * k + map[vs]]; dn3[3 * k + vs] = dn[3 * k + map[vs]]; nv3[3 * k + vs] = nv[3 * k + map[vs]];
          }
      v.up = (const int*)put(up3.data(), sizeof(int) * up3.size());
      v.dn = (const int*)put(dn3.data(), sizeof(int) * dn3.size());
      v.nvec = (const int*)put(nv3.data(), sizeof(int) * nv3.size());
      cudaStreamSynchronize(h->stream);
    }
  }
  if (h->bp.enabled && h->bp.tma && tma_configure(h->bp) != 0) { cudaGetLastError(); h->bp.tma = 0; }
  if (h->bp.enabled && !h->bp.fixed && !h->bp.tma) h->bp.enabled = 0;
  if (h->bp.enabled && h->bp.fixed && brick_configure(h->bp, M) != 0) { cudaGetLastError(); h->bp.fixed = 0; if (!h->bp.tma) h->bp.enabled = 0; }
  memset(&h->ct, 0, sizeof(h->ct));
  h->scratch = nullptr;
  if (desc->scheme == CHFPE_COMPACT6) {                                // elimination factors of tridiag(1/3, 1, 1/3), n rows
    for (int a = 0; a < 2 * M; a++) {
      const int n = op.n[a];
      std::vector<double> bet(n), cf(n);
      const double al = 1.0 / 3.0;
      bet[0] = 1.0; cf[0] = 0.0;
      for (int i = 1; i < n; i++) { cf[i] = al / bet[i - 1]; bet[i] = 1.0 - al * cf[i]; }
      h->ct.bet[a] = (const double*)put(bet.data(), sizeof(double) * n);
      h->ct.cfac[a] = (const double*)put(cf.data(), sizeof(double) * n);
      std::vector<double> ib(n);
      for (int i = 0; i < n; i++) ib[i] = 1.0 / bet[i];
      h->ct.ibet[a] = (const double*)put(ib.data(), sizeof(double) * n);
      cudaStreamSynchronize(h->stream);
    }
    h->scratch = (double*)(base + pl.off_scratch);
  }
  h->partial = (double*)(base + pl.off_partial);
  h->results = (double*)(base + pl.off_results);
  h->arrays = (double*)(base + pl.off_arrays);
  ce = cudaMemsetAsync(h->arrays, 0, sizeof(double) * (size_t)pl.n_arrays * h->state_doubles, h->stream);
  if (ce == cudaSuccess) ce = cudaStreamSynchronize(h->stream);       // host tables go out of scope below
  if (ce != cudaSuccess) {
    g_create_err = std::string("create: ") + cudaGetErrorString(ce);
    delete h;
    return CHFPE_ERR_CUDA;
  }
  *out = h;
  return CHFPE_OK;
}

extern "C" int chfpe_destroy(chfpe_handle* h) {
  if (h) for (cudaEvent_t e : h->prof_ev) cudaEventDestroy(e);
  delete h;
  return CHFPE_OK;
}

extern "C" const char* chfpe_last_error(const chfpe_handle* h) { return h ? h->err.c_str() : g_create_err.c_str(); }

extern "C" int chfpe_num_elements(const chfpe_handle* h, int32_t* K) {
  if (!h || !K) return CHFPE_ERR_INVALID;
  *K = h->K; return CHFPE_OK;
}

extern "C" int chfpe_element_index(const chfpe_handle* h, int32_t k, int32_t n_out[3]) {
  if (!h || !n_out || k < 0 || k >= h->K) return CHFPE_ERR_INVALID;
  for (int s = 0; s < 3; s++) n_out[s] = h->elem[3 * k + s];
  return CHFPE_OK;
}

extern "C" int chfpe_launch_count(const chfpe_handle* h, int64_t* n) {
  if (!h || !n) return CHFPE_ERR_INVALID;
  *n = h->launches; return CHFPE_OK;
}

extern "C" int chfpe_stage_kernel(const chfpe_handle* h, int32_t* kind) {
  if (!h || !kind) return CHFPE_ERR_INVALID;
  *kind = (h->op.scheme == CHFPE_COMPACT6) ? CHFPE_STAGE_COMPACT
          : (h->bp.enabled && h->bp.tma)   ? CHFPE_STAGE_TMA
          : h->bp.enabled                  ? CHFPE_STAGE_BRICK
                                           : CHFPE_STAGE_GENERIC;
  return CHFPE_OK;
}

static DevObs to_dev(const chfpe_observable* o) {
  DevObs d;
  memset(&d, 0, sizeof(d));
  if (o) memcpy(&d, o, sizeof(d));
  return d;
}

static int check_launch(chfpe_handle* h) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { h->err = std::string("kernel launch: ") + cudaGetErrorString(e); return CHFPE_ERR_CUDA; }
  return CHFPE_OK;
}

static int run_stage(chfpe_handle* h, const double* in, const double* y, double* out, double a, double c, int nb,
                     size_t ss) {
  if (h->op.scheme == CHFPE_COMPACT6)
    return launch_stage_compact(h->op, h->ct, in, y, out, a, c, nb, ss, h->scratch, h->stream);
  if (h->bp.enabled) {                                // (these kernels evaluate plain truncation: the slaved elements follow)
    int n = 0;
    if (h->bp.tma) n = launch_stage_tma(h->op3, h->bp, in, y, out, a, c, nb, ss, h->stream);
    else n = launch_stage_brick(h->op3, h->bp, in, y, out, a, c, nb, ss, h->stream);
    if (h->op.closure == CHFPE_CLOSURE_TERMINATOR) n += launch_terminator_add(h->op, in, out, c, nb, ss, h->stream);
    return n;
  }
  return launch_stage(h->op, in, y, out, a, c, nb, ss, h->stream);
}

// one RK stage launch, bracketed by events when profiling is on
static void stage(chfpe_handle* h, const double* in, const double* y, double* out, double a, double c, int nb,
                  size_t ss) {
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (h->prof) {
    if (h->prof_used + 2 > h->prof_ev.size()) {
      cudaEvent_t a0, a1;
      if (cudaEventCreate(&a0) == cudaSuccess && cudaEventCreate(&a1) == cudaSuccess) { h->prof_ev.push_back(a0); h->prof_ev.push_back(a1); }
    }
    if (h->prof_used + 2 <= h->prof_ev.size()) { e0 = h->prof_ev[h->prof_used]; e1 = h->prof_ev[h->prof_used + 1]; h->prof_used += 2; }
  }
  if (e0) cudaEventRecord(e0, h->stream);
  h->launches += run_stage(h, in, y, out, a, c, nb, ss);
  if (e1) cudaEventRecord(e1, h->stream);
}

// Tiny states (config 1: 295 KB) are stepped by the persistent cooperative kernel, one launch for any number of
// steps and samples.  Measured on B200: 18.9 vs 27.4 us per step + sample at config 1; at config 2 (1.7 MB) the
// grid-wide barriers cost more than the launches they replace (28.9 vs 25.4 us), hence the 1 MB limit.
// CHFPE_COOP=0 forces per-stage launches, CHFPE_COOP=2 lifts the limit to 24 MB (tests).
static bool coop_eligible(const chfpe_handle* h, int nb) {
  const size_t limit = (h->coop_mode == 2) ? ((size_t)24 << 20) : ((size_t)1 << 20);
  return nb == 1 && h->coop && h->op.scheme != CHFPE_COMPACT6 && h->state_doubles * sizeof(double) <= limit;
}

// n RK4 steps (Horner form, R13) on slots [b0, b0+nb)
static int step_slots(chfpe_handle* h, int b0, int nb, int64_t n_steps, double dt) {
  if (nb <= 0 || n_steps <= 0) return CHFPE_OK;
  if (coop_eligible(h, nb)) {
    DevObs none;
    memset(&none, 0, sizeof(none));
    const int n = launch_steps_coop(h->op, none, h->y(b0), h->va(b0), h->vb(b0), dt, 1, n_steps, 0, h->partial,
                                    h->red_blocks, h->results, h->stream);
    if (n > 0) { h->launches += n; return check_launch(h); }
    h->coop = false;                                   // not launchable on this device: fall through for good
  }
  const size_t ss = 3 * h->state_doubles;
  double *y = h->y(b0), *va = h->va(b0), *vb = h->vb(b0);
  for (int64_t i = 0; i < n_steps; i++) {
    stage(h, y, y, va, 1.0, dt / 4.0, nb, ss);
    stage(h, va, y, vb, 1.0, dt / 3.0, nb, ss);
    stage(h, vb, y, va, 1.0, dt / 2.0, nb, ss);
    stage(h, va, y, y, 1.0, dt, nb, ss);
  }
  return check_launch(h);
}

extern "C" int chfpe_profile_enable(chfpe_handle* h, int on) {
  if (!h) return CHFPE_ERR_INVALID;
  h->prof = on != 0;
  return CHFPE_OK;
}

extern "C" int chfpe_profile_read(chfpe_handle* h, double* total_ms, int64_t* n_launches) {
  if (!h || !total_ms || !n_launches) return CHFPE_ERR_INVALID;
  CU(h, cudaStreamSynchronize(h->stream));
  double tot = 0.0;
  for (size_t i = 0; i + 1 < h->prof_used; i += 2) {
    float ms = 0.f;
    CU(h, cudaEventElapsedTime(&ms, h->prof_ev[i], h->prof_ev[i + 1]));
    tot += ms;
  }
  *total_ms = tot; *n_launches = (int64_t)(h->prof_used / 2);
  h->prof_used = 0;
  return CHFPE_OK;
}

static int kick_slots(chfpe_handle* h, int b0, int nb, const chfpe_observable* X) {
  const size_t ss = 3 * h->state_doubles;
  DevObs o = to_dev(X);
  if (h->op.scheme != CHFPE_COMPACT6 && env_int("CHFPE_KICK_BRICK", 1)) {   // in place on the brick layout where it applies
    const int n = launch_kick_brick(h->op, o, h->y(b0), nb, ss, h->stream);
    if (n > 0) { h->launches += n; return check_launch(h); }
  }
  if (h->op.scheme == CHFPE_COMPACT6)
    h->launches += launch_kick_compact(h->op, h->ct, o, h->y(b0), h->va(b0), nb, ss, h->scratch, h->stream);
  else
    h->launches += launch_kick(h->op, o, h->y(b0), h->va(b0), nb, ss, h->stream);
  for (int b = b0; b < b0 + nb; b++)
    CU(h, cudaMemcpyAsync(h->y(b), h->va(b), sizeof(double) * h->state_doubles, cudaMemcpyDeviceToDevice, h->stream));
  return check_launch(h);
}

// <O> on element k of slots [b0, b0+nb) -> results[res_off + i*res_stride]
static int expect_slots(chfpe_handle* h, int b0, int nb, int k, const chfpe_observable* O, long long res_off,
                        long long res_stride) {
  DevObs o = to_dev(O);
  h->launches += launch_reduce(h->op, o, RED_EXPECT, h->y(b0), k, h->cells, nb, 3 * h->state_doubles, h->op.dV,
                               h->partial, h->red_blocks, h->results + res_off, res_stride, h->stream);
  return check_launch(h);
}

static int fetch_results(chfpe_handle* h, long long n, double* host) {
  CU(h, cudaMemcpyAsync(host, h->results, sizeof(double) * n, cudaMemcpyDeviceToHost, h->stream));
  CU(h, cudaStreamSynchronize(h->stream));
  for (long long i = 0; i < n; i++)
    if (!std::isfinite(host[i])) FAIL(h, CHFPE_ERR_DIVERGED, "non-finite expectation value");
  return CHFPE_OK;
}

extern "C" int chfpe_equilibrate(chfpe_handle* h, int64_t n_steps, double dt, double* residual_out) {
  if (!h || n_steps < 0) return CHFPE_ERR_INVALID;
  h->norm_ref_valid = false;
  DevObs none = to_dev(nullptr);
  h->launches += launch_init_eq(h->op, h->y(0), h->stream);
  const int mode = (h->op.gauge == CHFPE_GAUGE_SQRT_EQ) ? RED_SUMSQ : RED_SUM;   // Z_f = dV sum phi^2, Z_W = dV sum e^{-beta H}
  h->launches += launch_reduce(h->op, none, mode, h->y(0), 0, h->cells, 1, 0, h->op.dV, h->partial, h->red_blocks,
                               h->results, 1, h->stream);
  h->launches += launch_scale(h->y(0), h->cells, h->results, 1.0, h->stream);
  for (int b = 1; b < h->batch; b++)
    CU(h, cudaMemcpyAsync(h->y(b), h->y(0), sizeof(double) * h->state_doubles, cudaMemcpyDeviceToDevice, h->stream));
  int rc = check_launch(h);
  if (rc) return rc;
  h->initialised = true;
  rc = step_slots(h, 0, h->batch, n_steps, dt);
  if (rc) return rc;
  if (residual_out) {
    h->launches += run_stage(h, h->y(0), h->y(0), h->va(0), 0.0, 1.0, 1, 0);
    h->launches += launch_reduce(h->op, none, RED_SUMSQ, h->va(0), 0, (long long)h->state_doubles, 1, 0, 1.0,
                                 h->partial, h->red_blocks, h->results, 1, h->stream);
    h->launches += launch_reduce(h->op, none, RED_SUMSQ, h->y(0), 0, (long long)h->state_doubles, 1, 0, 1.0,
                                 h->partial, h->red_blocks, h->results + 1, 1, h->stream);
    rc = check_launch(h);
    if (rc) return rc;
    double r[2];
    rc = fetch_results(h, 2, r);
    if (rc) return rc;
    *residual_out = sqrt(r[0] / r[1]);
  }
  return CHFPE_OK;
}

// sum of squares of every slot's state -> host (synchronises the stream); non-finite values give CHFPE_ERR_DIVERGED
static int slot_norms(chfpe_handle* h, std::vector<double>* out) {
  DevObs none = to_dev(nullptr);
  out->resize(h->batch);
  h->launches += launch_reduce(h->op, none, RED_SUMSQ, h->y(0), 0, (long long)h->state_doubles, h->batch,
                               3 * h->state_doubles, 1.0, h->partial, h->red_blocks, h->results, 1, h->stream);
  int rc = check_launch(h);
  if (rc) return rc;
  return fetch_results(h, h->batch, out->data());
}

// Norm guard (SURVEY 8(b) errors): the literal W gauge of Eq. (8) is semi-discretely unstable on a (q,p) grid (R7;
// 1e30 by t = 3 on a config-2-like grid), so a propagation reports divergence from the call that diverged: the sum of
// squares of a slot must stay finite and below NORM_GROWTH times its value at the last equilibrate / import / kick /
// response call.  One deterministic reduction and one 8-byte read per call (0.5 ms at config 4).
static const double NORM_GROWTH = 1e8;

extern "C" int chfpe_step(chfpe_handle* h, int64_t n_steps, double dt) {
  if (!h || n_steps < 0) return CHFPE_ERR_INVALID;
  if (n_steps == 0) return CHFPE_OK;
  int rc;
  if (!h->norm_ref_valid) {
    rc = slot_norms(h, &h->norm_ref);
    if (rc) return rc;
    h->norm_ref_valid = true;
  }
  rc = step_slots(h, 0, h->batch, n_steps, dt);
  if (rc) return rc;
  std::vector<double> now;
  rc = slot_norms(h, &now);
  if (rc) return rc;
  for (int b = 0; b < h->batch; b++)
    if (h->norm_ref[b] > 0.0 && now[b] > NORM_GROWTH * h->norm_ref[b]) FAIL(h, CHFPE_ERR_DIVERGED, "norm growth guard: the propagation diverges");
  return CHFPE_OK;
}

extern "C" int chfpe_rk4_stage(chfpe_handle* h, int32_t stg, double dt) {
  if (!h || stg < 0 || stg > 3) return CHFPE_ERR_INVALID;
  const size_t ss = 3 * h->state_doubles;
  double *y = h->y(0), *va = h->va(0), *vb = h->vb(0);
  if (stg == 0) stage(h, y, y, va, 1.0, dt / 4.0, h->batch, ss);
  else if (stg == 1) stage(h, va, y, vb, 1.0, dt / 3.0, h->batch, ss);
  else if (stg == 2) stage(h, vb, y, va, 1.0, dt / 2.0, h->batch, ss);
  else stage(h, va, y, y, 1.0, dt, h->batch, ss);
  return check_launch(h);
}

extern "C" int chfpe_stage_input(chfpe_handle* h, int32_t replica, int32_t stg, double** dev, int64_t* plane_doubles) {
  if (!h || !dev || !plane_doubles || replica < 0 || replica >= h->batch || stg < 0 || stg > 3) return CHFPE_ERR_INVALID;
  *dev = (stg == 0) ? h->y(replica) : (stg == 2 ? h->vb(replica) : h->va(replica));
  *plane_doubles = (int64_t)(h->cells / h->desc.nq[0]);
  return CHFPE_OK;
}

extern "C" int chfpe_kick(chfpe_handle* h, const chfpe_observable* X) {
  if (!h || !X) return CHFPE_ERR_INVALID;
  h->norm_ref_valid = false;
  return kick_slots(h, 0, h->batch, X);
}

extern "C" int chfpe_expect(chfpe_handle* h, const chfpe_observable* O, double* out) {
  if (!h || !O || !out) return CHFPE_ERR_INVALID;
  int rc = expect_slots(h, 0, h->batch, 0, O, 0, 1);
  if (rc) return rc;
  return fetch_results(h, h->batch, out);
}

extern "C" int chfpe_expect_element(chfpe_handle* h, int32_t replica, int32_t k, const chfpe_observable* O, double* out) {
  if (!h || !O || !out || replica < 0 || replica >= h->batch || k < 0 || k >= h->K) return CHFPE_ERR_INVALID;
  int rc = expect_slots(h, replica, 1, k, O, 0, 1);
  if (rc) return rc;
  return fetch_results(h, 1, out);
}

extern "C" int chfpe_response_1d(chfpe_handle* h, const chfpe_observable* A, const chfpe_observable* C,
                                 int64_t n_samples, int64_t stride, double dt, double* R) {
  if (!h || !C || !R || n_samples < 0 || stride < 0) return CHFPE_ERR_INVALID;
  if (!h->initialised) FAIL(h, CHFPE_ERR_STATE, "response_1d before equilibrate/import");
  h->norm_ref_valid = false;
  int rc = A ? kick_slots(h, 0, 1, A) : CHFPE_OK;
  if (rc) return rc;
  int64_t done = 0;
  if (coop_eligible(h, 1) && n_samples > 0) {        // sample 0 now, then `stride` steps + one sample per round
    rc = expect_slots(h, 0, 1, 0, C, 0, 1);
    if (rc) return rc;
    rc = fetch_results(h, 1, R);
    if (rc) return rc;
    done = 1;
    DevObs o = to_dev(C);
    while (done < n_samples && h->coop) {
      int64_t chunk = n_samples - done;
      if (chunk > Plan::RESULTS) chunk = Plan::RESULTS;
      const int n = launch_steps_coop(h->op, o, h->y(0), h->va(0), h->vb(0), dt, chunk, stride, 1, h->partial,
                                      h->red_blocks, h->results, h->stream);
      if (n == 0) { h->coop = false; break; }
      h->launches += n;
      rc = check_launch(h);
      if (rc) return rc;
      rc = fetch_results(h, chunk, R + done);
      if (rc) return rc;
      done += chunk;
    }
    if (done >= n_samples) return CHFPE_OK;
    // cooperative launch unavailable: the trajectory stands at sample done-1; continue with per-stage launches
    rc = step_slots(h, 0, 1, stride, dt);
    if (rc) return rc;
  }
  while (done < n_samples) {                         // results buffer holds Plan::RESULTS samples per round trip
    int64_t chunk = n_samples - done;
    if (chunk > Plan::RESULTS) chunk = Plan::RESULTS;
    for (int64_t i = 0; i < chunk; i++) {
      rc = expect_slots(h, 0, 1, 0, C, i, 1);
      if (rc) return rc;
      if (done + i + 1 < n_samples) { rc = step_slots(h, 0, 1, stride, dt); if (rc) return rc; }
    }
    rc = fetch_results(h, chunk, R + done);
    if (rc) return rc;
    done += chunk;
  }
  return CHFPE_OK;
}

extern "C" int chfpe_response_2d(chfpe_handle* h, const chfpe_observable* A, const chfpe_observable* B,
                                 const chfpe_observable* C, const int64_t* t1, int32_t n1, const int64_t* t2,
                                 int32_t n2, double dt, double* R) {
  if (!h || !A || !B || !C || !t1 || !t2 || !R || n1 < 1 || n2 < 1) return CHFPE_ERR_INVALID;
  if (!h->initialised) FAIL(h, CHFPE_ERR_STATE, "response_2d before equilibrate/import");
  h->norm_ref_valid = false;
  for (int i = 0; i < n1; i++) if (t1[i] < 0 || (i && t1[i] < t1[i - 1])) FAIL(h, CHFPE_ERR_INVALID, "t1_steps must be ascending and >= 0");
  for (int i = 0; i < n2; i++) if (t2[i] < 0 || (i && t2[i] < t2[i - 1])) FAIL(h, CHFPE_ERR_INVALID, "t2_steps must be ascending and >= 0");
  const size_t sbytes = sizeof(double) * h->state_doubles;
  int rc = kick_slots(h, 0, 1, A);                   // T <- A^x X, slot 0 carries the t1 trajectory
  if (rc) return rc;
  int64_t now1 = 0;
  const int per_round = (h->batch >= 2) ? h->batch - 1 : 1;
  const long long rows_per_fetch = Plan::RESULTS / n2;
  if (rows_per_fetch < 1) FAIL(h, CHFPE_ERR_INVALID, "n2 too large for the results buffer");
  int k = 0, row0 = 0;                               // rows [row0, k) are in the device results buffer
  while (k < n1) {
    int nb = n1 - k; if (nb > per_round) nb = per_round;
    if (nb > rows_per_fetch) nb = (int)rows_per_fetch;   // a round never holds more rows than the results buffer
    if (k + nb - row0 > rows_per_fetch) {            // flush before the buffer overflows
      rc = fetch_results(h, (long long)(k - row0) * n2, R + (size_t)row0 * n2); if (rc) return rc;
      row0 = k;
    }
    int first;                                       // first slot of the replica group
    if (h->batch >= 2) {
      first = 1;
      for (int b = 0; b < nb; b++) {
        rc = step_slots(h, 0, 1, t1[k + b] - now1, dt); if (rc) return rc;
        now1 = t1[k + b];
        CU(h, cudaMemcpyAsync(h->y(1 + b), h->y(0), sbytes, cudaMemcpyDeviceToDevice, h->stream));
      }
    } else {
      first = 0;
      rc = step_slots(h, 0, 1, t1[k] - now1, dt); if (rc) return rc;
      now1 = t1[k];
      CU(h, cudaMemcpyAsync(h->spare(), h->y(0), sbytes, cudaMemcpyDeviceToDevice, h->stream));
    }
    rc = kick_slots(h, first, nb, B); if (rc) return rc;
    int64_t now2 = 0;
    for (int j = 0; j < n2; j++) {
      rc = step_slots(h, first, nb, t2[j] - now2, dt); if (rc) return rc;
      now2 = t2[j];
      rc = expect_slots(h, first, nb, 0, C, (long long)(k - row0) * n2 + j, n2); if (rc) return rc;
    }
    if (h->batch < 2) CU(h, cudaMemcpyAsync(h->y(0), h->spare(), sbytes, cudaMemcpyDeviceToDevice, h->stream));
    k += nb;
  }
  return fetch_results(h, (long long)(k - row0) * n2, R + (size_t)row0 * n2);
}

extern "C" int chfpe_response_3d(chfpe_handle* h, const chfpe_observable* A, const chfpe_observable* B,
                                 const chfpe_observable* C, const chfpe_observable* D, const int64_t* t1, int32_t n1,
                                 const int64_t* t2, int32_t n2, const int64_t* t3, int32_t n3, double dt, double* R) {
  if (!h || !A || !B || !C || !D || !t1 || !t2 || !t3 || !R || n1 < 1 || n2 < 1 || n3 < 1) return CHFPE_ERR_INVALID;
  if (!h->initialised) FAIL(h, CHFPE_ERR_STATE, "response_3d before equilibrate/import");
  h->norm_ref_valid = false;
  // slot 0 carries the t1 trajectory.  A group of nb t1 samples owns slots [1, 1+nb) for its t2 trajectories and,
  // unless the t2 sample is the last one (then C is applied in place), slots [1+nb, 1+2nb) for the t3 replicas.
  const int nb_max = (n2 == 1) ? h->batch - 1 : (h->batch - 1) / 2;
  if (nb_max < 1) FAIL(h, CHFPE_ERR_INVALID, "response_3d needs batch >= 3 (batch >= 2 if n2 == 1)");
  for (int i = 0; i < n1; i++) if (t1[i] < 0 || (i && t1[i] < t1[i - 1])) FAIL(h, CHFPE_ERR_INVALID, "t1_steps must be ascending and >= 0");
  for (int i = 0; i < n2; i++) if (t2[i] < 0 || (i && t2[i] < t2[i - 1])) FAIL(h, CHFPE_ERR_INVALID, "t2_steps must be ascending and >= 0");
  for (int i = 0; i < n3; i++) if (t3[i] < 0 || (i && t3[i] < t3[i - 1])) FAIL(h, CHFPE_ERR_INVALID, "t3_steps must be ascending and >= 0");
  if ((long long)nb_max * n3 > Plan::RESULTS) FAIL(h, CHFPE_ERR_INVALID, "replicas * n3 too large for the results buffer");
  const size_t sbytes = sizeof(double) * h->state_doubles;
  std::vector<double> tmp((size_t)nb_max * n3);
  int rc = kick_slots(h, 0, 1, A);                   // slot 0: T1 = G(t1) A^x X
  if (rc) return rc;
  int64_t now1 = 0;
  for (int k = 0; k < n1;) {
    int nb = n1 - k; if (nb > nb_max) nb = nb_max;
    for (int b = 0; b < nb; b++) {
      rc = step_slots(h, 0, 1, t1[k + b] - now1, dt); if (rc) return rc;
      now1 = t1[k + b];
      CU(h, cudaMemcpyAsync(h->y(1 + b), h->y(0), sbytes, cudaMemcpyDeviceToDevice, h->stream));
    }
    rc = kick_slots(h, 1, nb, B); if (rc) return rc;  // slots 1..nb: T2 = G(t2) B^x T1(t1_k)
    int64_t now2 = 0;
    for (int j = 0; j < n2; j++) {
      rc = step_slots(h, 1, nb, t2[j] - now2, dt); if (rc) return rc;
      now2 = t2[j];
      int rep = 1;                                   // last t2 sample: the t2 trajectories are not needed again
      if (j + 1 < n2) {
        rep = 1 + nb;
        for (int b = 0; b < nb; b++)
          CU(h, cudaMemcpyAsync(h->y(rep + b), h->y(1 + b), sbytes, cudaMemcpyDeviceToDevice, h->stream));
      }
      rc = kick_slots(h, rep, nb, C); if (rc) return rc;
      int64_t now3 = 0;
      for (int l = 0; l < n3; l++) {
        rc = step_slots(h, rep, nb, t3[l] - now3, dt); if (rc) return rc;
        now3 = t3[l];
        rc = expect_slots(h, rep, nb, 0, D, l, n3); if (rc) return rc;
      }
      rc = fetch_results(h, (long long)nb * n3, tmp.data()); if (rc) return rc;
      for (int b = 0; b < nb; b++)
        for (int l = 0; l < n3; l++) R[((size_t)(k + b) * n2 + j) * n3 + l] = tmp[(size_t)b * n3 + l];
    }
    k += nb;
  }
  return CHFPE_OK;
}

extern "C" int chfpe_export_state(chfpe_handle* h, int32_t replica, double* dst, int dst_is_device) {
  if (!h || !dst || replica < 0 || replica >= h->batch) return CHFPE_ERR_INVALID;
  if (dst_is_device) {
    h->launches += launch_permute(h->op, h->y(replica), dst, 0, h->stream);
    return check_launch(h);
  }
  h->launches += launch_permute(h->op, h->y(replica), h->va(replica), 0, h->stream);
  int rc = check_launch(h); if (rc) return rc;
  CU(h, cudaMemcpyAsync(dst, h->va(replica), sizeof(double) * h->state_doubles, cudaMemcpyDeviceToHost, h->stream));
  CU(h, cudaStreamSynchronize(h->stream));
  return CHFPE_OK;
}

extern "C" int chfpe_import_state(chfpe_handle* h, int32_t replica, const double* src, int src_is_device) {
  if (!h || !src || replica < 0 || replica >= h->batch) return CHFPE_ERR_INVALID;
  h->norm_ref_valid = false;
  if (src_is_device) {
    h->launches += launch_permute(h->op, src, h->y(replica), 1, h->stream);
  } else {
    CU(h, cudaMemcpyAsync(h->va(replica), src, sizeof(double) * h->state_doubles, cudaMemcpyHostToDevice, h->stream));
    h->launches += launch_permute(h->op, h->va(replica), h->y(replica), 1, h->stream);
    CU(h, cudaStreamSynchronize(h->stream));          // the caller may free src on return
  }
  h->initialised = true;
  return check_launch(h);
}

extern "C" int chfpe_export_rhs(chfpe_handle* h, int32_t replica, double* dst, int dst_is_device) {
  if (!h || !dst || replica < 0 || replica >= h->batch) return CHFPE_ERR_INVALID;
  h->launches += run_stage(h, h->y(replica), h->y(replica), h->va(replica), 0.0, 1.0, 1, 0);
  if (dst_is_device) {
    h->launches += launch_permute(h->op, h->va(replica), dst, 0, h->stream);
    return check_launch(h);
  }
  h->launches += launch_permute(h->op, h->va(replica), h->vb(replica), 0, h->stream);
  int rc = check_launch(h); if (rc) return rc;
  CU(h, cudaMemcpyAsync(dst, h->vb(replica), sizeof(double) * h->state_doubles, cudaMemcpyDeviceToHost, h->stream));
  CU(h, cudaStreamSynchronize(h->stream));
  return CHFPE_OK;
}
