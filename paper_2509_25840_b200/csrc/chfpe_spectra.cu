// Spectra (row f3 of DESIGN.md): the half-line Fourier integrals of Eq. (19)-(21) PAPER.md:138-146 over sampled
// response functions, as trapezoid sums on the uniform delay grid at caller-given frequencies (reading R22: the
// paper states no discretisation, window or padding).  The grids are small (<= 64 x 256 delays), so this is a direct
// O(n_omega n_t) transform: one warp per output entry, lanes stride over the delays, fixed-order shuffle reduction
// (deterministic).  The 2D transform is done as two passes (inner delay first) through a complex scratch array.
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/chfpe.h"

namespace {

__device__ __forceinline__ double trap_w(int i, int n) { return (n > 1 && (i == 0 || i == n - 1)) ? 0.5 : 1.0; }

__device__ __forceinline__ double2 warp_sum(double2 v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    v.x += __shfl_down_sync(0xffffffffu, v.x, o);
    v.y += __shfl_down_sync(0xffffffffu, v.y, o);
  }
  return v;
}

// T[k][b] = sum_j w_j e^{i sign om_b t_j} R[k][j]      (rows k = 0..n1-1; one warp per (k, b))
__global__ void __launch_bounds__(128) k_spec_inner(const double* __restrict__ R, int n1, int n2, double dt,
                                                    const double* __restrict__ om, int nw, double sign,
                                                    double2* __restrict__ T) {
  const long long w = ((long long)blockIdx.x * 128 + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (w >= (long long)n1 * nw) return;
  const int k = (int)(w / nw), b = (int)(w - (long long)k * nw);
  const double o = sign * om[b];
  double2 acc = make_double2(0.0, 0.0);
  for (int j = lane; j < n2; j += 32) {
    double s, c;
    sincos(o * (j * dt), &s, &c);
    const double r = trap_w(j, n2) * R[(size_t)k * n2 + j];
    acc.x = fma(r, c, acc.x);
    acc.y = fma(r, s, acc.y);
  }
  acc = warp_sum(acc);
  if (lane == 0) T[w] = acc;
}

// I[a][b] = scale * Im sum_k w_k e^{i sign om_a t_k} T[k][b]        (one warp per (a, b))
__global__ void __launch_bounds__(128) k_spec_outer(const double2* __restrict__ T, int n1, int nw2, double dt,
                                                    const double* __restrict__ om, int nw1, double sign, double scale,
                                                    double* __restrict__ I) {
  const long long w = ((long long)blockIdx.x * 128 + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (w >= (long long)nw1 * nw2) return;
  const int a = (int)(w / nw2), b = (int)(w - (long long)a * nw2);
  const double o = sign * om[a];
  double2 acc = make_double2(0.0, 0.0);
  for (int k = lane; k < n1; k += 32) {
    double s, c;
    sincos(o * (k * dt), &s, &c);
    const double wk = trap_w(k, n1);
    const double2 t = T[(size_t)k * nw2 + b];
    acc.y += wk * fma(c, t.y, s * t.x);                             // Im[(c + i s)(t.x + i t.y)]
  }
  acc = warp_sum(acc);
  if (lane == 0) I[w] = scale * acc.y;
}

// I[a] = om_a * dt * Im sum_k w_k e^{+i om_a t_k} R[k]               (Eq. 19; one warp per frequency)
__global__ void __launch_bounds__(128) k_spec_1d(const double* __restrict__ R, long long n, double dt,
                                                 const double* __restrict__ om, int nw, double* __restrict__ I) {
  const long long w = ((long long)blockIdx.x * 128 + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (w >= nw) return;
  const double o = om[w];
  double2 acc = make_double2(0.0, 0.0);
  for (long long k = lane; k < n; k += 32) {
    double s, c;
    sincos(o * ((double)k * dt), &s, &c);
    const double wk = (n > 1 && (k == 0 || k == n - 1)) ? 0.5 : 1.0;
    acc.y = fma(wk * R[k], s, acc.y);
  }
  acc = warp_sum(acc);
  if (lane == 0) I[w] = o * dt * acc.y;
}

int finish() { return cudaGetLastError() == cudaSuccess ? CHFPE_OK : CHFPE_ERR_CUDA; }

}  // namespace

extern "C" int chfpe_spectrum_1d(void* cuda_stream, const double* R, int64_t n, double dt, const double* omega,
                                 int32_t n_omega, double* I) {
  if (!R || !omega || !I || n < 1 || n_omega < 1 || !(dt > 0.0)) return CHFPE_ERR_INVALID;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  k_spec_1d<<<(unsigned)(((long long)n_omega * 32 + 127) / 128), 128, 0, s>>>(R, n, dt, omega, n_omega, I);
  return finish();
}

extern "C" int chfpe_spectrum_2d(void* cuda_stream, const double* R, int32_t n1, int32_t n2, double dt1, double dt2,
                                 const double* omega1, int32_t nw1, const double* omega2, int32_t nw2, int32_t sign1,
                                 int32_t sign2, double* scratch, double* I) {
  if (!R || !omega1 || !omega2 || !scratch || !I || n1 < 1 || n2 < 1 || nw1 < 1 || nw2 < 1 || !(dt1 > 0.0) ||
      !(dt2 > 0.0) || (sign1 != 1 && sign1 != -1) || (sign2 != 1 && sign2 != -1) || ((uintptr_t)scratch & 15))
    return CHFPE_ERR_INVALID;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  double2* T = reinterpret_cast<double2*>(scratch);
  k_spec_inner<<<(unsigned)(((long long)n1 * nw2 * 32 + 127) / 128), 128, 0, s>>>(R, n1, n2, dt2, omega2, nw2,
                                                                                   (double)sign2, T);
  k_spec_outer<<<(unsigned)(((long long)nw1 * nw2 * 32 + 127) / 128), 128, 0, s>>>(T, n1, nw2, dt1, omega1, nw1,
                                                                                    (double)sign1, dt1 * dt2, I);
  return finish();
}

// ------------------------------------------------------------------------------------------------
// chfpe_spectrum_2d_static: the same two-pass transform for callers that cannot provide (or allocate) the complex
// scratch array -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The scratch
// T[n1][n_omega2] lives in a file-scope device array of CHFPE_SPECTRUM_STATIC_MAX complex entries (1 MiB; every GPU
// that loads the library holds it until exit).  In host code `g_spec_scratch` is only a stand-in for the symbol, not a
// device address: its address on the current device is taken once per device with cudaGetSymbolAddress and that
// pointer is what the kernels get.  Nothing here calls cudaMalloc / cudaFree or an allocating library routine.
// All calls share the array and it keeps the last call's contents; nothing has to start at zero (the inner pass
// writes every entry the outer pass reads), but two calls that overlap on the GPU (different streams) race on it.
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) double2 g_spec_scratch[CHFPE_SPECTRUM_STATIC_MAX];

namespace {
const int MAX_DEVICES = 64;
double2* g_spec_scratch_addr[MAX_DEVICES];      // per device: address of g_spec_scratch, nullptr until first use
}  // namespace

extern "C" int chfpe_spectrum_2d_static(void* cuda_stream, const double* R, int32_t n1, int32_t n2, double dt1,
                                        double dt2, const double* omega1, int32_t nw1, const double* omega2, int32_t nw2,
                                        int32_t sign1, int32_t sign2, double* I) {
  if (!R || !omega1 || !omega2 || !I || n1 < 1 || n2 < 1 || nw1 < 1 || nw2 < 1 || !(dt1 > 0.0) || !(dt2 > 0.0) ||
      (sign1 != 1 && sign1 != -1) || (sign2 != 1 && sign2 != -1))
    return CHFPE_ERR_INVALID;
  if ((long long)n1 * nw2 > (long long)CHFPE_SPECTRUM_STATIC_MAX) return CHFPE_ERR_WORKSPACE;   // scratch too small
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) return CHFPE_ERR_CUDA;
  if (!g_spec_scratch_addr[dev]) {                 // set-up, once per device, with that device current
    double2* p = nullptr;
    if (cudaGetSymbolAddress((void**)&p, g_spec_scratch) != cudaSuccess || !p) { cudaGetLastError(); return CHFPE_ERR_CUDA; }
    g_spec_scratch_addr[dev] = p;
  }
  double2* T = g_spec_scratch_addr[dev];
  cudaStream_t s = (cudaStream_t)cuda_stream;
  k_spec_inner<<<(unsigned)(((long long)n1 * nw2 * 32 + 127) / 128), 128, 0, s>>>(R, n1, n2, dt2, omega2, nw2,
                                                                                   (double)sign2, T);
  k_spec_outer<<<(unsigned)(((long long)nw1 * nw2 * 32 + 127) / 128), 128, 0, s>>>(T, n1, nw2, dt1, omega1, nw1,
                                                                                    (double)sign1, dt1 * dt2, I);
  return finish();
}
