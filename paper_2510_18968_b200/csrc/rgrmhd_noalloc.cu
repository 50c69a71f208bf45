// rgrmhd_noalloc.cu -- rgrmhd_max_speed_static: the CFL reduction a7 (Eq. 30; with state-dependent
// wave speeds PAPER.md:424, 437, reading R16) for callers that may not allocate: code under CUDA graph capture, tight
// serving loops, harnesses that forbid cudaMalloc.  Stateless: no handle (rgrmhd_create allocates), the caller passes
// DEVICE pointers to the metric and primitive fields and to the result; the scratch memory of the reduction lives in a
// file-scope __device__ array of fixed size, so the entry point calls no cudaMalloc / cudaFree and no allocating
// library routine.  Same per-cell arithmetic as k_max_speed (cell_cfl_speed, rgrmhd_common.cuh); the maximum is exact
// in any order, so the result equals rgrmhd_max_speed's.
//
// Scratch: word 0 = arrival counter of the running launch, words 32.. = one partial maximum per CTA.  A CTA covers a
// fixed chunk of 2048 cells, so the array's 8192 partials bound the problem: n[0]*n[1]*n[2] <= 16,777,216 (256^3);
// larger sizes are rejected with RGRMHD_E_TOO_LARGE.  65,792 bytes per GPU that loads the library, held until exit.
// The array is SHARED by every call and keeps the last call's contents: the counter is cleared on the stream before
// every launch (and by the last CTA), the partials are overwritten before they are read.  Two calls that overlap on
// the GPU (different streams, different host threads) race on it; calls on one stream are ordered and safe.
#include <cstring>
#include <mutex>

#include "../../include/rgrmhd.h"
#include "rgrmhd_common.cuh"

namespace rg {
namespace {

constexpr int ST_THREADS = 256;
constexpr int ST_PER_THREAD = 8;
constexpr int ST_CHUNK = ST_THREADS * ST_PER_THREAD;          // cells per CTA
constexpr int ST_MAX_CTAS = 8192;
constexpr int ST_HDR = 32;                                     // header words (256 bytes); word 0 = arrival counter
constexpr long long ST_MAX_CELLS = (long long)ST_CHUNK * ST_MAX_CTAS;
static_assert(ST_MAX_CELLS == RGRMHD_STATIC_MAX_CELLS, "the header states the limit");

// In HOST code this name is a host-side stand-in, not a device address: the launcher below asks the runtime for the
// device address once per device (cudaGetSymbolAddress) and hands that to the kernel.
static __device__ __align__(256) unsigned long long g_static_scratch[ST_HDR + ST_MAX_CTAS];

__global__ void __launch_bounds__(ST_THREADS)
k_max_speed_static(const __grid_constant__ GridView G, unsigned long long* __restrict__ scratch, bool mhd_mode,
                   double* __restrict__ out) {
  const int nx = G.n[0], ny = G.n[1];
  const long long nint = (long long)nx * ny * G.n[2];
  double mx = 0.0;
  const long long t0 = (long long)blockIdx.x * ST_CHUNK + threadIdx.x;
#pragma unroll 1
  for (int q = 0; q < ST_PER_THREAD; ++q) {
    const long long t = t0 + (long long)q * ST_THREADS;
    if (t >= nint) break;
    const int i = (int)(t % nx);
    const long long r = t / nx;
    const int j = (int)(r % ny), k = (int)(r / ny);
    Met m;
    const long long c = cell_index(G, i, j, k);
    load_met_cell(G, c, m);
    const bool mhd = mhd_mode && G.P[RHO][c] > G.wave_rho_switch;   // the cell's own ideal-GRMHD speeds (reading R16)
    double P[NPRIM];
#pragma unroll
    for (int v = 0; v < NPRIM; ++v) P[v] = (mhd && (v <= VZ || (v >= BX && v <= BZ))) ? G.P[v][c] : 0.0;
    mx = fmax(mx, cell_cfl_speed(m, G.Gamma, P, mhd, G.inv_dx[0], G.inv_dx[1], G.inv_dx[2], G.n[0] > 1, G.n[1] > 1, G.n[2] > 1));
  }
  __shared__ double smx[ST_THREADS / 32];
  __shared__ bool last;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if (lane == 0) smx[warp] = mx;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < ST_THREADS / 32; ++w) mx = fmax(mx, smx[w]);
    scratch[ST_HDR + blockIdx.x] = (unsigned long long)__double_as_longlong(mx);
    __threadfence();                                              // the partial is visible before the arrival counts
    last = atomicAdd(&scratch[0], 1ull) == (unsigned long long)(gridDim.x - 1);
  }
  __syncthreads();
  if (!last) return;
  // the last CTA to arrive reduces the partials of this launch (slots beyond gridDim.x hold older launches' values
  // and are not read)
  __threadfence();
  double m2 = 0.0;
  for (unsigned b = threadIdx.x; b < gridDim.x; b += ST_THREADS)
    m2 = fmax(m2, __longlong_as_double((long long)__ldcg(&scratch[ST_HDR + b])));
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m2 = fmax(m2, __shfl_xor_sync(0xffffffffu, m2, o));
  if (lane == 0) smx[warp] = m2;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < ST_THREADS / 32; ++w) m2 = fmax(m2, smx[w]);
    *out = m2;
    scratch[0] = 0ull;                                            // leave the counter as the next launch needs it
  }
}

// device address of g_static_scratch, looked up once per device with that device current
constexpr int ST_MAX_DEVICES = 64;
std::mutex g_addr_mutex;
unsigned long long* g_scratch_addr[ST_MAX_DEVICES] = {nullptr};

struct StaticDeviceGuard {
  int prev = -1;
  bool ok = true;
  explicit StaticDeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
    if (prev != dev) ok = (cudaSetDevice(dev) == cudaSuccess);
  }
  ~StaticDeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

}  // namespace
}  // namespace rg

extern "C" {

int rgrmhd_max_speed_static(const int n[3], const double dx[3], const double* const metric_dev[10],
                            const double* const prims_dev[14], double gamma_eos, int wave_speed_mode,
                            double wave_rho_switch, int device, void* stream, double* max_speed_dev) {
  using namespace rg;
  if (!n || !dx || !metric_dev || !max_speed_dev) return RGRMHD_E_INVALID;
  if (wave_speed_mode != RGRMHD_WAVE_LIGHT && wave_speed_mode != RGRMHD_WAVE_MHD_INSIDE) return RGRMHD_E_INVALID;
  const bool mhd_mode = wave_speed_mode == RGRMHD_WAVE_MHD_INSIDE;
  for (int d = 0; d < 3; ++d)
    if (n[d] < 1 || !(dx[d] > 0.0)) return RGRMHD_E_INVALID;
  for (int q = 0; q < 10; ++q)
    if (!metric_dev[q]) return RGRMHD_E_INVALID;
  if (mhd_mode) {
    if (!prims_dev || !(gamma_eos > 1.0)) return RGRMHD_E_INVALID;
    for (int v = 0; v < NPRIM; ++v)
      if (!prims_dev[v]) return RGRMHD_E_INVALID;
  }
  if (device < 0 || device >= ST_MAX_DEVICES) return RGRMHD_E_INVALID;
  // the limit of the static scratch array, checked before anything is touched
  long long cells = 1;
  for (int d = 0; d < 3; ++d) {   // factor by factor: the product of three ints can overflow 64 bits
    cells *= n[d];
    if (cells > ST_MAX_CELLS) return RGRMHD_E_TOO_LARGE;
  }

  StaticDeviceGuard guard(device);
  if (!guard.ok) return RGRMHD_E_CUDA;
  unsigned long long* scratch = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_addr_mutex);
    if (!g_scratch_addr[device]) {   // set-up, once per device, with that device current
      void* p = nullptr;
      if (cudaGetSymbolAddress(&p, g_static_scratch) != cudaSuccess || !p) return RGRMHD_E_CUDA;
      g_scratch_addr[device] = (unsigned long long*)p;
    }
    scratch = g_scratch_addr[device];
  }

  GridView G;
  std::memset(&G, 0, sizeof(G));
  long long ntot = 1;
  for (int d = 0; d < 3; ++d) {
    G.n[d] = n[d];
    G.g[d] = n[d] > 1 ? 3 : 0;
    G.np[d] = n[d] + 2 * G.g[d];
    G.dx[d] = dx[d];
    G.inv_dx[d] = n[d] > 1 ? 1.0 / dx[d] : 0.0;                  // as rgrmhd_create sets them
    G.inv_12dx[d] = n[d] > 1 ? 1.0 / (12.0 * dx[d]) : 0.0;
    ntot *= G.np[d];
  }
  G.stride[0] = 1; G.stride[1] = G.np[0]; G.stride[2] = (long long)G.np[0] * G.np[1];
  G.ntot = ntot;
  G.Gamma = gamma_eos;
  G.wave_mode = wave_speed_mode;
  G.wave_rho_switch = wave_rho_switch;
  for (int q = 0; q < 10; ++q) G.met[q] = metric_dev[q];   // alpha, beta^x y z, gamma_xx xy xz yy yz zz = MALP .. MGZZ
  if (mhd_mode)
    for (int v = 0; v < NPRIM; ++v) G.P[v] = const_cast<double*>(prims_dev[v]);   // read only

  cudaStream_t st = (cudaStream_t)stream;
  // the counter must start at zero whatever an earlier (possibly aborted) launch left behind
  if (cudaMemsetAsync(scratch, 0, ST_HDR * sizeof(unsigned long long), st) != cudaSuccess) return RGRMHD_E_CUDA;
  const unsigned ctas = (unsigned)((cells + ST_CHUNK - 1) / ST_CHUNK);
  k_max_speed_static<<<ctas, ST_THREADS, 0, st>>>(G, scratch, mhd_mode, max_speed_dev);
  return cudaGetLastError() == cudaSuccess ? RGRMHD_OK : RGRMHD_E_CUDA;
}

}  // extern "C"
