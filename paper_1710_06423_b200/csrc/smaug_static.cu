// smaug_static.cu -- smaug_wavespeeds_static (include/smaug.h): the wave-speed reduction of c-4 for callers that may
// not allocate device memory.  Same per-cell arithmetic as wavespeed_kernel (cell_wavespeeds, smaug_aux_kernels.cuh);
// what differs is where the reduction's working memory lives: not in a context's workspace (which somebody had to
// allocate), but in the file-scope device array below, which is part of the loaded library image.
//
// Rules this file keeps:
//   * it calls no cudaMalloc / cudaFree / cudaMallocAsync and no library routine that allocates device memory;
//   * in host code `g_static_scratch` is only a handle for the runtime, never an address a kernel may be given: the
//     device address is looked up with cudaGetSymbolAddress, once per device, with that device current, and it is
//     that looked-up pointer which the launch passes on;
//   * the array is shared by every call in the process and keeps what the last call left in it, so the one word that
//     must start at zero (the arrival counter) is cleared in stream order before each launch, and two calls whose
//     kernels overlap on the GPU (different streams, no dependency) race on it -- the header says so.
#include "../../include/smaug.h"

#include <cstdio>
#include <mutex>

#include "smaug_aux_kernels.cuh"

namespace smaug {
int set_last_error(int code, const char* msg);   // smaug.cu: stores the message smaug_last_error() returns
}

namespace {

using namespace smaug;

constexpr int ST_THREADS = 256;                                   // threads per block
constexpr int ST_CELLS_PER_BLOCK = 4096;                          // each block reduces one run of 4096 cells
constexpr int ST_MAX_BLOCKS = 16384;                              // => at most 16384 * 4096 = 67,108,864 cells
constexpr int ST_HEADER_WORDS = 32;                               // 256 bytes; word 0 = arrival counter
constexpr int ST_WORDS = ST_HEADER_WORDS + 4 * ST_MAX_BLOCKS;     // 65,568 words = 524,544 bytes (about 0.5 MiB)
static_assert((long long)ST_MAX_BLOCKS * ST_CELLS_PER_BLOCK == SMAUG_WAVESPEEDS_STATIC_MAX_CELLS,
              "smaug.h states the limit this array gives");

// The reduction's scratch: [0] arrival counter, [32 + 4 b + k] maximum number k of block b (fp64 bit pattern).
// Every GPU that loads libsmaug.so holds these 524,544 bytes until the process exits.
static __device__ __align__(256) unsigned long long g_static_scratch[ST_WORDS];

// Device address of g_static_scratch per device ordinal; 0 = not looked up yet.
constexpr int ST_MAX_DEVICES = 64;
unsigned long long* g_scratch_addr[ST_MAX_DEVICES];
std::mutex g_scratch_mutex;

// Block b reduces cells [4096 b, 4096 (b + 1)) of the interior-only arrays to four maxima and stores them in the
// scratch; the block that arrives last (arrival counter) folds all blocks' maxima and writes out[0..3].
// w = [6][n] rho~, mx, my, e~, bx~, by~; bg = [4][n] rho_b, e_b, Bbx, Bby (read only when BG).
template <bool BG>
__global__ void __launch_bounds__(ST_THREADS) wavespeed_static_kernel(const double* __restrict__ w,
                                                                      const double* __restrict__ bg, long long n,
                                                                      double gamma, unsigned long long* scratch,
                                                                      double* __restrict__ out) {
  __shared__ double sh[4 * 32];
  __shared__ int last;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  double m[4] = {0.0, 0.0, 0.0, 0.0};
  const long long q0 = (long long)blockIdx.x * ST_CELLS_PER_BLOCK;
  for (int s = threadIdx.x; s < ST_CELLS_PER_BLOCK; s += ST_THREADS) {
    const long long q = q0 + s;
    if (q >= n) break;
    double rho = w[q], e = w[3 * n + q], Bx = w[4 * n + q], By = w[5 * n + q];
    if (BG) {
      rho = bg[q] + rho;
      e = bg[n + q] + e;
      Bx = bg[2 * n + q] + Bx;
      By = bg[3 * n + q] + By;
    }
    double o[4];
    cell_wavespeeds(rho, w[n + q], w[2 * n + q], e, Bx, By, gamma, true, o);
#pragma unroll
    for (int k = 0; k < 4; ++k) m[k] = fmax(m[k], o[k]);
  }
#pragma unroll
  for (int k = 0; k < 4; ++k) m[k] = warp_max(m[k]);
  if (lane == 0) {
#pragma unroll
    for (int k = 0; k < 4; ++k) sh[k * 32 + wid] = m[k];
  }
  __syncthreads();
  if (wid == 0) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      double v = lane < ST_THREADS / 32 ? sh[k * 32 + lane] : 0.0;
      v = warp_max(v);
      if (lane == 0) scratch[ST_HEADER_WORDS + 4 * blockIdx.x + k] = (unsigned long long)__double_as_longlong(v);
    }
    if (lane == 0) {
      __threadfence();                                             // the four stores above before the arrival
      last = atomicAdd(&scratch[0], 1ULL) == (unsigned long long)gridDim.x - 1ULL;
    }
  }
  __syncthreads();
  if (!last) return;
  __threadfence();                                                 // every other block's stores are visible from here
  const volatile unsigned long long* part = scratch + ST_HEADER_WORDS;
#pragma unroll
  for (int k = 0; k < 4; ++k) m[k] = 0.0;
  for (int b = threadIdx.x; b < (int)gridDim.x; b += ST_THREADS) {
#pragma unroll
    for (int k = 0; k < 4; ++k) m[k] = fmax(m[k], __longlong_as_double((long long)part[4 * b + k]));
  }
#pragma unroll
  for (int k = 0; k < 4; ++k) m[k] = warp_max(m[k]);
  __syncthreads();                                                 // sh is reused
  if (lane == 0) {
#pragma unroll
    for (int k = 0; k < 4; ++k) sh[k * 32 + wid] = m[k];
  }
  __syncthreads();
  if (wid == 0) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      double v = lane < ST_THREADS / 32 ? sh[k * 32 + lane] : 0.0;
      v = warp_max(v);
      if (lane == 0) out[k] = v;
    }
    if (lane == 0) scratch[0] = 0ULL;                              // leave the counter as the next call needs it
  }
}

int failf(int code, const char* fmt, long long a = 0, long long b = 0) {
  char buf[256];
  std::snprintf(buf, sizeof buf, fmt, a, b);
  return set_last_error(code, buf);
}

int fail_cuda(const char* what, cudaError_t e) {
  char buf[256];
  std::snprintf(buf, sizeof buf, "smaug_wavespeeds_static: %s: %s", what, cudaGetErrorString(e));
  return set_last_error(SMAUG_ECUDA, buf);
}

// Set-up, once per device, with that device current: ask the runtime where this device keeps g_static_scratch.
// (Using the name g_static_scratch itself as a pointer in host code would hand the kernel a host-side address.)
int scratch_for_current_device(unsigned long long** ptr) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail_cuda("no CUDA device (libsmaug has no CPU fallback)", e);
  if (dev < 0 || dev >= ST_MAX_DEVICES) return failf(SMAUG_EINVAL, "smaug_wavespeeds_static: device ordinal %lld is beyond %lld", dev, ST_MAX_DEVICES - 1);
  std::lock_guard<std::mutex> lock(g_scratch_mutex);
  if (!g_scratch_addr[dev]) {
    unsigned long long* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
    if (e != cudaSuccess || !p) return fail_cuda("cudaGetSymbolAddress of the static scratch array", e);
    g_scratch_addr[dev] = p;
  }
  *ptr = g_scratch_addr[dev];
  return SMAUG_OK;
}

bool on_device(const void* p) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

}  // namespace

extern "C" int smaug_wavespeeds_static(int nx, int ny, double gamma, const double* w, const double* bg, double* out,
                                       void* stream) {
  if (nx < 1 || ny < 1) return failf(SMAUG_EINVAL, "smaug_wavespeeds_static: nx and ny must be >= 1");
  if (!(gamma > 1.0)) return failf(SMAUG_EINVAL, "smaug_wavespeeds_static: gamma must be > 1");
  const long long n = (long long)nx * ny;
  if (n > SMAUG_WAVESPEEDS_STATIC_MAX_CELLS)
    return failf(SMAUG_EINVAL,
                 "smaug_wavespeeds_static: %lld cells exceed the %lld cells the library's static scratch array serves; "
                 "use a context (smaug_create_in_workspace + smaug_get_wavespeeds) for larger grids",
                 n, SMAUG_WAVESPEEDS_STATIC_MAX_CELLS);
  if (!w || !out) return failf(SMAUG_EINVAL, "smaug_wavespeeds_static: w or out is NULL");
  unsigned long long* scratch = nullptr;
  if (int rc = scratch_for_current_device(&scratch)) return rc;
  if (!on_device(w) || !on_device(out) || (bg && !on_device(bg)))
    return failf(SMAUG_EINVAL, "smaug_wavespeeds_static: w, bg and out must be DEVICE pointers (this call makes no staging copies)");
  cudaStream_t st = (cudaStream_t)stream;
  const int blocks = (int)((n + ST_CELLS_PER_BLOCK - 1) / ST_CELLS_PER_BLOCK);
  cudaError_t e = cudaMemsetAsync(scratch, 0, sizeof(unsigned long long), st);   // the arrival counter starts at zero
  if (e != cudaSuccess) return fail_cuda("clearing the arrival counter", e);
  if (bg)
    wavespeed_static_kernel<true><<<blocks, ST_THREADS, 0, st>>>(w, bg, n, gamma, scratch, out);
  else
    wavespeed_static_kernel<false><<<blocks, ST_THREADS, 0, st>>>(w, bg, n, gamma, scratch, out);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail_cuda("kernel launch", e);
  return SMAUG_OK;
}
