// fs_noalloc.cu -- fs_divergence_noalloc (include/fs_noalloc.h): the continuity check of the projected field (PAPER.md
// Eq. 2 / Eq. 6) as ONE entry point that allocates nothing.  The kernel is the variant of the
// divergence + max-norm reduction of the projection pass whose per-block partials and arrival counter live in a file-scope
// static __device__ array instead of the grid's workspace.  Self-contained on purpose: it shares no code with the hot path
// (csrc/*.cu) and changes none of it.
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

#include "../../../include/fs_noalloc.h"

namespace {

constexpr int kThreads = 256;
constexpr int kCellsPerThread = 8;
constexpr int kCellsPerBlock = kThreads * kCellsPerThread;                       // 2048
constexpr int kMaxBlocks = (int)(FS_NOALLOC_MAX_CELLS / kCellsPerBlock);         // 8192
constexpr int kTicketAt = 2 * kMaxBlocks;                                        // the arrival counter sits behind the partials
constexpr int kScratchDoubles = 2 * kMaxBlocks + 32;                             // 131,328 bytes
static_assert((long long)kMaxBlocks * kCellsPerBlock == FS_NOALLOC_MAX_CELLS, "scratch size and stated limit must agree");

// [0, kMaxBlocks): per-block max |div|; [kMaxBlocks, 2 kMaxBlocks): per-block sum div^2; then the arrival counter.
// In HOST code this name is a host-side stand-in, not a device address: the kernel gets the pointer that
// cudaGetSymbolAddress returns (scratch_for_current_device below).  Shared by every call on the device.
static __device__ __align__(256) double g_fs_noalloc_scratch[kScratchDoubles];

__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ double warp_add(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
// block-wide (max, sum) in a fixed order; the totals are valid in thread 0
__device__ __forceinline__ void block_max_sum(double& m, double& s, double* sh /*[16]*/) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  m = warp_max(m); s = warp_add(s);
  __syncthreads();                       // sh may still be read by the previous use
  if (lane == 0) { sh[wid] = m; sh[8 + wid] = s; }
  __syncthreads();
  if (wid == 0) {
    double a = lane < kThreads / 32 ? sh[lane] : 0.0, b = lane < kThreads / 32 ? sh[8 + lane] : 0.0;
    m = warp_max(a); s = warp_add(b);
  }
}

template <class T>
__global__ void __launch_bounds__(kThreads) k_divergence_noalloc(const T* __restrict__ u, const T* __restrict__ v, const T* __restrict__ w,
                                                                 T* __restrict__ out, double* __restrict__ result, double* scratch,
                                                                 int nx, int ny, int nz, T ihx, T ihy, T ihz) {
  __shared__ double sh[16];
  __shared__ int last;
  const int N = nx * ny * nz;            // <= 2^24
  const int sxy = nx * ny;
  double m = 0.0, s = 0.0;
  const int q0 = blockIdx.x * kCellsPerBlock + threadIdx.x;
#pragma unroll
  for (int it = 0; it < kCellsPerThread; ++it) {
    const int q = q0 + it * kThreads;    // consecutive threads, consecutive cells: coalesced
    if (q < N) {
      const int i = q % nx, t = q / nx, j = t % ny, k = t / ny;
      const int qe = i + 1 == nx ? q + 1 - nx : q + 1;
      const int qn = j + 1 == ny ? q + nx - sxy : q + nx;
      const int qt = k + 1 == nz ? q + sxy - N : q + sxy;
      const T d = (u[qe] - u[q]) * ihx + (v[qn] - v[q]) * ihy + (w[qt] - w[q]) * ihz;
      if (out) out[q] = d;
      const double dd = (double)d;
      m = fmax(m, fabs(dd));
      s += dd * dd;
    }
  }
  block_max_sum(m, s, sh);
  unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch + kTicketAt);
  if (threadIdx.x == 0) {
    __stcg(&scratch[blockIdx.x], m);
    __stcg(&scratch[kMaxBlocks + blockIdx.x], s);
    __threadfence();
    last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  // the last block to arrive adds the partials in a fixed order: the result does not depend on block scheduling
  __threadfence();
  m = 0.0; s = 0.0;
  for (int b = threadIdx.x; b < (int)gridDim.x; b += kThreads) {
    m = fmax(m, __ldcg(&scratch[b]));
    s += __ldcg(&scratch[kMaxBlocks + b]);
  }
  block_max_sum(m, s, sh);
  if (threadIdx.x == 0) { result[0] = m; result[1] = s; *ticket = 0u; }
}

// Device address of the scratch array for the CURRENT device: looked up once per device (set-up), cached afterwards.
cudaError_t scratch_for_current_device(double** out) {
  constexpr int kMaxDevices = 64;
  static std::mutex mu;
  static double* cache[kMaxDevices] = {nullptr};
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(mu);
  if (!cache[dev]) {
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_fs_noalloc_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    cache[dev] = p;
  }
  *out = cache[dev];
  return cudaSuccess;
}

// true if p is device memory of device dev (a host pointer, a managed-on-host or another GPU's pointer is refused)
bool on_device(const void* p, int dev) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeDevice && a.device == dev;
}

}  // namespace

extern "C" fs_status fs_divergence_noalloc(int nx, int ny, int nz, double hx, double hy, double hz, fs_dtype dtype,
                                           const void* u, const void* v, const void* w, void* div_out, double* result,
                                           void* cuda_stream) {
  if (nx < 1 || ny < 1 || nz < 1 || !(hx > 0.0) || !(hy > 0.0) || !(hz > 0.0)) return FS_ERR_INVALID_ARG;
  if (!u || !v || !w || !result || (dtype != FS_F32 && dtype != FS_F64)) return FS_ERR_INVALID_ARG;
  const long long cells = (long long)nx * ny * nz;
  if (cells > FS_NOALLOC_MAX_CELLS) {
    std::fprintf(stderr, "libfs: fs_divergence_noalloc: %d x %d x %d = %lld cells exceed FS_NOALLOC_MAX_CELLS = %lld "
                 "(the static scratch holds one pair of partials per %d cells); use a grid (fs_grid_create) for larger boxes\n",
                 nx, ny, nz, cells, (long long)FS_NOALLOC_MAX_CELLS, kCellsPerBlock);
    return FS_ERR_UNSUPPORTED;
  }
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return FS_ERR_CUDA;
  if (!on_device(u, dev) || !on_device(v, dev) || !on_device(w, dev) || !on_device(result, dev) || (div_out && !on_device(div_out, dev)))
    return FS_ERR_INVALID_ARG;
  double* scratch = nullptr;
  cudaError_t e = scratch_for_current_device(&scratch);
  if (e != cudaSuccess) {
    std::fprintf(stderr, "libfs: fs_divergence_noalloc: cudaGetSymbolAddress(scratch) failed: %s\n", cudaGetErrorString(e));
    return FS_ERR_CUDA;
  }
  cudaStream_t s = (cudaStream_t)cuda_stream;
  // the arrival counter must start at zero whatever an earlier (possibly aborted) call left behind
  if (cudaMemsetAsync(scratch + kTicketAt, 0, sizeof(unsigned int), s) != cudaSuccess) return FS_ERR_CUDA;
  const int blocks = (int)((cells + kCellsPerBlock - 1) / kCellsPerBlock);
  if (dtype == FS_F64)
    k_divergence_noalloc<double><<<blocks, kThreads, 0, s>>>((const double*)u, (const double*)v, (const double*)w, (double*)div_out, result, scratch,
                                                            nx, ny, nz, 1.0 / hx, 1.0 / hy, 1.0 / hz);
  else
    k_divergence_noalloc<float><<<blocks, kThreads, 0, s>>>((const float*)u, (const float*)v, (const float*)w, (float*)div_out, result, scratch,
                                                           nx, ny, nz, (float)(1.0 / hx), (float)(1.0 / hy), (float)(1.0 / hz));
  e = cudaGetLastError();
  if (e != cudaSuccess) {
    std::fprintf(stderr, "libfs: fs_divergence_noalloc: launch failed: %s\n", cudaGetErrorString(e));
    return FS_ERR_CUDA;
  }
  return FS_OK;
}
