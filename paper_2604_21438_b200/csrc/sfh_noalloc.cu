// sfh_noalloc.cu — sfh_cfl_dt_noalloc: the CFL reduction (a10; "grid-level reductions", reading R16)
// for callers that must not allocate.
//
// Who that is: code running while a memory pool owns the whole device (a framework's caching allocator that has
// already claimed HBM, so that a cudaMalloc from a library either fails or fragments it), code inside a
// latency-critical loop where cudaMalloc / cudaFree would synchronise the whole device, and plug-ins loaded into a
// host program whose rules forbid any allocation after start-up.  Everywhere else in libsfh the reduction's
// intermediate results (the per-block maximum speeds and the running maximum that the CTAs combine with atomicMax)
// live in the work buffer the caller binds with sfh_bind, and sfh_bind itself cudaMallocs the mesh tables.  Here
// the same two intermediates live in ONE file-scope device array that is part of the library image: every GPU
// that loads libsfh.so holds it (SFH_NOALLOC_MAX_BLOCKS * 8 + 256 bytes = 512.25 KB) until the process exits,
// whether this entry point is ever called or not.  Nothing in this file calls cudaMalloc, cudaFree, a host
// allocator of CUDA, or a library routine that allocates.
//
// The array's name is only a handle in host code (passing it to a kernel would hand the kernel a host address):
// the device address is looked up once per device with cudaGetSymbolAddress, with that device current, on the
// first call made on that device -- make that first call outside any stream capture.
//
// All calls on one device share the array and it keeps whatever the last call left in it.  The running maximum is
// therefore cleared at the start of every call (on the caller's stream), the per-block maxima are overwritten
// before they are read.  Two calls whose kernels may overlap on the GPU (different streams without an event
// between them, or two host threads on different streams) race on the array and give wrong results; calls on one
// stream, or ordered by events, are safe.
#include <cmath>
#include <mutex>
#include <string>

#include "sfh_device.cuh"
#include "sfh_internal.h"

namespace sfh {
namespace {

constexpr int NOALLOC_MAX_BLOCKS = SFH_NOALLOC_MAX_BLOCKS;
constexpr int NOALLOC_HEAD = 32;   // 256 bytes: word 0 = running maximum (bit pattern of a non-negative double)

// [0, NOALLOC_HEAD): head, only word 0 used; [NOALLOC_HEAD, NOALLOC_HEAD + NOALLOC_MAX_BLOCKS): per-block maxima
static __device__ __align__(256) unsigned long long g_noalloc_scratch[NOALLOC_HEAD + NOALLOC_MAX_BLOCKS];

constexpr int MAX_DEVICES = 64;
struct DeviceSetup {
  bool ready = false;
  unsigned long long* scratch = nullptr;   // DEVICE address of g_noalloc_scratch on this device
  int sms = 1;
};
DeviceSetup g_setup[MAX_DEVICES];
std::mutex g_setup_mutex;

int cuda_error(cudaError_t e, const char* where) {
  set_error(std::string("sfh_cfl_dt_noalloc: ") + where + ": " + cudaGetErrorString(e));
  return SFH_ECUDA;
}

// Once per device, with that device current: the device address of the static array and the SM count.
int setup_current_device(DeviceSetup** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return cuda_error(e, "cudaGetDevice");
  if (dev < 0 || dev >= MAX_DEVICES) {
    set_error("sfh_cfl_dt_noalloc: device ordinal beyond " + std::to_string(MAX_DEVICES - 1));
    return SFH_EINVAL;
  }
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  DeviceSetup& s = g_setup[dev];
  if (!s.ready) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (e != cudaSuccess) return cuda_error(e, "cudaGetSymbolAddress");
    int sms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return cuda_error(e, "cudaDeviceGetAttribute");
    s.scratch = static_cast<unsigned long long*>(p);
    s.sms = sms > 0 ? sms : 1;
    s.ready = true;
  }
  *out = &s;
  return SFH_OK;
}

__device__ __forceinline__ double cta_max8(double x, double* wm) {   // 256 threads; valid in thread 0
  x = warp_max(x);
  if ((threadIdx.x & 31) == 0) wm[threadIdx.x >> 5] = x;
  __syncthreads();
  if (threadIdx.x < 32) {
    x = threadIdx.x < 8 ? wm[threadIdx.x] : 0.0;
    x = warp_max(x);
  }
  return x;
}

// Step 1: the maximum of max_d |v_d| + c_s over the 512 cells of every block, one double per block, into the scratch.
// A NaN speed never wins (reading R28: bad cells are reported by sfh_status, not floored), as in max_speed_kernel.
__global__ void __launch_bounds__(256) noalloc_block_max_kernel(const double* __restrict__ U, int count, double gamma,
                                                                double* __restrict__ bmax) {
  __shared__ double wm[8];
  const double gm1 = gamma - 1.0;
  for (int b = blockIdx.x; b < count; b += gridDim.x) {
    const double* Ub = U + size_t(b) * BLK;
    double smax = 0.0;
#pragma unroll
    for (int c = threadIdx.x; c < NC; c += 256) {
      double u[5];
#pragma unroll
      for (int v = 0; v < NV; ++v) u[v] = Ub[v * NC + c];
      const double s = cell_speed(u, gamma, gm1);
      if (s > smax) smax = s;
    }
    smax = cta_max8(smax, wm);
    if (threadIdx.x == 0) bmax[b] = smax;
    __syncthreads();   // wm is reused by the next block of this CTA
  }
}

// Step 2: the maximum of the per-block maxima: one atomicMax per CTA on the bit pattern (non-negative doubles order
// like unsigned integers), onto the word the call cleared.
__global__ void __launch_bounds__(256) noalloc_level_max_kernel(const double* __restrict__ bmax, int count,
                                                                unsigned long long* smax_bits) {
  __shared__ double wm[8];
  double smax = 0.0;
  for (int b = blockIdx.x * 256 + threadIdx.x; b < count; b += gridDim.x * 256) smax = fmax(smax, bmax[b]);
  smax = cta_max8(smax, wm);
  if (threadIdx.x == 0) atomicMax(smax_bits, (unsigned long long)__double_as_longlong(smax));
}

// Step 3: the caller's output.
__global__ void noalloc_finalize_kernel(const unsigned long long* smax_bits, double cfl, double h, double* out) {
  const double s = __longlong_as_double((long long)*smax_bits);
  out[0] = cfl * h / s;
  out[1] = s;
}

}  // namespace
}  // namespace sfh

extern "C" int sfh_cfl_dt_noalloc(const double* d_U, int64_t nblocks, double gamma, double cfl, double h,
                                  double* d_out, void* stream) {
  using namespace sfh;
  if (!d_U || !d_out) {
    set_error("sfh_cfl_dt_noalloc: null state or output pointer");
    return SFH_EINVAL;
  }
  if (nblocks < 1) {
    set_error("sfh_cfl_dt_noalloc: nblocks must be at least 1");
    return SFH_EINVAL;
  }
  if (nblocks > NOALLOC_MAX_BLOCKS) {
    set_error("sfh_cfl_dt_noalloc: " + std::to_string(nblocks) + " blocks exceed the built-in scratch of SFH_NOALLOC_MAX_BLOCKS = " +
              std::to_string(NOALLOC_MAX_BLOCKS) + " blocks; use sfh_cfl_dt on a bound mesh (caller-allocated work buffer) instead");
    return SFH_EINVAL;
  }
  if (!(gamma > 1.0) || !(cfl > 0.0) || !(h > 0.0)) {
    set_error("sfh_cfl_dt_noalloc: needs gamma > 1, cfl > 0, h > 0");
    return SFH_EINVAL;
  }
  DeviceSetup* s = nullptr;
  if (int rc = setup_current_device(&s)) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  unsigned long long* smax_bits = s->scratch;
  double* bmax = reinterpret_cast<double*>(s->scratch + NOALLOC_HEAD);
  const int count = int(nblocks);

  cudaError_t e = cudaMemsetAsync(smax_bits, 0, sizeof(unsigned long long), st);   // the last call's maximum goes
  if (e != cudaSuccess) return cuda_error(e, "cudaMemsetAsync");
  const int grid1 = count < s->sms * 8 ? count : s->sms * 8;
  noalloc_block_max_kernel<<<grid1, 256, 0, st>>>(d_U, count, gamma, bmax);
  if ((e = cudaGetLastError()) != cudaSuccess) return cuda_error(e, "noalloc_block_max_kernel");
  const int need = (count + 2047) / 2048;
  noalloc_level_max_kernel<<<need < s->sms ? need : s->sms, 256, 0, st>>>(bmax, count, smax_bits);
  if ((e = cudaGetLastError()) != cudaSuccess) return cuda_error(e, "noalloc_level_max_kernel");
  noalloc_finalize_kernel<<<1, 1, 0, st>>>(smax_bits, cfl, h, d_out);
  if ((e = cudaGetLastError()) != cudaSuccess) return cuda_error(e, "noalloc_finalize_kernel");
  return SFH_OK;
}
