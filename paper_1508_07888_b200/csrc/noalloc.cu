// noalloc.cu -- emma_rt_photons_total_noalloc (include/emma_rt.h): the photon total of A15, sum_i N_i dV, of a caller-owned
// radiation array, with NO allocation of any kind.  For callers that cannot call cudaMalloc (code under CUDA graph capture,
// tight serving loops, harnesses that forbid it) and therefore cannot create a handle, whose arena holds the scratch of every
// other kernel.
//
// It is a variant of the state query of emma_rt_step (n_steps = 0; util.cu: sum_N_kernel + sum_parts_kernel): the same grid,
// the same per-thread strides, the same fixed-shape reduction tree, so the same bits -- but the per-block partial sums live in
// a file-scope `static __device__` array instead of the handle's arena.  Every GPU that loads the library holds that array
// (NOALLOC_MAX_BLOCKS x sizeof(Partial) = 1024 x 88 B = 88 KB) until the process exits.
//
// The array's NAME is a host-side stand-in in host code, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, looked up once per device with that device current (first call on that device) and kept.
//
// All calls share the array.  Every slot the second kernel reads is written by the first kernel of the same call (blocks
// 0 .. nb-1 write slots 0 .. nb-1, nb slots are read), so nothing has to start at zero and nothing is left over from the
// last call that a later call could see; but two calls that OVERLAP on the GPU (different streams, or graphs replayed
// concurrently) race on it.  Calls on one stream are safe.
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>

#include "emma_rt.h"
#include "emma_rt_internal.cuh"

namespace emma {
namespace {

constexpr int NOALLOC_MAX_BLOCKS = 1024;       // as launch_sum_N: at most 1024 blocks of 256 threads, grid-stride
constexpr int NOALLOC_MAX_DEVICES = 64;

static __device__ __align__(256) Partial g_noalloc_parts[NOALLOC_MAX_BLOCKS];

// device address of g_noalloc_parts per CUDA ordinal (0 = not looked up yet).  Two threads racing through the first call on
// a device both look the address up and store the same value.
std::atomic<Partial*> g_noalloc_addr[NOALLOC_MAX_DEVICES];

// sum of U[i].x over i < n, times dV: per-block fp64 partials in index order (the arithmetic of util.cu: sum_N_kernel)
__global__ void __launch_bounds__(256)
noalloc_sum_N_kernel(const float4* __restrict__ U, long long n, double dV, Partial* __restrict__ parts)
{
  Acc a;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
    a.total += (double)U[i].x;
  a.total *= dV;
  block_reduce_store(a, parts + blockIdx.x);
}
// one block adds the partials in index order (util.cu: sum_parts_kernel)
__global__ void __launch_bounds__(256)
noalloc_sum_parts_kernel(const Partial* __restrict__ parts, int n_parts, double* __restrict__ out)
{
  __shared__ Partial s_tot;
  Acc a;
  for (int i = threadIdx.x; i < n_parts; i += blockDim.x) a.total += parts[i].total;
  block_reduce_store(a, &s_tot);
  __syncthreads();
  if (threadIdx.x == 0) *out = s_tot.total;
}

int refuse(char* err, size_t err_len, int code, const char* fmt, ...)
{
  if (err && err_len > 0) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(err, err_len, fmt, ap);
    va_end(ap);
  }
  return code;
}

}  // namespace
}  // namespace emma

extern "C" EMMA_RT_API int emma_rt_photons_total_noalloc(const void* U_dev, int64_t n_cellgroups, double dV, double* total_dev,
                                                         void* stream, char* err, size_t err_len)
{
  using namespace emma;
  if (err && err_len > 0) err[0] = 0;
  if (!total_dev) return refuse(err, err_len, EMMA_RT_EINVAL, "total_dev is NULL (it must point to one double in device memory)");
  if (n_cellgroups < 0) return refuse(err, err_len, EMMA_RT_EINVAL, "n_cellgroups = %lld is negative", (long long)n_cellgroups);
  if (n_cellgroups > (int64_t)EMMA_RT_NOALLOC_MAX_CELLGROUPS)
    return refuse(err, err_len, EMMA_RT_EINVAL, "n_cellgroups = %lld exceeds EMMA_RT_NOALLOC_MAX_CELLGROUPS = %lld (the static scratch holds "
                  "%d block sums; sum the array in pieces)", (long long)n_cellgroups, (long long)EMMA_RT_NOALLOC_MAX_CELLGROUPS, NOALLOC_MAX_BLOCKS);
  if (n_cellgroups > 0 && !U_dev) return refuse(err, err_len, EMMA_RT_EINVAL, "U_dev is NULL with n_cellgroups = %lld", (long long)n_cellgroups);
  if ((reinterpret_cast<uintptr_t>(U_dev) & 15u) != 0) return refuse(err, err_len, EMMA_RT_EINVAL, "U_dev is not 16-byte aligned");
  if (!(dV > 0.0) || !std::isfinite(dV)) return refuse(err, err_len, EMMA_RT_EINVAL, "dV = %g is not a positive finite volume", dV);

  // set-up, once per device, with that device current: the device address of the static scratch
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return refuse(err, err_len, EMMA_RT_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return refuse(err, err_len, EMMA_RT_ECUDA, "CUDA ordinal %d is outside 0..%d", dev, NOALLOC_MAX_DEVICES - 1);
  Partial* parts = g_noalloc_addr[dev].load(std::memory_order_acquire);
  if (!parts) {
    e = cudaGetSymbolAddress((void**)&parts, g_noalloc_parts);
    if (e != cudaSuccess || !parts)
      return refuse(err, err_len, EMMA_RT_ECUDA, "cudaGetSymbolAddress(static scratch) on device %d: %s", dev, cudaGetErrorString(e));
    g_noalloc_addr[dev].store(parts, std::memory_order_release);
  }

  // the launch configuration of launch_sum_N (util.cu): same grid -> same summation order -> same bits
  const long long n = (long long)n_cellgroups;
  const long long want = (n + 255) / 256;
  const int nb = (int)(want < NOALLOC_MAX_BLOCKS ? (want > 0 ? want : 1) : NOALLOC_MAX_BLOCKS);
  cudaStream_t st = (cudaStream_t)stream;
  noalloc_sum_N_kernel<<<nb, 256, 0, st>>>((const float4*)U_dev, n, dV, parts);
  noalloc_sum_parts_kernel<<<1, 256, 0, st>>>(parts, nb, total_dev);
  e = cudaPeekAtLastError();
  if (e != cudaSuccess) return refuse(err, err_len, EMMA_RT_ECUDA, "kernel launch: %s", cudaGetErrorString(e));
  return EMMA_RT_OK;
}
