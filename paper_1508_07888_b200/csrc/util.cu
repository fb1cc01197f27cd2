// util.cu -- diagnostics reduction and unit conversions at the C-ABI boundary.
#include "emma_rt_internal.cuh"

namespace emma {

namespace {

constexpr float KB15 = 1.5f * 1.380649e-16f;

// Sum the per-block partials of every kernel of this step in a fixed order (thread i takes slots i, i+256, ...;
// then the block tree of block_reduce_store) -> the step's diagnostics; also re-arms the deferral queue counters.
__global__ void __launch_bounds__(256)
finalize_kernel(const Partial* __restrict__ parts, int n_parts, DiagDev* __restrict__ out, unsigned int* __restrict__ qcount,
                double t_sim)
{
  __shared__ Partial s_tot;
  Acc a;
  for (int i = threadIdx.x; i < n_parts; i += blockDim.x) {
    const Partial q = parts[i];
    a.total += q.total; a.injected += q.injected; a.absorbed += q.absorbed; a.recomb += q.recomb; a.outflow += q.outflow;
    a.dtau_min = fminf(a.dtau_min, q.dtau_min); a.nsub_max = max(a.nsub_max, q.nsub_max); a.err |= q.err;
    a.nsub += q.nsub; a.nhalv += q.nhalv; a.nonfinite += q.nonfinite; a.ndefer += q.ndefer;
  }
  block_reduce_store(a, &s_tot);
  __syncthreads();
  if (threadIdx.x == 0) {
    const Partial t = s_tot;
    emma_rt_diag d;
    d.photons_total = t.total; d.photons_injected = t.injected; d.photons_absorbed = t.absorbed;
    d.photons_recomb_emitted = t.recomb; d.photons_outflow = t.outflow; d.dtau_min = (double)t.dtau_min;
    d.subcycles_total = (long long)t.nsub; d.subcycles_max = (long long)t.nsub_max; d.halvings_total = (long long)t.nhalv;
    d.n_nonfinite = (long long)t.nonfinite; d.n_deferred = (long long)t.ndefer; d.t_sim = t_sim;
    out->d = d;
    out->err_last = t.err | (t.nonfinite ? 2u : 0u);
    out->err_sticky |= out->err_last;
    qcount[0] = 0; qcount[1] = 0;
  }
}

__device__ __forceinline__ void decode_x(float xs, float& x, float& y)
{
  if (__float_as_int(xs) < 0) { y = -xs; x = 1.f - y; } else { x = xs; y = 1.f - xs; }
}

__global__ void export_kernel(int field, const LevelDev L, const float4* __restrict__ Ug, float c_red, long long off,
                              long long cnt, void* __restrict__ dst)
{
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < cnt; i += (long long)gridDim.x * blockDim.x) {
    const long long cell = off + i;
    float x, y;
    switch (field) {
      case EMMA_RT_FIELD_U: { const float4 u = Ug[cell]; ((float4*)dst)[i] = make_float4(u.x, u.y * c_red, u.z * c_red, u.w * c_red); break; }
      case EMMA_RT_FIELD_N: ((float*)dst)[i] = Ug[cell].x; break;
      case EMMA_RT_FIELD_F: { const float4 u = Ug[cell]; float* d = (float*)dst + 3 * i; d[0] = u.y * c_red; d[1] = u.z * c_red; d[2] = u.w * c_red; break; }
      case EMMA_RT_FIELD_X: decode_x(L.xs[cell], x, y); ((float*)dst)[i] = x; break;
      case EMMA_RT_FIELD_XNEUTRAL: decode_x(L.xs[cell], x, y); ((float*)dst)[i] = y; break;
      case EMMA_RT_FIELD_T: decode_x(L.xs[cell], x, y); ((float*)dst)[i] = L.eps[cell] / (KB15 * (1.f + x)); break;
      case EMMA_RT_FIELD_E: ((float*)dst)[i] = L.eps[cell] * L.n0[cell]; break;
      case EMMA_RT_FIELD_N0: ((float*)dst)[i] = L.n0[cell]; break;
      case EMMA_RT_FIELD_SUBCYCLES: ((unsigned int*)dst)[i] = L.subc[cell]; break;
    }
  }
}

// src may be the destination itself (emma_rt_step_host uploads raw bytes into the state arrays and converts in place):
// every thread reads its element before it writes it, and no pointer is declared restrict
__global__ void import_kernel(int field, const LevelDev L, float4* Ug, float c_red, long long off,
                              long long cnt, const void* src, unsigned int* bad)
{
  const float rc = 1.f / c_red;
  unsigned int n_bad = 0;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < cnt; i += (long long)gridDim.x * blockDim.x) {
    const long long cell = off + i;
    switch (field) {
      case EMMA_RT_FIELD_U: { const float4 u = ((const float4*)src)[i]; Ug[cell] = make_float4(u.x, u.y * rc, u.z * rc, u.w * rc); break; }
      case EMMA_RT_FIELD_X: {
        const float xin = ((const float*)src)[i];
        if (!(xin >= 0.f && xin <= 1.f)) n_bad++;                      // also NaN
        const float x = (xin != xin) ? xin : fminf(fmaxf(xin, 0.f), 1.f);
        // 1-x is exact in fp32 for x in [0.5, 1] (Sterbenz), so the neutral fraction of the input is kept exactly
        L.xs[cell] = (x <= 0.5f) ? x : __int_as_float(__float_as_int(1.f - x) | 0x80000000);
        break;
      }
      case EMMA_RT_FIELD_T: {
        float x, y;
        decode_x(L.xs[cell], x, y);
        const float Tin = ((const float*)src)[i];
        if (!(Tin > 0.f && Tin < __int_as_float(0x7f800000))) n_bad++;
        // A10 in fp64, rounded once: eps = e/n0 = (3/2)(1+x) k_B T
        L.eps[cell] = (float)(1.5 * 1.380649e-16 * (1.0 + (double)x) * (double)Tin);
        break;
      }
      case EMMA_RT_FIELD_N0: {
        const float v = ((const float*)src)[i];
        if (!(v > 0.f && v < __int_as_float(0x7f800000))) n_bad++;
        L.n0[cell] = v;
        break;
      }
    }
  }
  if (bad && n_bad) atomicAdd(bad, n_bad);                             // rare: only invalid inputs get here
}

// sum of U[i].x over i < n, times dV: per-block fp64 partials in index order, then one block adds them in index order
__global__ void __launch_bounds__(256)
sum_N_kernel(const float4* __restrict__ U, long long n, double dV, Partial* __restrict__ parts)
{
  Acc a;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
    a.total += (double)U[i].x;
  a.total *= dV;
  block_reduce_store(a, parts + blockIdx.x);
}
__global__ void __launch_bounds__(256)
sum_parts_kernel(const Partial* __restrict__ parts, int n_parts, double* __restrict__ out)
{
  __shared__ Partial s_tot;
  Acc a;
  for (int i = threadIdx.x; i < n_parts; i += blockDim.x) a.total += parts[i].total;
  block_reduce_store(a, &s_tot);
  __syncthreads();
  if (threadIdx.x == 0) *out = s_tot.total;
}

__global__ void set_bits_kernel(unsigned int* mask, const int* __restrict__ cells, int n)
{
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) atomicOr(mask + (cells[i] >> 5), 1u << (cells[i] & 31));
}

}  // namespace

int launch_set_bits(unsigned int* mask, const int* cells, int n, cudaStream_t st)
{
  if (n <= 0) return 0;
  set_bits_kernel<<<(n + 127) / 128, 128, 0, st>>>(mask, cells, n);
  return 1;
}

int launch_finalize(const Partial* parts, int n_parts, DiagDev* diag, unsigned int* qcount, double t_sim, cudaStream_t st)
{
  finalize_kernel<<<1, 256, 0, st>>>(parts, n_parts, diag, qcount, t_sim);
  return 1;
}

int launch_export(int field, const LevelDev& L, const float4* Ug, float c_red, long long off, long long cnt, void* dst,
                  cudaStream_t st)
{
  if (cnt <= 0) return 0;
  long long want = (cnt + 255) / 256;
  const int nb = (int)(want < 148 * 16 ? want : 148 * 16);
  export_kernel<<<nb, 256, 0, st>>>(field, L, Ug, c_red, off, cnt, dst);
  return 1;
}

int launch_sum_N(const float4* U, long long n, double dV, Partial* scratch, double* out, cudaStream_t st)
{
  const long long want = (n + 255) / 256;
  const int nb = (int)(want < 1024 ? (want > 0 ? want : 1) : 1024);
  sum_N_kernel<<<nb, 256, 0, st>>>(U, n, dV, scratch);
  sum_parts_kernel<<<1, 256, 0, st>>>(scratch, nb, out);
  return 2;
}

int launch_import(int field, const LevelDev& L, float4* Ug, float c_red, long long off, long long cnt, const void* src,
                  unsigned int* bad, cudaStream_t st)
{
  if (cnt <= 0) return 0;
  long long want = (cnt + 255) / 256;
  const int nb = (int)(want < 148 * 16 ? want : 148 * 16);
  import_kernel<<<nb, 256, 0, st>>>(field, L, Ug, c_red, off, cnt, src, bad);
  return 1;
}

}  // namespace emma
