// async_copy.cuh -- the one copy of the mbarrier + TMA (cp.async.bulk / cp.async.bulk.tensor) helpers of the sm_100a
// kernels that feed shared-memory rings asynchronously (transport_tma.cu, transport_hll.cu, fused.cu, chemistry.cu).
// Elected threads issue the copies; every consumer waits on the stage's mbarrier phase.
#pragma once
#include <cuda.h>

namespace emma {
namespace acp {

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init()
{
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes)
{
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
// plain arrive (release): one count of the current phase
__device__ __forceinline__ void mbar_arrive(unsigned bar)
{
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(bar) : "memory");
}
// Wait for a phase.  `try_wait` with a suspend-time hint parks the thread in hardware until the phase completes (or the hint,
// in ns, runs out) -- a waiting warp then costs one instruction per wake-up instead of a polling loop that takes issue slots
// from the warps it is waiting for (profiles/r2a_summary.md: polls were 13 % of the fused pass's issued instructions).
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
  unsigned done;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done) : "r"(bar), "r"(parity), "r"(20000u) : "memory");
  } while (!done);
}
// waits on other warps (not on data): the same
template <int SLEEP_NS = 64>
__device__ __forceinline__ void mbar_wait_relaxed(unsigned bar, unsigned parity)
{
  mbar_wait(bar, parity);
}
// one box of a rank-3 tensor -> shared memory, completion (bytes) on an mbarrier
__device__ __forceinline__ void tma_load_3d(unsigned dst, const CUtensorMap* map, unsigned bar, int cx, int cy, int cz)
{
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
      :: "r"(dst), "l"(map), "r"(bar), "r"(cx), "r"(cy), "r"(cz) : "memory");
}

// a contiguous run of bytes (multiple of 16, 16-byte aligned on both sides) -> shared memory, completion on an mbarrier
__device__ __forceinline__ void bulk_load(unsigned dst, const void* src, unsigned bytes, unsigned bar)
{
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               :: "r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

}  // namespace acp
}  // namespace emma
