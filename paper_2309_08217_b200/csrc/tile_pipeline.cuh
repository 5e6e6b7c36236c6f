// tile_pipeline.cuh -- shared-memory staging of j-tiles for the all-pairs kernels:
// 1-D bulk asynchronous copies (cp.async.bulk, the TMA engine's UBLKCP path) completing on
// mbarriers, double buffered; plus the warp-aggregated candidate push.
#pragma once

#include "genga_internal.cuh"

namespace genga {

__device__ __forceinline__ uint32_t smem_u32(const void* p)
{
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}

__device__ __forceinline__ void fence_barrier_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

__device__ __forceinline__ void fence_proxy_async()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}

__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}

// Append (body, chunk) for every lane with flag set; one atomic per warp (__ballot_sync + popc).
// Must be executed by all 32 lanes.  Entries past the capacity are dropped; the count keeps
// growing so that the near-field kernel can see the overflow and take the exact path.
__device__ __forceinline__ void push_candidates(unsigned int ballot, bool flag, int body, int chunk,
                                                unsigned int* count, int2* list, unsigned int cap)
{
    const unsigned int lane = threadIdx.x & 31u;
    const int leader = __ffs(ballot) - 1;
    unsigned int base = 0;
    if ((int)lane == leader) base = atomicAdd(count, (unsigned int)__popc(ballot));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (flag) {
        const unsigned int idx = base + __popc(ballot & ((1u << lane) - 1u));
        if (idx < cap) list[idx] = make_int2(body, chunk);
    }
}

}  // namespace genga
