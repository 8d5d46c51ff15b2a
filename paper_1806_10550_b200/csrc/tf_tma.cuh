// tf_tma.cuh -- TMA (cp.async.bulk.tensor) + mbarrier helpers for the shared-memory rings.
// A marching warp owns 32 lines and only 256 such warps exist at 8192^2, so (a) occupancy cannot hide HBM
// latency and (b) a single warp cannot afford per-element copy instructions.  One elected lane issues ONE
// TMA instruction per [rows x 32] box; completion is signalled on an mbarrier (complete_tx::bytes).
// Out-of-range parts of a box are zero-filled by the hardware, which also handles the ragged edges.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace tf {

__device__ __forceinline__ uint32_t s_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(s_addr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(s_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(s_addr(bar)) : "memory");
}
// Wait for the phase with the given parity.  A failed probe backs off with nanosleep: all warps of a
// sub-problem share one SM sub-partition, and a tight polling loop of the waiting warps was measured to take
// ~20 % of that sub-partition's issue slots away from the warps they are waiting for.
#ifndef TF_WAIT_SLEEP_NS
#define TF_WAIT_SLEEP_NS 100
#endif
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(s_addr(bar)), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    while (!mbar_try_wait(bar, parity)) __nanosleep(TF_WAIT_SLEEP_NS);
}
// global -> shared, 2-D box at (c0 = inner/contiguous coordinate, c1 = outer coordinate)
__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n" ::
            "r"(s_addr(smem_dst)), "l"(map), "r"(c0), "r"(c1), "r"(s_addr(bar))
        : "memory");
}
// shared -> global, 2-D box (out-of-range part is clipped)
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* map, int c0, int c1, const void* smem_src)
{
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.tile.bulk_group [%0, {%1, %2}], [%3];\n" ::"l"(map),
                 "r"(c0), "r"(c1), "r"(s_addr(smem_src))
                 : "memory");
}
__device__ __forceinline__ void tma_store_commit() { asm volatile("cp.async.bulk.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void tma_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;\n" ::"n"(N) : "memory"); }
template <int N>
__device__ __forceinline__ void tma_store_wait_all() { asm volatile("cp.async.bulk.wait_group %0;\n" ::"n"(N) : "memory"); }
// make generic-proxy writes to shared memory visible to the async proxy (before a TMA store)
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }

// round a dynamic-shared-memory base up to 1024 B (the 128-byte swizzle pattern repeats every 1024 B)
__device__ __forceinline__ unsigned char* align1024(unsigned char* p)
{
    const uint32_t a = s_addr(p);
    return p + ((1024u - (a & 1023u)) & 1023u);
}

}  // namespace tf
