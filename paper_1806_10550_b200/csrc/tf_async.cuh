// tf_async.cuh -- cp.async (LDGSTS) helpers for the multi-stage shared-memory rings.
// The sweeps have only nx (or ny) independent lines, i.e. 256 warps at 8192^2 on 148 SMs; occupancy
// cannot hide HBM latency, so bytes in flight are decoupled from the warp count: every marching warp
// keeps a ring of NST stages of its next rows in shared memory, filled by cp.async.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tf {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem_u32(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gmem_src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(smem_u32(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

// Warp-cooperative copy of a [rows][W] block of doubles (W = 32 or 16 ... a multiple of 2) from a
// row-major global array (leading dimension ld, first element g) into shared memory (leading dimension
// sld doubles).  Rows >= rows_ok and columns >= cols_ok are skipped (their shared memory is left as is).
// VEC: 16-byte copies (needs ld even, g and s 16-byte aligned, sld even); else 8-byte copies.
template <int ROWS, int W, bool VEC>
__device__ __forceinline__ void warp_copy_block(double* s, int sld, const double* g, size_t ld,
                                                int rows_ok, int cols_ok, int lane)
{
    if (VEC) {
        constexpr int CPR = W / 2;                  // 16-byte chunks per row
        constexpr int TOT = ROWS * CPR;
#pragma unroll
        for (int k = 0; k < (TOT + 31) / 32; ++k) {
            const int idx = k * 32 + lane;
            const int r = idx / CPR, c = (idx % CPR) * 2;
            if (idx < TOT && r < rows_ok && c < cols_ok) cp_async16(s + r * sld + c, g + (size_t)r * ld + c);
        }
    } else {
        constexpr int TOT = ROWS * W;
#pragma unroll
        for (int k = 0; k < (TOT + 31) / 32; ++k) {
            const int idx = k * 32 + lane;
            const int r = idx / W, c = idx % W;
            if (idx < TOT && r < rows_ok && c < cols_ok) cp_async8(s + r * sld + c, g + (size_t)r * ld + c);
        }
    }
}

}  // namespace tf
