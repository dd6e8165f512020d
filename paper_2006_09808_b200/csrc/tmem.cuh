// tmem.cuh -- Blackwell tensor memory (TMEM) used as THREAD-PRIVATE state storage of the resident kernel.
//
// TMEM is 128 lanes x 512 columns x 32 bit per SM (256 KB), reached only with tcgen05.ld / tcgen05.st.  With the
// 32x32b shape thread t of a warp reads or writes lane 32*(warp % 4) + t, n consecutive columns per instruction: a
// register-file-like private array per thread, with no addressing arithmetic, that costs neither shared memory nor
// L1/L2 traffic.  Measured on B200 (16 warps, one CTA per SM): 475 B/clk/SM for loads, 860 B/clk/SM for stores
// (profiles/r02/README.md), against 128 B/clk/SM of shared memory.  The resident kernel keeps p^, phi^, qx and chi
// there (pd_resident_tm.cuh): the arrays only their owning thread ever touches.
//
// No tensor-core instruction is issued anywhere: nothing on this path is a dense contraction (BASELINE.json north_star).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace pdk {

// Allocate `ncols` columns (power of two >= 32) for the CTA: executed by warp 0, the base address is published
// through *slot (shared memory) to all threads.  One CTA per SM here, so the allocation cannot block.
__device__ __forceinline__ uint32_t tmem_alloc(uint32_t *slot, const uint32_t ncols) {
    if (threadIdx.x < 32) {
        const uint32_t sa = (uint32_t)__cvta_generic_to_shared(slot);
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(sa), "r"(ncols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    return *slot;
}
// Executed by all threads at the end of the kernel (warp 0 frees after everyone is done).
__device__ __forceinline__ void tmem_free(const uint32_t base, const uint32_t ncols) {
    __syncthreads();
    if (threadIdx.x < 32)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(base), "r"(ncols) : "memory");
}
// This thread's private window: lane quarter of its warp, and one column range per warp of that quarter.
__device__ __forceinline__ uint32_t tmem_thread_window(const uint32_t base, const int cols_per_thread) {
    const uint32_t warp = threadIdx.x >> 5;
    return base + ((32u * (warp & 3u)) << 16) + (warp >> 2) * (uint32_t)cols_per_thread;
}
// All earlier tcgen05.st of this thread have completed (needed before the same thread reads the data back).
__device__ __forceinline__ void tm_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// 4 float2 (8 columns) of this thread's lane, starting at column address `addr`; returns with the data ready
__device__ __forceinline__ void tm_ld(const uint32_t addr, float2 (&v)[4]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];\n\t"
                 "tcgen05.wait::ld.sync.aligned;"
                 : "=f"(v[0].x), "=f"(v[0].y), "=f"(v[1].x), "=f"(v[1].y), "=f"(v[2].x), "=f"(v[2].y), "=f"(v[3].x), "=f"(v[3].y)
                 : "r"(addr)
                 : "memory");
}
__device__ __forceinline__ void tm_st(const uint32_t addr, const float2 (&v)[4]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};"
                 :
                 : "r"(addr), "f"(v[0].x), "f"(v[0].y), "f"(v[1].x), "f"(v[1].y), "f"(v[2].x), "f"(v[2].y), "f"(v[3].x), "f"(v[3].y)
                 : "memory");
}
// 8 float2 (16 columns) of this thread's lane, starting at column address `addr`; returns with the data ready
__device__ __forceinline__ void tm_ld(const uint32_t addr, float2 (&v)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];\n\t"
                 "tcgen05.wait::ld.sync.aligned;"
                 : "=f"(v[0].x), "=f"(v[0].y), "=f"(v[1].x), "=f"(v[1].y), "=f"(v[2].x), "=f"(v[2].y), "=f"(v[3].x), "=f"(v[3].y), "=f"(v[4].x), "=f"(v[4].y), "=f"(v[5].x), "=f"(v[5].y), "=f"(v[6].x), "=f"(v[6].y), "=f"(v[7].x), "=f"(v[7].y)
                 : "r"(addr)
                 : "memory");
}
__device__ __forceinline__ void tm_st(const uint32_t addr, const float2 (&v)[8]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
                 :
                 : "r"(addr), "f"(v[0].x), "f"(v[0].y), "f"(v[1].x), "f"(v[1].y), "f"(v[2].x), "f"(v[2].y), "f"(v[3].x), "f"(v[3].y), "f"(v[4].x), "f"(v[4].y), "f"(v[5].x), "f"(v[5].y), "f"(v[6].x), "f"(v[6].y), "f"(v[7].x), "f"(v[7].y)
                 : "memory");
}
// 16 float2 (32 columns) of this thread's lane, starting at column address `addr`; returns with the data ready
__device__ __forceinline__ void tm_ld(const uint32_t addr, float2 (&v)[16]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];\n\t"
                 "tcgen05.wait::ld.sync.aligned;"
                 : "=f"(v[0].x), "=f"(v[0].y), "=f"(v[1].x), "=f"(v[1].y), "=f"(v[2].x), "=f"(v[2].y), "=f"(v[3].x), "=f"(v[3].y), "=f"(v[4].x), "=f"(v[4].y), "=f"(v[5].x), "=f"(v[5].y), "=f"(v[6].x), "=f"(v[6].y), "=f"(v[7].x), "=f"(v[7].y), "=f"(v[8].x), "=f"(v[8].y), "=f"(v[9].x), "=f"(v[9].y), "=f"(v[10].x), "=f"(v[10].y), "=f"(v[11].x), "=f"(v[11].y), "=f"(v[12].x), "=f"(v[12].y), "=f"(v[13].x), "=f"(v[13].y), "=f"(v[14].x), "=f"(v[14].y), "=f"(v[15].x), "=f"(v[15].y)
                 : "r"(addr)
                 : "memory");
}
__device__ __forceinline__ void tm_st(const uint32_t addr, const float2 (&v)[16]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};"
                 :
                 : "r"(addr), "f"(v[0].x), "f"(v[0].y), "f"(v[1].x), "f"(v[1].y), "f"(v[2].x), "f"(v[2].y), "f"(v[3].x), "f"(v[3].y), "f"(v[4].x), "f"(v[4].y), "f"(v[5].x), "f"(v[5].y), "f"(v[6].x), "f"(v[6].y), "f"(v[7].x), "f"(v[7].y), "f"(v[8].x), "f"(v[8].y), "f"(v[9].x), "f"(v[9].y), "f"(v[10].x), "f"(v[10].y), "f"(v[11].x), "f"(v[11].y), "f"(v[12].x), "f"(v[12].y), "f"(v[13].x), "f"(v[13].y), "f"(v[14].x), "f"(v[14].y), "f"(v[15].x), "f"(v[15].y)
                 : "memory");
}

}  // namespace pdk
