// cp.async (LDGSTS) staging helpers shared by the step kernels: every thread stages what it will itself read, so no
// barrier protects the copies -- a thread waits for its own group only.
#pragma once
#include <cuda_runtime.h>

namespace aton {

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp_async16(void *smem, const void *gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async4(void *smem, const void *gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(smem)), "l"(gmem) : "memory");
}
// L2 prefetches of data a later iteration reads with plain loads (x, T, n_H, the source bits): no register and no shared
// memory is held while the line travels from HBM (profiles/r02_d_step_v5.md)
__device__ __forceinline__ void prefetch_l2(const void *gmem) {
    asm volatile("prefetch.global.L2 [%0];" ::"l"(gmem));
}
__device__ __forceinline__ void prefetch_l2_bulk(const void *gmem, unsigned bytes) {   // 16-byte aligned, bytes % 16 == 0
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(gmem), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_1() { asm volatile("cp.async.wait_group 1;" ::: "memory"); }   // all but the newest group
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

}  // namespace aton
