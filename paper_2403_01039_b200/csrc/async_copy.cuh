// async_copy.cuh -- asynchronous global -> shared staging (sm_80+ cp.async, 16 bytes per request, L2 only) used by
// the persistent, double-buffered FFT pass kernels: the tile of the NEXT work item streams into one shared-memory
// buffer while the line FFTs of the current one run on the other, so that HBM requests stay in flight during the
// arithmetic and across the barriers of a pass.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace r3d {

__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// 16-byte asynchronous copy, bypassing L1 (.cg): dst in shared memory, src in global memory, both 16-byte aligned
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem_addr(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

}  // namespace r3d
