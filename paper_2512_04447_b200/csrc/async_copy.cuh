// cp.async (LDGSTS) helpers shared by the librsdft kernels: 16-byte global -> shared copies that
// bypass registers, grouped with commit/wait.  Part of the CUDA path only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace rsdft {

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem)
{
    const uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" :: "n"(N) : "memory"); }

}  // namespace rsdft
