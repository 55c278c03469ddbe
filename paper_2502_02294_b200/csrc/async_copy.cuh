// async_copy.cuh -- cp.async (LDGSTS) helpers shared by the marching sweeps (sweep_march.cu) and the pipelined particle
// kernels (pm.cu).  Every thread copies 4-byte words it alone will read back, so cp.async.wait_group is the only
// synchronisation these kernels need -- no barrier.  Product code: shares nothing with oracle/.
#pragma once

namespace dh {

__device__ __forceinline__ void cp_async4(float* smem_dst, const float* gsrc) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int PENDING>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(PENDING) : "memory"); }


}  // namespace dh
