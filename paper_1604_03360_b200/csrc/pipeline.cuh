// pipeline.cuh -- the few inline-PTX helpers the marching kernels share: per-thread asynchronous global -> shared
// copies (cp.async, SASS LDGSTS) with commit / wait groups, and the one-lane warp shuffle.
//
// Every global read inside a marching loop is a cp.async into the issuing thread's OWN shared-memory slots, a few
// cells ahead of use: no load latency is exposed to the fp64 pipe, and because no thread reads another thread's
// slots no barrier is needed for them (cp.async.wait_group orders a thread's own copies).
#pragma once
#include <cuda_runtime.h>

namespace hydro {

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

template <int BYTES>
__device__ __forceinline__ void cp_async(void* smem, const void* gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(smem_u32(smem)), "l"(gmem), "n"(BYTES) : "memory");
}
// the same with the shared-memory address already converted (keeps the generic -> shared conversion out of loops)
template <int BYTES>
__device__ __forceinline__ void cp_async_s(unsigned smem_addr, const void* gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(smem_addr), "l"(gmem), "n"(BYTES) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <class T>
__device__ __forceinline__ T shfl_up1(T v) { return __shfl_up_sync(0xffffffffu, v, 1); }

// warp-wide max of a non-negative double over the lanes of `mask` (a ballot taken while all 32 lanes were still
// present: lanes outside it have exited), pushed to *bits by the lowest lane of the mask.  The butterfly runs over
// all five offsets; a partner outside the mask contributes nothing.
__device__ __forceinline__ void warp_max_to(double m, unsigned long long* bits, unsigned mask = 0xffffffffu) {
    const unsigned lane = threadIdx.x & 31;
    __syncwarp(mask);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned partner = lane ^ o;
        const unsigned src = (mask >> partner) & 1u ? partner : lane;   // own value when the partner is gone
        m = fmax(m, __shfl_sync(mask, m, src));
    }
    if (lane == (unsigned)(__ffs(mask) - 1) && m > 0.0) atomicMax(bits, (unsigned long long)__double_as_longlong(m));
}

}  // namespace hydro
