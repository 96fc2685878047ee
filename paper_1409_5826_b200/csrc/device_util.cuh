// device_util.cuh -- warp-level helpers shared by the zone kernels (internal).
#pragma once
#include <cuda_runtime.h>

namespace kinnet {

// Barrier 0 over the whole CTA, written as the PTX instruction itself.  In the staircase of the
// two-species kernel (zone_pull2.cuh) every warp of a CTA runs its own compiled copy of the
// sub-step loop, so the warps meet at barrier call sites that differ from warp to warp.  That is
// what PTX defines: a barrier resource counts the warps that arrive, whatever their program
// counter, and .aligned only asks that all threads of ONE warp execute the same instance (they
// do: the copy is chosen per warp).  CUDA C++ makes no such promise for __syncthreads() under a
// condition that differs across the block, so the design's contract is spelled out here instead
// of resting on how __syncthreads() happens to compile.  The contract the callers keep: every
// copy executes the same number of barriers per sub-step (two: A behind the publishes, B before
// the finalize) and leaves the loop on values read from shared memory after B, identical in
// every warp.
__device__ __forceinline__ void cta_barrier() { asm volatile("barrier.sync.aligned 0;" ::: "memory"); }

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Minimum over the warp of non-negative doubles (or +inf; NaN loses): the bit
// patterns order like unsigned integers, so two REDUX.MIN do it.
__device__ __forceinline__ double warp_min_pos(double c) {
    const unsigned hi = static_cast<unsigned>(__double2hiint(c));
    const unsigned mh = __reduce_min_sync(0xffffffffu, hi);
    const unsigned lo = (hi == mh) ? static_cast<unsigned>(__double2loint(c)) : 0xffffffffu;
    const unsigned ml = __reduce_min_sync(0xffffffffu, lo);
    return __hiloint2double(static_cast<int>(mh), static_cast<int>(ml));
}

// Maximum over the warp of non-negative doubles (a NaN wins; callers treat it as no
// candidate): the same two REDUX on the bit pattern.
__device__ __forceinline__ double warp_max_pos(double c) {
    const unsigned hi = static_cast<unsigned>(__double2hiint(c));
    const unsigned mh = __reduce_max_sync(0xffffffffu, hi);
    const unsigned lo = (hi == mh) ? static_cast<unsigned>(__double2loint(c)) : 0u;
    const unsigned ml = __reduce_max_sync(0xffffffffu, lo);
    return __hiloint2double(static_cast<int>(mh), static_cast<int>(ml));
}

// Integrated energy release of one zone (reading Q19):
// sum over the CTA of the per-thread terms B_i (Y_i - Y_i(0)), in a fixed order (warp
// butterfly, then warps in index order).  scratch: >= 32 doubles of shared memory that
// nobody else touches any more; every thread of the CTA must call.
__device__ __forceinline__ void zone_energy_out(double e, double* scratch, double* out) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nw = (blockDim.x + 31) >> 5;
    e = warp_sum(e);
    __syncthreads();
    if (lane == 0) scratch[warp] = e;
    __syncthreads();
    if (tid == 0) {
        double s = 0.0;
        for (int w = 0; w < nw; ++w) s += scratch[w];
        *out = s;
    }
}

}  // namespace kinnet
