// device_util.cuh -- warp-level helpers shared by the zone kernels (internal).
#pragma once
#include <cuda_runtime.h>

namespace kinnet {

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
