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

}  // namespace kinnet
