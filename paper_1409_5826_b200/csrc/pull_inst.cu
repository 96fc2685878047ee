// pull_inst.cu -- the pull kernel instantiated for one (state type, mode) pair.
// build.py compiles this file four times, in parallel, with
//   -DPULL_REAL=double|float -DPULL_ADAPT=1|0 -DPULL_FN=pull_kernel_f{64,32}_{adaptive,fixed}
// so that the block-size x slot-capacity classes do not serialise the build.
#define KINNET_PULL_INSTANTIATE
#include "zone_pull.cuh"

#if !defined(PULL_REAL) || !defined(PULL_ADAPT) || !defined(PULL_FN)
#error "compile with -DPULL_REAL=... -DPULL_ADAPT=... -DPULL_FN=..."
#endif

namespace kinnet {

pull_fn PULL_FN(const PullSchedule& P, int method) { return pick_pull_real<PULL_REAL, PULL_ADAPT != 0>(P, method); }

}  // namespace kinnet
