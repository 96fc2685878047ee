// pull2_inst.cu -- the two-species-per-thread pull kernel instantiated for one
// (state type, mode) pair; compiled four times by build.py like pull_inst.cu, with
//   -DPULL_REAL=double|float -DPULL_ADAPT=1|0 -DPULL_FN=pull2_kernel_f{64,32}_{adaptive,fixed} -DPULL_CAP=20|24
// (eight times: once per side-a slot capacity, so that the two halves build in parallel)
#define KINNET_PULL_INSTANTIATE
#include "zone_pull2.cuh"

#if !defined(PULL_REAL) || !defined(PULL_ADAPT) || !defined(PULL_FN) || !defined(PULL_CAP)
#error "compile with -DPULL_REAL=... -DPULL_ADAPT=... -DPULL_FN=... -DPULL_CAP=20|24"
#endif

namespace kinnet {

#define KINNET_CAT2(a, b) a##b
#define KINNET_CAT(a, b) KINNET_CAT2(a, b)
#define PULL_FN_CAP24 KINNET_CAT(PULL_FN, _cap24)

#if PULL_CAP == 24
// the half with side-a capacity 24, reached through the capacity-20 half's entry point
pull_fn PULL_FN_CAP24(const PullSchedule& P, int method) { return pick_pull2<PULL_REAL, 24, PULL_ADAPT != 0>(P, method); }
#else
pull_fn PULL_FN_CAP24(const PullSchedule& P, int method);
pull_fn PULL_FN(const PullSchedule& P, int method) {
    const pull_fn f = pick_pull2<PULL_REAL, 20, PULL_ADAPT != 0>(P, method);
    return f ? f : PULL_FN_CAP24(P, method);
}
#endif

#if PULL_ADAPT != 0 && defined(PULL2_DEFINE_SUPPORTED) && PULL_CAP == 20
bool pull2_supported(const PullSchedule& P, int* spill) {
    int sa, sb, s2;
    if (!pull2_sides(P, sa, sb, s2) || pull2_kernel_f64_adaptive(P, 0) == nullptr) return false;
    if (spill) *spill = pull2_cap_a(sa) - kPull2RegA + kPull2SpillB + (P.nslots > 0 ? 2 * kPullNSlots : 0);
    return true;
}

int pull2_stair_class(const PullSchedule& P) {
    int sa, sb, s2;
    if (!pull2_sides(P, sa, sb, s2) || P.T / 64 < 2) return 0;
    if (P.T / 2 > 128) return 0;  // 160/192-thread blocks run the branching loop (zone_pull2.cuh: BRF), no per-warp copies
    const int nw = P.T / 64, cap_a = pull2_cap_a(sa);
    int cls = 1 | 2;
    for (int t = 0; t < P.T; ++t) {
        const int vw = t / 32;
        if (vw < nw) {
            if (P.n_slots[t] > pull2_stair_a(cap_a, vw)) return 0;
        } else {
            const int w = 2 * nw - 1 - vw;
            if (P.n_slots[t] > pull2_stair_b(kPull2CapB, nw, w)) cls |= 1 << (8 + w);
            if (w == 0 && P.owner[t] >= 0) cls &= ~2;
        }
    }
    return cls;
}
#endif

}  // namespace kinnet
