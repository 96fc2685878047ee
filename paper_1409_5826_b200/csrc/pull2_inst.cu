// pull2_inst.cu -- the two-species-per-thread pull kernel instantiated for one
// (state type, mode) pair; compiled four times by build.py like pull_inst.cu, with
//   -DPULL_REAL=double|float -DPULL_ADAPT=1|0 -DPULL_FN=pull2_kernel_f{64,32}_{adaptive,fixed}
#define KINNET_PULL_INSTANTIATE
#include "zone_pull2.cuh"

#if !defined(PULL_REAL) || !defined(PULL_ADAPT) || !defined(PULL_FN)
#error "compile with -DPULL_REAL=... -DPULL_ADAPT=... -DPULL_FN=..."
#endif

namespace kinnet {

pull_fn PULL_FN(const PullSchedule& P, int method) { return pick_pull2<PULL_REAL, PULL_ADAPT != 0>(P, method); }

#if PULL_ADAPT != 0 && defined(PULL2_DEFINE_SUPPORTED)
bool pull2_supported(const PullSchedule& P, int* spill) {
    int sa, sb, s2;
    if (!pull2_sides(P, sa, sb, s2) || pick_pull2<double, true>(P) == nullptr) return false;
    if (spill) *spill = pull2_cap_a(sa) - kPull2RegA + kPull2SpillB + (P.nslots > 0 ? 2 * kPullNSlots : 0);
    return true;
}

int pull2_stair_class(const PullSchedule& P) {
    int sa, sb, s2;
    if (!pull2_sides(P, sa, sb, s2) || P.T / 64 < 2) return 0;
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
