// zone_pull.cuh -- the pull kernel (internal; the public face is include/kinnet.h).
// Included by kinnet.cu (launch side) and by pull_inst.cu, which is compiled once per
// (state type, adaptive/fixed) pair so that the instantiations build in parallel.
#pragma once
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>

#include "../../include/kinnet.h"
#include "device_util.cuh"
#include "schedule.h"

namespace kinnet {

enum Mode { kAdaptive = 0, kFixed = 1, kRhs = 2, kRates = 3 };

// ---------------------------------------------------------------------------
// Pull kernel (the one bench.py times when the network qualifies, see
// schedule.h "Pull schedule"): no flux array, two barriers per sub-step.
//
//   publish   YP[c][t] = y * {1, Y_hub0, Y_hub1, Y_hub2}[c]            4 STS
//   rate sums k = F-/y and the six hub-row partials from the per-thread
//             coefficients K, G0, Gx (sums of rates formed once per call)
//   ------------------------------------------------------------------- barrier
//   P-slots   F+ = sum_e R[e] * YP[f1[e]] (* YP[f2[e]])   fluxes at the consumer
//   dt        candidate eps*max(y,floor)/|F+ - k y|, warp min -> redmin[warp]
//   hub rows  transposed warp butterfly of the six partials -> red[warp][row]
//   ------------------------------------------------------------------- barrier
//   finalize  every warp redundantly: lanes 0..2 sum the hub rows over warps,
//             zone-wide dt, hub update, shuffle-broadcast of the new hub Y
//   update    k dt >= kappa ? (y + dt F+)/(1 + k dt) : y + dt (F+ - k y)
// Rates, rate sums and every gather offset of a thread stay in registers for
// the whole hydro step (topology is static, sub-steps number 1e2..1e4).
// ---------------------------------------------------------------------------
constexpr int kJ2C = kinnet::kPullMaxSlots2;

// resident CTAs per SM the 160-thread instantiation is compiled for (register budget
// 65536 / (160 * MINB)); build.py may override it for A/B runs
#ifndef KINNET_MINB160
#define KINNET_MINB160 3
#endif

struct KPull {
    int N, M, nbs;
    int hub[kinnet::kPullHubs];
    int mode;                 // Mode: kAdaptive, kFixed or kRhs
    const double* coef;       // [8][M] reaction order: a0 + ln p, a1..a6, n_react - 1
    const int32_t* owner;     // [T]
    const uint32_t* cnt;      // [T] n_slots | n_slots2 << 8
    const int32_t* slot_rxn;  // [kPullMaxSlots][T] reaction | nu << 24, -1 = empty
    const uint32_t* f1_pack;  // [kPullMaxSlots / 2][T] two 16-bit YP byte offsets per word
    const uint32_t* f2_pack;  // [kPullMaxSlots2 / 2][T]
    const uint16_t* agg_ptr;  // [kPullCoefs + 1][T]
    const int32_t* agg_ent;   // [agg_max][T]
    const double* T9;
    const double* rho;
    void* Y;
    double* dt;
    int* n_steps;
    int* status;
    void* Fplus;
    void* Fminus;
    double t_hydro, dt_fixed;
    double kappa, eps_y, y_floor, growth;
    int n_fixed, max_steps;
};


typedef void (*pull_fn)(const KPull);

template <typename real>
__host__ __device__ inline size_t pull_smem_bytes(int T, int W, int M) {
#ifndef KINNET_PAD_SMEM
#define KINNET_PAD_SMEM 0  // occupancy experiments: extra bytes that lower the CTAs per SM
#endif
    return 32 * sizeof(double) + sizeof(real) * (static_cast<size_t>(W) * 8 + 4 * T + 4) +
           sizeof(double) * static_cast<size_t>(M) + KINNET_PAD_SMEM;
}

// Kernel for a compiled pull schedule; one definition per (state type, adaptive/fixed)
// pair, each in its own translation unit (pull_inst.cu).
pull_fn pull_kernel_f64_adaptive(const PullSchedule& P);
pull_fn pull_kernel_f64_fixed(const PullSchedule& P);
pull_fn pull_kernel_f32_adaptive(const PullSchedule& P);
pull_fn pull_kernel_f32_fixed(const PullSchedule& P);

#ifdef KINNET_PULL_INSTANTIATE

__device__ __forceinline__ double rcp_pos(double b) {  // b normal, positive
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(b));
    // r0 is good to 2^-23 (PTX rcp.approx.ftz.f64); one third-order step leaves e^3 < 2^-69,
    // i.e. a result within an ulp or two -- far inside the 1e-9 parity bound, and three
    // dependent FMAs instead of five on the critical path of every sub-step
    double e = fma(-b, r, 1.0);
    e = fma(e, e, e);
    r = fma(r, e, r);
    return r;
}
__device__ __forceinline__ float rcp_pos(float b) { return __frcp_rn(b); }

template <typename real> struct Tiny;
template <> struct Tiny<double> { static __device__ __forceinline__ double v() { return 1e-290; } };
template <> struct Tiny<float> { static __device__ __forceinline__ float v() { return 1e-30f; } };

// Field extraction from the packed offset words.  volatile: the words are loop
// invariant, and without it the compiler hoists every unpacked field out of the
// sub-step loop into its own register (and then spills).
__device__ __forceinline__ uint32_t lo16(uint32_t x) {
    uint32_t r;
    asm volatile("and.b32 %0, %1, 0xffff;" : "=r"(r) : "r"(x));
    return r;
}
__device__ __forceinline__ uint32_t hi16(uint32_t x) {
    uint32_t r;
    asm volatile("shr.u32 %0, %1, 16;" : "=r"(r) : "r"(x));
    return r;
}
// Shared memory through 32-bit shared-window addresses.  With generic pointers the
// compiler rebuilds the window base (S2UR CgaCtaId, UMOV, ULEA) in front of every
// group of accesses and adds it to each gather offset; here the base is folded into
// the packed offsets once and an access is one LDS/STS on a register.
__device__ __forceinline__ void lds(double& v, uint32_t a) {
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a) : "memory");
}
__device__ __forceinline__ void lds(float& v, uint32_t a) {
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a) : "memory");
}
__device__ __forceinline__ void sts(uint32_t a, double v) {
    asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v) : "memory");
}
__device__ __forceinline__ void sts(uint32_t a, float v) {
    asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory");
}
template <typename real>
__device__ __forceinline__ real lds_at(uint32_t a) {
    real v;
    lds(v, a);
    return v;
}


// dt candidate of one species: eps max(y, floor) / |F+ - F-|   (reading Q7).
// Branch-free: the reciprocal is always formed, of 1 when the change is (near) zero.
template <typename real>
__device__ __forceinline__ double dt_candidate(real y, real a, real eps_y, real y_floor) {
    a = a < 0 ? -a : a;
    const bool moves = a > Tiny<real>::v();
    const real c = eps_y * (y > y_floor ? y : y_floor) * rcp_pos(moves ? a : static_cast<real>(1));
    return moves ? static_cast<double>(c) : static_cast<double>(INFINITY);
}

// Sum rows 0..5 of v over the warp (rows 0..2 = F+ shares of the hubs, 3..5 = F-
// shares).  On return the lanes 0, 8, 4, 16, 24, 20 hold the totals of rows
// 0, 1, 2, 3, 4, 5.  Fixed order: deterministic.  14 shuffles of 4-byte halves
// per 8-byte value instead of 60 for six plain butterflies.
template <typename real>
__device__ __forceinline__ real warp_sum_rows6(const real (&v)[6], int lane) {
    const bool up16 = lane & 16, up8 = lane & 8, up4 = lane & 4;
    real a[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const real send = up16 ? v[i] : v[i + 3];
        const real keep = up16 ? v[i + 3] : v[i];
        a[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
    real b0, b1;
    {
        const real send = up8 ? a[0] : a[1];
        const real keep = up8 ? a[1] : a[0];
        b0 = keep + __shfl_xor_sync(0xffffffffu, send, 8);
        b1 = a[2] + __shfl_xor_sync(0xffffffffu, a[2], 8);
    }
    real c;
    {
        const real send = up4 ? b0 : b1;
        const real keep = up4 ? b1 : b0;
        c = keep + __shfl_xor_sync(0xffffffffu, send, 4);
    }
    c += __shfl_xor_sync(0xffffffffu, c, 2);
    c += __shfl_xor_sync(0xffffffffu, c, 1);
    return c;
}

// Explicit asymptotic / forward Euler update of one species from F+ and k = F-/y
// (Eq. (3); y = 0 takes the Euler branch, reading Q8).
// Branch-free: both candidates are formed, 1 + k dt >= 1 is always a safe divisor.
template <typename real>
__device__ __forceinline__ real update_k(real y, real Fp, real k, real h, real kappa) {
    const real kh = k * h;
    const real ya = fma(h, Fp, y) * rcp_pos(static_cast<real>(1) + kh);
    const real ye = fma(h, Fp - k * y, y);
    return (y > 0 && kh >= kappa) ? ya : ye;
}

// Same update from F+ and F- (hub species): Eq. (3) as Y (Y + dt F+) / (Y + dt F-).
template <typename real>
__device__ __forceinline__ real update_fm(real y, real Fp, real Fm, real h, real kappa) {
    const real hFm = h * Fm;
    const bool pos = y > Tiny<real>::v();
    const real ya = fma(h, Fp, y) * (y * rcp_pos(pos ? y + hFm : static_cast<real>(1)));
    const real ye = fma(h, Fp - Fm, y);
    return (pos && hFm >= kappa * y) ? ya : ye;
}

template <typename real, int TB, int MINB, int CP, bool ADAPT>
__global__ void __launch_bounds__(TB, MINB) zone_kernel_pull(const KPull p) {
    static_assert(CP % 4 == 0 && CP <= kinnet::kPullMaxSlots, "slot capacity");
    constexpr int T = TB, NW = TB / 32;  // the schedule is built for exactly TB threads
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int N = p.N, M = p.M, nbs = p.nbs;
    const int z = blockIdx.x;

    double* redmin = reinterpret_cast<double*>(smem_raw);        // [32] per-warp dt minima
    real* red = reinterpret_cast<real*>(redmin + 32);            // [NW][8] per-warp hub-row sums
    real* YP = red + NW * 8;                                     // [4][T] published products, then 1
    double* Rbuf = reinterpret_cast<double*>(YP + 4 * T + 4);    // [M] rates, used during set-up only
    constexpr uint32_t SZ = sizeof(real);
    const uint32_t s_redmin = static_cast<uint32_t>(__cvta_generic_to_shared(smem_raw));
    const uint32_t s_red = s_redmin + 32 * 8;
    const uint32_t s_YP = s_red + NW * 8 * SZ;
    if (s_YP + (4 * T + 4) * SZ > 0xffffu) __trap();  // the packed gather addresses are 16-bit

    // ---- gather offsets -> registers -------------------------------------------
    uint32_t f1[CP / 2], f2[kJ2C / 2];
#pragma unroll
    for (int e = 0; e < CP / 2; ++e) f1[e] = p.f1_pack[e * T + tid] + s_YP * 0x10001u;
#pragma unroll
    for (int e = 0; e < kJ2C / 2; ++e) f2[e] = p.f2_pack[e * T + tid] + s_YP * 0x10001u;
    int wn, wn2;
    {
        const uint32_t cnt = p.cnt[tid];
        wn = __reduce_max_sync(0xffffffffu, cnt & 255u);  // warp-wide trip counts
        wn2 = __reduce_max_sync(0xffffffffu, (cnt >> 8) & 255u);
    }

    // ---- S1: rates, once per zone per call -----------
    {
        const double T9 = p.T9[z], rho = p.rho[z];
        const double t13 = cbrt(T9);
        const double t53 = T9 * t13 * t13;
        const double lnT = log(T9), lnrho = log(rho);
        for (int r = tid; r < M; r += T) {
            const double* c = p.coef + r;
            const double lnR = c[0] + c[1 * (size_t)M] / T9 + c[2 * (size_t)M] / t13 +
                               c[3 * (size_t)M] * t13 + c[4 * (size_t)M] * T9 +
                               c[5 * (size_t)M] * t53 + c[6 * (size_t)M] * lnT;
            Rbuf[r] = exp(c[7 * (size_t)M] * lnrho + lnR);
        }
    }
    if (tid < 4) YP[4 * T + tid] = static_cast<real>(1);
    __syncthreads();

    // rates of the P-slots and the rate sums of this thread, kept in registers
    real R[CP];
#pragma unroll
    for (int e = 0; e < CP; ++e) {
        const int32_t v = p.slot_rxn[e * T + tid];
        R[e] = v < 0 ? static_cast<real>(0)
                     : static_cast<real>(static_cast<double>(v >> 24) * Rbuf[v & 0xffffff]);
    }
    real C[kinnet::kPullCoefs];
    {
        int q = p.agg_ptr[tid];
#pragma unroll
        for (int s = 0; s < kinnet::kPullCoefs; ++s) {
            const int qe = p.agg_ptr[(s + 1) * T + tid];
            double acc = 0.0;
            for (; q < qe; ++q) {  // fixed (reaction) order
                const int32_t v = p.agg_ent[(size_t)q * T + tid];
                acc += static_cast<double>(v >> 24) * Rbuf[v & 0xffffff];
            }
            C[s] = static_cast<real>(acc);
        }
    }
    const real K0 = C[0], K1 = C[1], K2 = C[2], K3 = C[3], K00 = C[4], K01 = C[5], K02 = C[6],
               K11 = C[7], K12 = C[8], K22 = C[9];

    // ---- S6: zone state in ---------------------------------------------------------
    real* Yg = reinterpret_cast<real*>(p.Y) + (size_t)z * N;
    const int own = p.owner[tid];
    const bool hub_owner = tid < nbs;  // hub h is owned by thread h
    const bool plain_owner = own >= 0 && !hub_owner;
    real y = (own >= 0) ? Yg[own] : static_cast<real>(0);
    real yh0 = nbs > 0 ? Yg[p.hub[0]] : static_cast<real>(0);
    real yh1 = nbs > 1 ? Yg[p.hub[1]] : static_cast<real>(0);
    real yh2 = nbs > 2 ? Yg[p.hub[2]] : static_cast<real>(0);

    const real kappa = static_cast<real>(p.kappa);
    const real eps_y = static_cast<real>(p.eps_y);
    const real y_floor = static_cast<real>(p.y_floor);
    const double growth = p.growth, t_hydro = p.t_hydro;
    const bool rhs_only = p.mode == kRhs;

    double t = 0.0, dt_prev = 0.0;
    int steps = 0;
    int status = 0;
    bool run = true;
    if (ADAPT) {
        const double dt_in = p.dt ? p.dt[z] : 0.0;
        dt_prev = (dt_in > 0.0) ? dt_in : t_hydro;
        run = t_hydro > 0.0;
        if (!run) dt_prev = dt_in;  // nothing to do: the trial dt is returned unchanged
    } else if (!rhs_only) {
        run = p.n_fixed > 0;
    }
    const int max_steps = ADAPT ? p.max_steps : p.n_fixed;

    const uint32_t s_pub = s_YP + tid * SZ;
    while (run) {
        // ---- publish y x {1, hubs} ------------------------------------------------
        sts(s_pub, y);
        sts(s_pub + T * SZ, y * yh0);
        sts(s_pub + 2 * T * SZ, y * yh1);
        sts(s_pub + 3 * T * SZ, y * yh2);

        // ---- rate sums: k = F-/y (Eq. (1)) and this thread's share of the hub rows ---
        real k, share[6];
        {
            real e0 = fma(K00, yh0, K1);
            e0 = fma(K01, yh1, e0);
            e0 = fma(K02, yh2, e0);
            real e1 = fma(K11, yh1, K2);
            e1 = fma(K12, yh2, e1);
            const real e2 = fma(K22, yh2, K3);
            k = fma(yh0, e0, K0);
            k = fma(yh1, e1, k);
            k = fma(yh2, e2, k);
            // F-_hub share / y: Y_h dk/dY_h (each hub co-reactant occurrence counts once)
            real m0 = fma(K00, yh0, e0);
            real m1 = fma(K01, yh0, e1);
            m1 = fma(K11, yh1, m1);
            real m2 = fma(K02, yh0, e2);
            m2 = fma(K12, yh1, m2);
            m2 = fma(K22, yh2, m2);
            m0 *= yh0;
            m1 *= yh1;
            m2 *= yh2;
            if (tid == 0) m0 += k;  // the owner's own consumption in a hub-only reaction
            if (tid == 1) m1 += k;
            if (tid == 2) m2 += k;
            // F+_hub share / y
            real g0 = fma(C[13], yh1, C[10]);
            g0 = fma(C[14], yh2, g0);
            real g1 = fma(C[15], yh0, C[11]);
            g1 = fma(C[16], yh2, g1);
            real g2 = fma(C[17], yh0, C[12]);
            g2 = fma(C[18], yh1, g2);
            share[0] = y * g0;
            share[1] = y * g1;
            share[2] = y * g2;
            share[3] = y * m0;
            share[4] = y * m1;
            share[5] = y * m2;
        }
        __syncthreads();

        // ---- hub rows: warp totals of the six shares ---------------------------------------
        if (nbs > 0) {
            const real tot = warp_sum_rows6(share, lane);
            const int row = 3 * (lane >> 4) + ((lane & 4) ? 2 : ((lane >> 3) & 1));
            if ((lane & 3) == 0 && (lane & 12) != 12) sts(s_red + (warp * 8 + row) * SZ, tot);
        }

        // ---- S2+S3: F+ = sum of the incoming fluxes, each evaluated here -----------------
        real Fp;
        {
            real s0 = 0, s1 = 0, s2 = 0, s3 = 0;
#pragma unroll
            for (int g = 0; g < CP / 4; ++g) {
                if (4 * g < wn) {  // warp-uniform
                    const uint32_t w0 = f1[2 * g], w1 = f1[2 * g + 1];
                    real a0 = lds_at<real>(lo16(w0));
                    real a1 = lds_at<real>(hi16(w0));
                    real a2 = lds_at<real>(lo16(w1));
                    real a3 = lds_at<real>(hi16(w1));
                    if (4 * g < kJ2C) {
                        if (4 * g < wn2) {  // second factors (three-body reactions)
                            const uint32_t v0 = f2[(2 * g) % (kJ2C / 2)],
                                           v1 = f2[(2 * g + 1) % (kJ2C / 2)];
                            a0 *= lds_at<real>(lo16(v0));
                            a1 *= lds_at<real>(hi16(v0));
                            a2 *= lds_at<real>(lo16(v1));
                            a3 *= lds_at<real>(hi16(v1));
                        }
                    }
                    s0 = fma(R[4 * g], a0, s0);
                    s1 = fma(R[4 * g + 1], a1, s1);
                    s2 = fma(R[4 * g + 2], a2, s2);
                    s3 = fma(R[4 * g + 3], a3, s3);
                }
            }
            Fp = (s0 + s1) + (s2 + s3);
        }

        // ---- S5: dt candidates of the non-hub species ------------------------------------
        if (ADAPT) {
            double c = dt_candidate(y, Fp - k * y, eps_y, y_floor);
            if (!plain_owner) c = INFINITY;
            c = warp_min_pos(c);
            if (lane == 0) sts(s_redmin + warp * 8, c);
        }
        __syncthreads();

        // ---- finalize (every warp redundantly): hub rows over warps, zone-wide dt -----------
        real hFp = 0, hFm = 0;
        const real yme = lane == 0 ? yh0 : (lane == 1 ? yh1 : yh2);
        if (lane < nbs) {  // three active lanes: one wavefront per load instead of two
            real vp[NW], vm[NW];
#pragma unroll
            for (int w = 0; w < NW; ++w) {
                vp[w] = lds_at<real>(s_red + (w * 8 + lane) * SZ);
                vm[w] = lds_at<real>(s_red + (w * 8 + 3 + lane) * SZ);
            }
#pragma unroll
            for (int s = 1; s < NW; s *= 2)  // fixed pairwise order over warps (log depth)
#pragma unroll
                for (int w = 0; w + s < NW; w += 2 * s) {
                    vp[w] += vp[w + s];
                    vm[w] += vm[w + s];
                }
            hFp = vp[0];
            hFm = vm[0];
        }
        if (!ADAPT && rhs_only) {
            real* Fpo = reinterpret_cast<real*>(p.Fplus) + (size_t)z * N;
            real* Fmo = reinterpret_cast<real*>(p.Fminus) + (size_t)z * N;
            if (hub_owner) {
                Fpo[own] = hFp;
                Fmo[own] = hFm;
            } else if (own >= 0) {
                Fpo[own] = Fp;
                Fmo[own] = k * y;
            }
            return;
        }

        double dts;
        bool last;
        if (ADAPT) {
            double cand = INFINITY;
            if (lane >= 8 && lane < 8 + NW) cand = lds_at<double>(s_redmin + (lane - 8) * 8);
            const double hc = dt_candidate(yme, hFp - hFm, eps_y, y_floor);
            if (lane < nbs) cand = hc;
            const double cmin = warp_min_pos(cand);
            double dt_ctrl = growth * dt_prev;
            if (cmin < dt_ctrl) dt_ctrl = cmin;
            const double rem = t_hydro - t;
            last = dt_ctrl >= rem * (1.0 - 1e-12);
            dts = last ? rem : dt_ctrl;
            dt_prev = dt_ctrl;
        } else {
            dts = p.dt_fixed;
            last = (steps + 1 >= max_steps);
        }
        const real h = static_cast<real>(dts);

        // ---- S4: update (Eq. (3)) -------------------------------------------
        const real yn = update_k(y, Fp, k, h, kappa);
        if (nbs > 0) {  // hub species, on lanes 0..nbs-1 of every warp, from F+ and F-
            const real hn = update_fm(yme, hFp, hFm, h, kappa);
            yh0 = __shfl_sync(0xffffffffu, hn, 0);
            if (nbs > 1) yh1 = __shfl_sync(0xffffffffu, hn, 1);
            if (nbs > 2) yh2 = __shfl_sync(0xffffffffu, hn, 2);
        }
        y = hub_owner ? (tid == 0 ? yh0 : (tid == 1 ? yh1 : yh2)) : yn;
        t = last ? t_hydro : t + dts;
        ++steps;
        if (last) run = false;
        else if (ADAPT && steps >= max_steps) {
            status |= NET_STATUS_MAX_STEPS;
            run = false;
        }
    }

    // ---- S6: zone state out ------------------------------------------------------------------
    const int bad = (own >= 0) && !isfinite(static_cast<double>(y));
    if (__syncthreads_or(bad)) status |= NET_STATUS_NONFINITE;
    if (own >= 0) Yg[own] = y;
    if (tid == 0) {
        if (ADAPT && p.dt) p.dt[z] = dt_prev;
        if (p.n_steps) p.n_steps[z] = steps;
        if (p.status) p.status[z] = status;
    }
}

// pull kernel: block-size classes with the residency the register file allows
// (65536 / (TB * MINB) registers per thread) x P-slot capacity classes

template <typename real, int CP, bool ADAPT>
pull_fn pick_pull_block(int T) {
    switch (T) {
        case 32: return zone_kernel_pull<real, 32, 12, CP, ADAPT>;
        case 64: return zone_kernel_pull<real, 64, 6, CP, ADAPT>;
        case 160: return zone_kernel_pull<real, 160, KINNET_MINB160, CP, ADAPT>;
        case 256: return zone_kernel_pull<real, 256, 2, CP, ADAPT>;
        case 384: return zone_kernel_pull<real, 384, 1, CP, ADAPT>;
        default: return zone_kernel_pull<real, 512, 1, CP, ADAPT>;
    }
}

template <typename real, bool ADAPT>
pull_fn pick_pull_real(const kinnet::PullSchedule& P) {
    if (P.slots <= 12) return pick_pull_block<real, 12, ADAPT>(P.T);
    if (P.slots <= 20) return pick_pull_block<real, 20, ADAPT>(P.T);
    return pick_pull_block<real, 24, ADAPT>(P.T);
}

#endif  // KINNET_PULL_INSTANTIATE

}  // namespace kinnet
