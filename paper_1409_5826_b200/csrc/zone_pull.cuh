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
// Pull kernel, one species per thread (zone_pull2.cuh is its two-species form; see
// schedule.h "Pull schedule" and DESIGN.md 4.2-4.3): no flux array, two barriers per
// sub-step, the dt controller carried as q = 1/dt.
//
//   publish   YP[c][t] = y * {1, Y_hub0, Y_hub1, Y_hub2}[c]            4 STS
//   rate sums k = F-/y and the six hub-row shares from the per-thread
//             coefficients K, G0, Gx (sums of rates formed once per call);
//             inv = 1 / (eps max(y, floor)) for the dt candidate
//   ------------------------------------------------------------------- barrier A
//   P-slots   F+ = sum_e R[e] * YP[f1[e]] (* YP[f2[e]])   fluxes at the consumer,
//   hub rows  interleaved with the transposed warp butterfly of the six shares
//             -> red[warp][row]
//   dt        candidate |F+ - k y| * inv, warp max -> redmin[warp]
//   ------------------------------------------------------------------- barrier B
//   finalize  every warp redundantly: lanes 0..2 sum the hub rows over warps,
//             zone-wide q = max(candidates, q_prev / g), end clamp, hub update,
//             shuffle-broadcast of the new hub Y
//   update    k dt >= kappa ? (y q + F+)/(q + k) : y + dt (F+ - k y)
// Rates, rate sums and every gather address of a thread stay in registers for
// the whole hydro step (topology is static, sub-steps number 1e2..1e4).
// ---------------------------------------------------------------------------
constexpr int kJ2C = kinnet::kPullMaxSlots2;
// P-slot rates beyond the first CP - kPullSpillSlots of a thread live in shared memory:
// only the warp with the longest rows reaches them (the species are dealt to threads by
// falling in-degree), and every thread gets the registers back.  Measured on configs[3]
// (zone-networks/s): 0 -> 161.7k, 4 -> 172.7k, 8 -> 165.0k, 12 -> 171.2k, 16 -> 173.1k.
constexpr int kPullSpillSlots = 4;
// (the 160-thread instantiation is compiled for 3 resident CTAs per SM, 4 with fp32 state:
// register budget 65536 / (160 * MINB); 4 with fp64 state spills: 152.6k against 172.5k)

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
    const int* order;         // [zones] launch order (zone of CTA b), NULL = identity
    void* Y;
    double* dt;
    int* n_steps;
    int* status;
    const double* bind;       // [N] binding energies, NULL unless energy is asked for
    double* energy;           // [zones] out: sum_i bind_i (Y_i - Y_i(0)), or NULL
    void* Fplus;
    void* Fminus;
    double t_hydro, dt_fixed;
    double kappa, eps_y, y_floor, growth;
    int n_fixed, max_steps;
    int method;               // 0 = asymptotic / Euler, 1 = QSS variant (net_params_t.method)
    int stair;                // two-species kernel: the schedule fits the staircase of live slots (zone_pull2.cuh)
};


typedef void (*pull_fn)(const KPull);

template <typename real>
__host__ __device__ inline size_t pull_smem_bytes(int T, int W, int M) {
    return 32 * sizeof(double) +
           sizeof(real) * (static_cast<size_t>(W) * 8 + 4 * T + 4 + kPullSpillSlots * T) +
           sizeof(double) * static_cast<size_t>(M);
}

// Kernel for a compiled pull schedule; one definition per (state type, adaptive/fixed)
// pair, each in its own translation unit (pull_inst.cu).
pull_fn pull_kernel_f64_adaptive(const PullSchedule& P, int method);
pull_fn pull_kernel_f64_fixed(const PullSchedule& P, int method);
pull_fn pull_kernel_f32_adaptive(const PullSchedule& P, int method);
pull_fn pull_kernel_f32_fixed(const PullSchedule& P, int method);

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
// the same under a predicate (0 where it is false): a predicated LDS, no branch
template <typename real>
__device__ __forceinline__ real lds_if(bool on, uint32_t a);
template <>
__device__ __forceinline__ double lds_if<double>(bool on, uint32_t a) {
    double v = 0.0;
    asm volatile("{ .reg .pred q; setp.ne.u32 q, %2, 0; @q ld.shared.f64 %0, [%1]; }"
                 : "+d"(v) : "r"(a), "r"(static_cast<uint32_t>(on)) : "memory");
    return v;
}
template <>
__device__ __forceinline__ float lds_if<float>(bool on, uint32_t a) {
    float v = 0.0f;
    asm volatile("{ .reg .pred q; setp.ne.u32 q, %2, 0; @q ld.shared.f32 %0, [%1]; }"
                 : "+f"(v) : "r"(a), "r"(static_cast<uint32_t>(on)) : "memory");
    return v;
}


// QSS variant (reading Q20): alpha(a) k with a = k dt, the weight of
// the loss term in  y' = y + dt (F+ - k y)/(1 + alpha a) = y + (F+ - k y)/(q + alpha k),  q = 1/dt.
template <typename real>
__device__ __forceinline__ real qss_alpha_k(real k, real h) {
    const real a = k * h;
    const real num = fma(fma(a + static_cast<real>(11), a, static_cast<real>(60)), a, static_cast<real>(180));
    const real den = fma(fma(a + static_cast<real>(12), a, static_cast<real>(60)), a, static_cast<real>(360));
    return num * rcp_pos(den) * k;
}

// |a| as an operand modifier of the multiply that follows (a select costs four instructions in fp64)
__device__ __forceinline__ double abs_of(double a) { return fabs(a); }
__device__ __forceinline__ float abs_of(float a) { return fabsf(a); }

template <typename real, int TB, int MINB, int CP, int J2, bool ADAPT, bool QSS>
__global__ void __launch_bounds__(TB, MINB) zone_kernel_pull(const KPull p) {
    static_assert(CP % 4 == 0 && CP <= kinnet::kPullMaxSlots, "slot capacity");
    static_assert(J2 % 4 == 0 && J2 <= kJ2C, "second-factor slot capacity");
    constexpr int CPR = CP > 12 ? CP - kPullSpillSlots : CP;  // slots whose rate stays in a register
    constexpr int T = TB, NW = TB / 32;  // the schedule is built for exactly TB threads
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int N = p.N, M = p.M, nbs = p.nbs;
    const int z = p.order ? p.order[blockIdx.x] : blockIdx.x;

    double* redmin = reinterpret_cast<double*>(smem_raw);        // [32] per-warp dt minima
    real* red = reinterpret_cast<real*>(redmin + 32);            // [NW][8] per-warp hub-row sums
    real* YP = red + NW * 8;                                     // [4][T] published products, then 1
    real* Rx = YP + 4 * T + 4;                                   // [kPullSpillSlots][T] spilled slot rates
    double* Rbuf = reinterpret_cast<double*>(Rx + kPullSpillSlots * T);  // [M] rates, set-up only
    constexpr uint32_t SZ = sizeof(real);
    // opaque to the compiler: otherwise it rebuilds the window base (S2UR CgaCtaId + ULEA,
    // ~30 exposed cycles) in front of every group of accesses instead of keeping a register
    uint32_t s_redmin;
    asm volatile("mov.u32 %0, %1;"
                 : "=r"(s_redmin)
                 : "r"(static_cast<uint32_t>(__cvta_generic_to_shared(smem_raw))));
    const uint32_t s_red = s_redmin + 32 * 8;
    const uint32_t s_YP = s_red + NW * 8 * SZ;
    const uint32_t s_Rx = s_YP + (4 * T + 4) * SZ + tid * SZ;
    if (s_YP + (4 * T + 4) * SZ > 0xffffu) __trap();  // the packed gather addresses are 16-bit

    // ---- gather offsets -> registers -------------------------------------------
    uint32_t f1[CP / 2], f2[J2 / 2];
#pragma unroll
    for (int e = 0; e < CP / 2; ++e) f1[e] = p.f1_pack[e * T + tid] + s_YP * 0x10001u;
#pragma unroll
    for (int e = 0; e < J2 / 2; ++e) f2[e] = p.f2_pack[e * T + tid] + s_YP * 0x10001u;
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
    real R[CPR];
#pragma unroll
    for (int e = 0; e < CP; ++e) {
        const int32_t v = p.slot_rxn[e * T + tid];
        const real r = v < 0 ? static_cast<real>(0)
                             : static_cast<real>(static_cast<double>(v >> 24) * Rbuf[v & 0xffffff]);
        if (e < CPR) R[e] = r;
        else Rx[(e - CPR) * T + tid] = r;
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
    constexpr bool qss = QSS;  // net_params_t.method = 1, an instantiation (see zone_pull2.cuh)

    // The controller runs on q = 1/dt: the candidates become
    // |F+ - F-| / (eps max(y, floor)), their reciprocal factor is formed while the
    // gathers are in flight, the zone-wide reduction is a maximum, and Eq. (3) reads
    // (y q + F+) / (q + k), so no reciprocal sits between the reduction and the update
    // chain except the ones that run side by side.
    double t = 0.0, q_prev = 0.0, dt_out = 0.0;
    int steps = 0;
    int status = 0;
    bool run = true;
    if (ADAPT) {
        const double dt_in = p.dt ? p.dt[z] : 0.0;
        run = t_hydro > 0.0;
        dt_out = dt_in;  // nothing to do: the trial dt is returned unchanged
        if (run) q_prev = 1.0 / ((dt_in > 0.0) ? dt_in : t_hydro);
    } else if (!rhs_only) {
        run = p.n_fixed > 0;
    }
    const int max_steps = ADAPT ? p.max_steps : p.n_fixed;
    const double ginv = 1.0 / growth;
    const double q_fixed = ADAPT ? 0.0 : 1.0 / p.dt_fixed;
    const real kappa_ = kappa;
    const uint32_t s_pub = s_YP + tid * SZ;
    const uint32_t s_own = s_redmin + 16 * 8;  // [3] own-consumption terms of the hub owners
    const real yfl_eps = eps_y * y_floor;

    while (run) {
        // ---- publish y x {1, hubs} ------------------------------------------------
        const real p1 = y * yh0, p2 = y * yh1, p3 = y * yh2;
        sts(s_pub, y);
        sts(s_pub + T * SZ, p1);
        sts(s_pub + 2 * T * SZ, p2);
        sts(s_pub + 3 * T * SZ, p3);

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
            // F-_hub share / (y Y_h): dk/dY_h (each hub co-reactant occurrence counts once)
            const real m0 = fma(K00, yh0, e0);
            real m1 = fma(K01, yh0, e1);
            m1 = fma(K11, yh1, m1);
            real m2 = fma(K02, yh0, e2);
            m2 = fma(K12, yh1, m2);
            m2 = fma(K22, yh2, m2);
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
            share[3] = p1 * m0;
            share[4] = p2 * m1;
            share[5] = p3 * m2;
        }
        // reciprocal factors of the dt candidates, off the critical path
        real inv = 0;
        if (ADAPT) {
            inv = rcp_pos(y > y_floor ? eps_y * y : yfl_eps);
            if (!plain_owner) inv = 0;  // hub owners are judged on their full rows in finalize
        }
        __syncthreads();
        // the owner's own consumption in a hub-only reaction joins its F- row in finalize.  Stored
        // between the barriers: B orders it before this step's reads, the next A orders those
        // reads before the next store.
        if (hub_owner) sts(s_own + tid * SZ, k * y);

        // ---- S2+S3 interleaved with the hub-row butterfly -------------------------------------
        // F+ = sum of the incoming fluxes, each evaluated here (groups of four P-slots), and
        // the six hub-row shares summed over the warp (rows 0..2 = F+, 3..5 = F-; the lanes
        // 0, 8, 4, 16, 24, 20 end up with the totals of rows 0, 1, 2, 3, 4, 5; 14 shuffles
        // of 4-byte halves per 8-byte value instead of 60 for six plain butterflies).  The two
        // are independent latency chains (SHFL and LDS), so one stage of each alternates.
        real Fp;
        {
            real s0, s1, s2, s3;  // group 0 always runs (wn >= 4: holes carry rate 0)
            real a0, a1, a2, a3;
#define KINNET_LOADS(g)                                                                 \
    if ((g) == 0 || (4 * (g) < CP && 4 * (g) < wn)) {                                   \
        const uint32_t w0 = f1[(2 * (g)) % (CP / 2)], w1 = f1[(2 * (g) + 1) % (CP / 2)]; \
        a0 = lds_at<real>(lo16(w0));                                                    \
        a1 = lds_at<real>(hi16(w0));                                                    \
        a2 = lds_at<real>(lo16(w1));                                                    \
        a3 = lds_at<real>(hi16(w1));                                                    \
        if (4 * (g) < J2 && 4 * (g) < wn2) { /* second factors (three-body reactions) */ \
            const uint32_t v0 = f2[(2 * (g)) % (J2 / 2)], v1 = f2[(2 * (g) + 1) % (J2 / 2)]; \
            a0 *= lds_at<real>(lo16(v0));                                               \
            a1 *= lds_at<real>(hi16(v0));                                               \
            a2 *= lds_at<real>(lo16(v1));                                               \
            a3 *= lds_at<real>(hi16(v1));                                               \
        }                                                                               \
    }
// byte offset of spilled slot e (dead branches of the unrolled groups clamp to 0)
#define KINNET_XOFF(e) (static_cast<uint32_t>((e) >= CPR ? (e) - CPR : 0) * T * SZ)
#define KINNET_FMAS(g)                                                          \
    if ((g) == 0) {                                                             \
        s0 = R[0] * a0;                                                         \
        s1 = R[1] * a1;                                                         \
        s2 = R[2] * a2;                                                         \
        s3 = R[3] * a3;                                                         \
    } else if (4 * (g) < CPR && 4 * (g) < wn) {                                        \
        s0 = fma(R[(4 * (g)) % CPR], a0, s0);                                   \
        s1 = fma(R[(4 * (g) + 1) % CPR], a1, s1);                               \
        s2 = fma(R[(4 * (g) + 2) % CPR], a2, s2);                               \
        s3 = fma(R[(4 * (g) + 3) % CPR], a3, s3);                               \
    } else if (4 * (g) < CP && 4 * (g) < wn) {                                  \
        s0 = fma(lds_at<real>(s_Rx + KINNET_XOFF(4 * (g))), a0, s0);        \
        s1 = fma(lds_at<real>(s_Rx + KINNET_XOFF(4 * (g) + 1)), a1, s1);    \
        s2 = fma(lds_at<real>(s_Rx + KINNET_XOFF(4 * (g) + 2)), a2, s2);    \
        s3 = fma(lds_at<real>(s_Rx + KINNET_XOFF(4 * (g) + 3)), a3, s3);    \
    }
            const bool up16 = lane & 16, up8 = lane & 8, up4 = lane & 4;
            // level 16
            real r0 = __shfl_xor_sync(0xffffffffu, up16 ? share[0] : share[3], 16);
            real r1 = __shfl_xor_sync(0xffffffffu, up16 ? share[1] : share[4], 16);
            real r2 = __shfl_xor_sync(0xffffffffu, up16 ? share[2] : share[5], 16);
            KINNET_LOADS(0)
            const real b0_ = (up16 ? share[3] : share[0]) + r0;
            const real b1_ = (up16 ? share[4] : share[1]) + r1;
            const real b2_ = (up16 ? share[5] : share[2]) + r2;
            // level 8
            r0 = __shfl_xor_sync(0xffffffffu, up8 ? b0_ : b1_, 8);
            r1 = __shfl_xor_sync(0xffffffffu, b2_, 8);
            KINNET_FMAS(0)
            KINNET_LOADS(1)
            const real c0_ = (up8 ? b1_ : b0_) + r0;
            const real c1_ = b2_ + r1;
            // level 4
            r0 = __shfl_xor_sync(0xffffffffu, up4 ? c0_ : c1_, 4);
            KINNET_FMAS(1)
            KINNET_LOADS(2)
            real tot = (up4 ? c1_ : c0_) + r0;
            r0 = __shfl_xor_sync(0xffffffffu, tot, 2);
            KINNET_FMAS(2)
            KINNET_LOADS(3)
            tot += r0;
            r0 = __shfl_xor_sync(0xffffffffu, tot, 1);
            KINNET_FMAS(3)
            KINNET_LOADS(4)
            tot += r0;
            KINNET_FMAS(4)
            KINNET_LOADS(5)
            KINNET_FMAS(5)
#undef KINNET_LOADS
#undef KINNET_FMAS
#undef KINNET_XOFF
            const int row = 3 * (lane >> 4) + ((lane & 4) ? 2 : ((lane >> 3) & 1));
            if ((lane & 3) == 0 && (lane & 12) != 12) sts(s_red + (warp * 8 + row) * SZ, tot);
            Fp = (s0 + s1) + (s2 + s3);
        }

        // ---- S5: q candidates of the non-hub species: |F+ - F-| / (eps max(y, floor)) ------
        const real change = fma(-k, y, Fp);
        if (ADAPT) {
            const double c = warp_max_pos(static_cast<double>(fabs(change) * inv));
            if (lane == 0) sts(s_redmin + warp * 8, c);
        }
        __syncthreads();

        // ---- finalize (every warp redundantly): hub rows over warps, zone-wide dt -----------
        // (the reciprocals below depend on nothing the barrier waited for: they run beside
        // the loads and the sums over warps)
        const real yme = lane == 0 ? yh0 : (lane == 1 ? yh1 : yh2);
        real invh = 0;
        double q_rem = 0.0, rem = 0.0;
        if (ADAPT) {
            invh = rcp_pos(yme > y_floor ? eps_y * yme : yfl_eps);
            rem = t_hydro - t;
            q_rem = rcp_pos(rem);
        }
        real hFp = 0, hFm = 0;
        if (lane < nbs) {  // three active lanes: one wavefront per load instead of two
            real vp[NW], vm[NW];
#pragma unroll
            for (int w = 0; w < NW; ++w) {
                vp[w] = lds_at<real>(s_red + (w * 8 + lane) * SZ);
                vm[w] = lds_at<real>(s_red + (w * 8 + 3 + lane) * SZ);
            }
            const real own_term = lds_at<real>(s_own + lane * SZ);
#pragma unroll
            for (int s = 1; s < NW; s *= 2)  // fixed pairwise order over warps (log depth)
#pragma unroll
                for (int w = 0; w + s < NW; w += 2 * s) {
                    vp[w] += vp[w + s];
                    vm[w] += vm[w + s];
                }
            hFp = vp[0];
            hFm = vm[0] + own_term;
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

        double q, hd;
        bool last;
        if (ADAPT) {
            double cand = 0.0;
            if (lane >= 8 && lane < 8 + NW) cand = lds_at<double>(s_redmin + (lane - 8) * 8);
            const double qh = static_cast<double>(abs_of(hFp - hFm) * invh);
            if (lane < nbs) cand = qh;
            const double qmax = warp_max_pos(cand);
            const double qg = q_prev * ginv;             // growth cap: dt <= g dt_prev
            const double q_ctrl = (qmax > qg) ? qmax : qg;  // a NaN candidate loses
            // dt_ctrl >= rem (1 - 1e-12); written so that rem <= 0 (t rounded onto t_hydro:
            // q_rem is then NaN or negative) also ends the call, with a zero-length step
            last = !(q_ctrl > q_rem * (1.0 / (1.0 - 1e-12))) || !(rem > 0.0);
            q = last ? q_rem : q_ctrl;
            hd = last ? rem : rcp_pos(q_ctrl);
            q_prev = q_ctrl;
        } else {
            q = q_fixed;
            hd = p.dt_fixed;
            last = (steps + 1 >= max_steps);
        }
        const real h = static_cast<real>(hd), qr = static_cast<real>(q);

        // ---- S4: update (Eq. (3)) -------------------------------------------
        // Eq. (3) times q/q: (y + dt F+) / (1 + k dt) = (y q + F+) / (q + k); y = 0 takes the
        // Euler branch (reading Q8).  Branch-free: both candidates are formed.
        real yn;
        {
            const real ya = fma(y, qr, Fp) * rcp_pos(qr + k);
            const real ye = fma(h, change, y);
            yn = (y > 0 && k * h >= kappa_) ? ya : ye;
            if (qss) yn = fma(change, rcp_pos(qr + qss_alpha_k(y > 0 ? k : static_cast<real>(0), h)), y);  // uniform
        }
        {  // hub species, on lanes 0..nbs-1 of every warp: Y (Y q + F+) / (Y q + F-)
            const bool pos = yme > Tiny<real>::v();
            const real den = fma(yme, qr, hFm);
            const real ya = fma(yme, qr, hFp) * (yme * rcp_pos(pos ? den : static_cast<real>(1)));
            const real ye = fma(h, hFp - hFm, yme);
            real hn = (pos && h * hFm >= kappa_ * yme) ? ya : ye;
            if (qss) {
                const real kh = pos ? hFm * rcp_pos(pos ? yme : static_cast<real>(1)) : static_cast<real>(0);
                hn = fma(hFp - hFm, rcp_pos(qr + qss_alpha_k(kh, h)), yme);
            }
            if (lane >= nbs) hn = 0;  // a missing hub reads as abundance 0
            yh0 = __shfl_sync(0xffffffffu, hn, 0);  // unconditional: the three go out back to back
            yh1 = __shfl_sync(0xffffffffu, hn, 1);
            yh2 = __shfl_sync(0xffffffffu, hn, 2);
            y = hub_owner ? hn : yn;  // hub h lives on thread h: warp 0, lane h
        }
        t = last ? t_hydro : t + hd;
        ++steps;
        if (last) run = false;
        else if (ADAPT && steps >= max_steps) {
            status |= NET_STATUS_MAX_STEPS;
            run = false;
        }
    }
    if (ADAPT && steps > 0) dt_out = 1.0 / q_prev;

    // ---- S6: zone state out ------------------------------------------------------------------
    const int bad = (own >= 0) && !isfinite(static_cast<double>(y));
    if (__syncthreads_or(bad)) status |= NET_STATUS_NONFINITE;
    if (p.energy) {  // uniform; Yg still holds the start-of-call abundances
        const double e = (own >= 0) ? p.bind[own] * (static_cast<double>(y) - static_cast<double>(Yg[own])) : 0.0;
        zone_energy_out(e, redmin, p.energy + z);
    }
    if (own >= 0) Yg[own] = y;
    if (tid == 0) {
        if (ADAPT && p.dt) p.dt[z] = dt_out;
        if (p.n_steps) p.n_steps[z] = steps;
        if (p.status) p.status[z] = status;
    }
}

// pull kernel: block-size classes with the residency the register file allows
// (65536 / (TB * MINB) registers per thread) x P-slot capacity classes

template <typename real, int CP, int J2, bool ADAPT, bool QSS>
pull_fn pick_pull_block(int T) {
    switch (T) {
        case 32: return zone_kernel_pull<real, 32, 12, CP, J2, ADAPT, QSS>;
        case 64: return zone_kernel_pull<real, 64, 6, CP, J2, ADAPT, QSS>;
        case 160: return zone_kernel_pull<real, 160, sizeof(real) == 8 ? 3 : 4, CP, J2, ADAPT, QSS>;  // fp32 state halves the rate registers
        case 256: return zone_kernel_pull<real, 256, 2, CP, J2, ADAPT, QSS>;
        case 384: return zone_kernel_pull<real, 384, 1, CP, J2, ADAPT, QSS>;
        default: return zone_kernel_pull<real, 512, 1, CP, J2, ADAPT, QSS>;
    }
}

template <typename real, int J2, bool ADAPT, bool QSS>
pull_fn pick_pull_slots(const kinnet::PullSchedule& P) {
    if (P.slots <= 12) return pick_pull_block<real, 12, J2, ADAPT, QSS>(P.T);
    if (P.slots <= 20) return pick_pull_block<real, 20, J2, ADAPT, QSS>(P.T);
    return pick_pull_block<real, 24, J2, ADAPT, QSS>(P.T);
}

// P-slot capacity classes x second-factor capacity classes (the packed offsets of
// the unused capacity would only hold registers); the QSS variant is instantiated for the
// larger second-factor class only
template <typename real, bool ADAPT>
pull_fn pick_pull_real(const kinnet::PullSchedule& P, int method = 0) {
    if (method == 1) return pick_pull_slots<real, 8, ADAPT, true>(P);
    if (P.slots2 <= 4) return pick_pull_slots<real, 4, ADAPT, false>(P);
    return pick_pull_slots<real, 8, ADAPT, false>(P);
}

#endif  // KINNET_PULL_INSTANTIATE

}  // namespace kinnet
