// kinnet.cu -- sm_100a kernels and the C ABI of include/kinnet.h.
//
// One CTA integrates one zone over the whole hydro step (PAPER.md L104-110,
// Fig. 3: rates once, then the sub-step loop entirely on the GPU); the whole
// batch of zones is ONE launch instead of the paper's one asynchronous launch
// per network from OpenMP threads.
//
// Sub-step (Eq. (1), Eq. (3)), three barriers:
//   flux     f[j*T+t] = R * Y[a] * Y[b] * Y[c]        every thread, rs slots
//   ---------------------------------------------------------------- barrier
//   sums     small rows: the owner thread gathers F+_i, F-_i from f
//            big rows:   own-column readback + warp butterfly -> red[warp][row]
//   dt       candidate eps*max(Y,floor)/|F+ - F-| , warp min -> redmin[warp]
//   ---------------------------------------------------------------- barrier
//   finalize every warp redundantly: min over warps and big species -> dt
//   update   k dt >= kappa ? (Y + dt F+)/(1 + k dt) : Y + dt (F+ - F-)
//   ---------------------------------------------------------------- barrier
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>

#include "../../include/kinnet.h"
#include "schedule.h"

namespace {

using kinnet::Schedule;

thread_local std::string g_last_error;

int fail(int code, const std::string& msg) {
    g_last_error = msg;
    return code;
}

#define CUDA_TRY(expr)                                                                      \
    do {                                                                                    \
        cudaError_t e_ = (expr);                                                            \
        if (e_ != cudaSuccess)                                                              \
            return fail(NET_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(e_));     \
    } while (0)

constexpr int kMaxBig = kinnet::kMaxBigSpecies;
constexpr int kRedStride = 2 * kMaxBig;

enum Mode { kAdaptive = 0, kFixed = 1, kRhs = 2, kRates = 3 };

struct KParams {
    // schedule
    int N, M, T, W, rs, j2, j3, nbs;
    int big_species[kMaxBig];
    const int32_t* flux_rxn;
    const ushort4* flux_react;
    const double* coef;
    const int32_t* owner;
    const uint16_t* small_plus;
    const uint16_t* small_minus;
    const uint16_t* small_src;
    const uint8_t* big_cnt;
    const uint8_t* big_slot;
    // packed tables of the register-resident kernel
    const uint32_t* fx_pack;
    const uint32_t* fxc_pack;
    const uint32_t* plus_pack;
    const uint32_t* minus_pack;
    const uint32_t* rb_pack;
    const uint32_t* cnt_pack;
    const uint32_t* rbcnt_pack;
    // zones
    const double* T9;
    const double* rho;
    void* Y;
    double* dt;
    int* n_steps;
    int* status;
    void* Fplus;
    void* Fminus;
    double* Rout;
    double t_hydro, dt_fixed;
    long long n_fixed;
    // integrator parameters
    double kappa, eps_y, y_floor, growth;
    long long max_steps;
};

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

__host__ __device__ inline int real_words_before_flux(int N) { return (N + 1 + 3) & ~3; }

template <typename real>
size_t smem_bytes(const Schedule& S) {
    return 64 * sizeof(double) +
           sizeof(real) * (static_cast<size_t>(real_words_before_flux(S.N)) +
                           2 * static_cast<size_t>(S.rs) * S.T +
                           static_cast<size_t>(S.W) * kRedStride);
}

template <typename real, int MODE, int TB>
__global__ void __launch_bounds__(TB) zone_kernel(const KParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int T = p.T, N = p.N, W = p.W, rs = p.rs, slots = rs * T, nbs = p.nbs;
    const int z = blockIdx.x;

    double* redmin = reinterpret_cast<double*>(smem_raw);            // [32] per-warp dt minima
    double* ybig = redmin + 32;                                      // [kMaxBig] start-of-step Y of big species
    real* Ybuf = reinterpret_cast<real*>(redmin + 64);               // [N] + constant one
    real* Rbuf = Ybuf + real_words_before_flux(N);                   // [rs*T]
    real* fbuf = Rbuf + slots;                                       // [rs*T]
    real* red = fbuf + slots;                                        // [W][kRedStride]

    // ---- S1: rates, once per zone per call -----
    {
        const double T9 = p.T9[z], rho = p.rho[z];
        const double t13 = cbrt(T9);
        const double t53 = T9 * t13 * t13;
        const double lnT = log(T9), lnrho = log(rho);
        for (int j = 0; j < rs; ++j) {
            const int idx = j * T + tid;
            const double* c = p.coef + idx;
            const double lnR = c[0] + c[1 * (size_t)slots] / T9 + c[2 * (size_t)slots] / t13 +
                               c[3 * (size_t)slots] * t13 + c[4 * (size_t)slots] * T9 +
                               c[5 * (size_t)slots] * t53 + c[6 * (size_t)slots] * lnT;
            const double R = exp(c[7 * (size_t)slots] * lnrho + lnR);
            if (MODE == kRates) {
                const int r = p.flux_rxn[idx];
                if (r >= 0) p.Rout[(size_t)z * p.M + r] = R;
            } else {
                Rbuf[idx] = static_cast<real>(R);
            }
        }
        if (MODE == kRates) return;
    }

    // ---- S6: zone state in ----------------------------------------------
    real* Yg = reinterpret_cast<real*>(p.Y) + (size_t)z * N;
    for (int i = tid; i < N; i += T) Ybuf[i] = Yg[i];
    if (tid == 0) Ybuf[N] = static_cast<real>(1);
    const int own = p.owner[tid];
    const int np = p.small_plus[tid], nm = p.small_minus[tid];
    const bool is_big = (tid >= W && tid < W + nbs);
    unsigned bigcnt[2 * kMaxBig];
#pragma unroll
    for (int b = 0; b < 2 * kMaxBig; ++b)
        bigcnt[b] = (b < 2 * nbs) ? p.big_cnt[(size_t)b * T + tid] : 0u;
    __syncthreads();
    real y = (own >= 0) ? Ybuf[own] : static_cast<real>(0);

    const real kappa = static_cast<real>(p.kappa);
    const real eps_y = static_cast<real>(p.eps_y);
    const real y_floor = static_cast<real>(p.y_floor);

    double t = 0.0, dt_prev = 0.0;
    long long steps = 0;
    int status = 0;
    bool run = true;
    if (MODE == kAdaptive) {
        const double dt_in = p.dt ? p.dt[z] : 0.0;
        dt_prev = (dt_in > 0.0) ? dt_in : p.t_hydro;
        run = p.t_hydro > 0.0;
        if (!run) dt_prev = dt_in;  // nothing to do: the trial dt is returned unchanged
    } else if (MODE == kFixed) {
        run = p.n_fixed > 0;
    }

    while (run) {
        // ---- S2: fluxes ------------------------------------
        for (int j = 0; j < rs; ++j) {
            const int idx = j * T + tid;
            const ushort4 re = __ldg(p.flux_react + idx);
            real v = Rbuf[idx] * Ybuf[re.x];
            if (j < p.j2) v = v * Ybuf[re.y];
            if (j < p.j3) v = v * Ybuf[re.z];
            fbuf[idx] = v;
        }
        __syncthreads();

        // ---- S3: sums F+_i, F-_i (Eq. (1)) --------
        real Fp = 0, Fm = 0;
        {
            int e = 0;
            for (; e < np; ++e) Fp += fbuf[__ldg(p.small_src + (size_t)e * T + tid)];
            for (; e < np + nm; ++e) Fm += fbuf[__ldg(p.small_src + (size_t)e * T + tid)];
        }
        if (nbs > 0) {
            int e = 0;
#pragma unroll
            for (int b = 0; b < 2 * kMaxBig; ++b) {
                if (b < 2 * nbs) {
                    real acc = 0;
                    for (unsigned q = 0; q < bigcnt[b]; ++q, ++e)
                        acc += fbuf[(int)__ldg(p.big_slot + (size_t)e * T + tid) * T + tid];
                    acc = warp_sum(acc);
                    if (lane == 0) red[warp * kRedStride + b] = acc;
                }
            }
        }
        // ---- S5: dt candidates of the small species ------------------------
        if (MODE == kAdaptive) {
            double c = INFINITY;
            if (own >= 0 && !is_big) {
                real a = Fp - Fm;
                a = a < 0 ? -a : a;
                if (a > 0) c = static_cast<double>(eps_y * (y > y_floor ? y : y_floor) / a);
            }
            c = warp_min_pos(c);
            if (lane == 0) redmin[warp] = c;
            // Ybuf[big species] is overwritten by its owner right after the barrier
            // while other warps still need the old value: hand it over separately.
            if (is_big) ybig[tid - W] = static_cast<double>(y);
        }
        __syncthreads();

        // ---- finalize: big species sums, zone-wide dt -----------------------
        real bFp = 0, bFm = 0;
        double cand = INFINITY;
        if (lane >= W && lane < W + nbs) {
            const int s = lane - W;
            for (int w = 0; w < W; ++w) {  // fixed order over warps
                bFp += red[w * kRedStride + 2 * s];
                bFm += red[w * kRedStride + 2 * s + 1];
            }
            if (MODE == kAdaptive) {
                const real yb = static_cast<real>(ybig[s]);
                real a = bFp - bFm;
                a = a < 0 ? -a : a;
                if (a > 0) cand = static_cast<double>(eps_y * (yb > y_floor ? yb : y_floor) / a);
            }
        } else if (MODE == kAdaptive && lane < W) {
            cand = redmin[lane];
        }
        if (is_big) {  // warp 0, lane == tid: this lane just summed its own rows
            Fp = bFp;
            Fm = bFm;
        }
        if (MODE == kRhs) {
            if (own >= 0) {
                reinterpret_cast<real*>(p.Fplus)[(size_t)z * N + own] = Fp;
                reinterpret_cast<real*>(p.Fminus)[(size_t)z * N + own] = Fm;
            }
            return;
        }

        double dts;
        bool last;
        if (MODE == kAdaptive) {
            const double cmin = warp_min_pos(cand);
            double dt_ctrl = p.growth * dt_prev;
            if (cmin < dt_ctrl) dt_ctrl = cmin;
            const double rem = p.t_hydro - t;
            if (dt_ctrl >= rem * (1.0 - 1e-12)) {
                dts = rem;
                last = true;
            } else {
                dts = dt_ctrl;
                last = false;
            }
            dt_prev = dt_ctrl;
        } else {
            dts = p.dt_fixed;
            last = (steps + 1 >= p.n_fixed);
        }

        // ---- S4: update (Eq. (3)) -------------------------
        if (own >= 0) {
            const real h = static_cast<real>(dts);
            const real k = (y > 0) ? Fm / y : static_cast<real>(0);
            const real kdt = k * h;
            if (kdt >= kappa)
                y = (y + h * Fp) / (static_cast<real>(1) + kdt);
            else
                y = y + h * (Fp - Fm);
            Ybuf[own] = y;
        }
        t = last ? p.t_hydro : t + dts;
        ++steps;
        if (last) run = false;
        else if (MODE == kAdaptive && steps >= p.max_steps) {
            status |= NET_STATUS_MAX_STEPS;
            run = false;
        }
        __syncthreads();
    }

    // ---- S6: zone state out ----------------------------------------------
    const int bad = (own >= 0) && !isfinite(static_cast<double>(y));
    if (__syncthreads_or(bad)) status |= NET_STATUS_NONFINITE;
    for (int i = tid; i < N; i += T) Yg[i] = Ybuf[i];
    if (tid == 0) {
        if (MODE == kAdaptive && p.dt) p.dt[z] = dt_prev;
        if (p.n_steps) p.n_steps[z] = static_cast<int>(steps);
        if (p.status) p.status[z] = status;
    }
}

// ---------------------------------------------------------------------------
// Register-resident variant (the one bench.py times when the network fits the
// kFast* capacities): same schedule, same three barriers, but
//   * rates and every index table of a thread live in registers for the whole
//     hydro step (topology is static, sub-steps number 1e2..1e4), loops are
//     fully unrolled, so the sub-step issues no global loads and no address math;
//   * the six big-row partial sums are combined by ONE transposed butterfly
//     (9 shuffle rounds instead of 30);
//   * one reciprocal per dt candidate and one per asymptotic update (MUFU seed
//     + Newton) replace three IEEE divisions.
// ---------------------------------------------------------------------------
constexpr int kRS = kinnet::kFastSlots;
constexpr int kPC = kinnet::kFastPlus;
constexpr int kMC = kinnet::kFastMinus;

__device__ __forceinline__ double rcp_pos(double b) {  // b normal, positive
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(b));
    double e = fma(-b, r, 1.0);
    e = fma(e, e, e);
    r = fma(r, e, r);
    e = fma(-b, r, 1.0);
    r = fma(r, e, r);
    return r;
}
__device__ __forceinline__ float rcp_pos(float b) { return __frcp_rn(b); }

template <typename real> struct Tiny;
template <> struct Tiny<double> { static __device__ __forceinline__ double v() { return 1e-290; } };
template <> struct Tiny<float> { static __device__ __forceinline__ float v() { return 1e-30f; } };

// Sum rows 0..7 of acc over the warp; on return lane l holds, in the returned
// value, the warp total of row (l >> 2) & 7.  Fixed order: deterministic.
template <typename real>
__device__ __forceinline__ real warp_sum_rows8(const real (&acc)[8], int lane) {
    real a[4], b[2], c;
    const bool up16 = lane & 16, up8 = lane & 8, up4 = lane & 4;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const real send = up16 ? acc[i] : acc[i + 4];
        const real keep = up16 ? acc[i + 4] : acc[i];
        a[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const real send = up8 ? a[i] : a[i + 2];
        const real keep = up8 ? a[i + 2] : a[i];
        b[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    }
    {
        const real send = up4 ? b[0] : b[1];
        const real keep = up4 ? b[1] : b[0];
        c = keep + __shfl_xor_sync(0xffffffffu, send, 4);
    }
    c += __shfl_xor_sync(0xffffffffu, c, 2);
    c += __shfl_xor_sync(0xffffffffu, c, 1);
    return c;
}

template <typename real>
size_t smem_bytes_reg(const Schedule& S) {
    return 64 * sizeof(double) +
           sizeof(real) * (static_cast<size_t>(real_words_before_flux(S.N)) +
                           static_cast<size_t>(S.rs + 1) * S.T +
                           static_cast<size_t>(S.W) * kRedStride);
}

// Field extraction from the packed tables.  volatile: the tables are loop
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
__device__ __forceinline__ uint32_t nib(uint32_t x, int q) {
    uint32_t r;
    asm volatile("bfe.u32 %0, %1, %2, 4;" : "=r"(r) : "r"(x), "r"(4 * q));
    return r;
}

template <typename real>
__device__ __forceinline__ real lds_at(const unsigned char* base, uint32_t byte_off) {
    return *reinterpret_cast<const real*>(base + byte_off);
}

template <typename real, int MODE, int TB, int MINB>
__global__ void __launch_bounds__(TB, MINB) zone_kernel_reg(const KParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int T = p.T, N = p.N, W = p.W, rs = p.rs, nbs = p.nbs;
    const int j2 = p.j2, j3 = p.j3;
    const int z = blockIdx.x;

    double* redmin = reinterpret_cast<double*>(smem_raw);
    double* ybig = redmin + 32;
    real* Ybuf = reinterpret_cast<real*>(redmin + 64);
    real* fbuf = Ybuf + real_words_before_flux(N);  // [rs + 1][T]; row rs stays zero
    real* red = fbuf + (rs + 1) * T;
    real* fcol = fbuf + tid;  // this thread's bank-aligned flux column
    const unsigned char* Yb = reinterpret_cast<const unsigned char*>(Ybuf);
    const unsigned char* fb = reinterpret_cast<const unsigned char*>(fbuf);
    const uint32_t col_stride = static_cast<uint32_t>(T) * sizeof(real);

    // ---- tables -> registers -------------------------------------------------
    uint32_t fx[kRS], fxc[kinnet::kFastSlots3], pl[kPC / 2], mi[kMC / 2], rb[2 * kMaxBig];
#pragma unroll
    for (int j = 0; j < kRS; ++j) fx[j] = (j < rs) ? p.fx_pack[j * T + tid] : 0u;
#pragma unroll
    for (int j = 0; j < kinnet::kFastSlots3; ++j) fxc[j] = (j < rs) ? p.fxc_pack[j * T + tid] : 0u;
#pragma unroll
    for (int e = 0; e < kPC / 2; ++e) pl[e] = p.plus_pack[e * T + tid];
#pragma unroll
    for (int e = 0; e < kMC / 2; ++e) mi[e] = p.minus_pack[e * T + tid];
#pragma unroll
    for (int b = 0; b < 2 * kMaxBig; ++b) rb[b] = p.rb_pack[b * T + tid];
    // warp-wide trip counts (threads of a warp own rows of similar length)
    int wnp, wnm;
    uint32_t wrb = 0;
    {
        const uint32_t cnt = p.cnt_pack[tid], rbcnt = p.rbcnt_pack[tid];
        wnp = __reduce_max_sync(0xffffffffu, cnt & 255u);
        wnm = __reduce_max_sync(0xffffffffu, (cnt >> 8) & 255u);
#pragma unroll
        for (int b = 0; b < 2 * kMaxBig; ++b)
            wrb |= __reduce_max_sync(0xffffffffu, (rbcnt >> (4 * b)) & 15u) << (4 * b);
    }

    // ---- S1: rates, once per zone per call, kept in registers ------------------
    real R[kRS];
    {
        const int slots = rs * T;
        const double T9 = p.T9[z], rho = p.rho[z];
        const double t13 = cbrt(T9);
        const double t53 = T9 * t13 * t13;
        const double lnT = log(T9), lnrho = log(rho);
#pragma unroll
        for (int j = 0; j < kRS; ++j) {
            R[j] = 0;
            if (j < rs) {
                const double* c = p.coef + (j * T + tid);
                const double lnR = c[0] + c[1 * (size_t)slots] / T9 + c[2 * (size_t)slots] / t13 +
                                   c[3 * (size_t)slots] * t13 + c[4 * (size_t)slots] * T9 +
                                   c[5 * (size_t)slots] * t53 + c[6 * (size_t)slots] * lnT;
                R[j] = static_cast<real>(exp(c[7 * (size_t)slots] * lnrho + lnR));
            }
        }
    }

    // ---- S6: zone state in ------------------------------------------------------
    real* Yg = reinterpret_cast<real*>(p.Y) + (size_t)z * N;
    for (int i = tid; i < N; i += T) Ybuf[i] = Yg[i];
    if (tid == 0) Ybuf[N] = static_cast<real>(1);
    fcol[rs * T] = static_cast<real>(0);
    const int own = p.owner[tid];
    const bool is_big = (tid >= W && tid < W + nbs);
    __syncthreads();
    real y = (own >= 0) ? Ybuf[own] : static_cast<real>(0);

    const real kappa = static_cast<real>(p.kappa);
    const real eps_y = static_cast<real>(p.eps_y);
    const real y_floor = static_cast<real>(p.y_floor);
    const double growth = p.growth, t_hydro = p.t_hydro;

    double t = 0.0, dt_prev = 0.0;
    int steps = 0;
    int status = 0;
    bool run = true;
    if (MODE == kAdaptive) {
        const double dt_in = p.dt ? p.dt[z] : 0.0;
        dt_prev = (dt_in > 0.0) ? dt_in : t_hydro;
        run = t_hydro > 0.0;
        if (!run) dt_prev = dt_in;
    } else if (MODE == kFixed) {
        run = p.n_fixed > 0;
    }
    const int max_steps = static_cast<int>(MODE == kFixed ? p.n_fixed : p.max_steps);

    while (run) {
        // ---- S2: fluxes -------------------------------------------------------
#pragma unroll
        for (int j = 0; j < kRS; ++j) {
            if (j < rs) {
                real v = R[j] * lds_at<real>(Yb, lo16(fx[j]));
                if (j < j2) v = v * lds_at<real>(Yb, hi16(fx[j]));
                if (j < kinnet::kFastSlots3 && j < j3) v = v * lds_at<real>(Yb, fxc[j]);
                fcol[j * T] = v;
            }
        }
        __syncthreads();

        // ---- S3: sums (zero-padded lists: no per-lane predicates) ------------------
        real Fp = 0, Fm = 0;
        {
            real Fp1 = 0, Fm1 = 0;
#pragma unroll
            for (int g = 0; g < kPC / 4; ++g) {
                if (4 * g < wnp) {
                    const uint32_t w0 = pl[2 * g], w1 = pl[2 * g + 1];
                    Fp += lds_at<real>(fb, lo16(w0));
                    Fp1 += lds_at<real>(fb, hi16(w0));
                    Fp += lds_at<real>(fb, lo16(w1));
                    Fp1 += lds_at<real>(fb, hi16(w1));
                }
            }
#pragma unroll
            for (int g = 0; g < kMC / 4; ++g) {
                if (4 * g < wnm) {
                    const uint32_t w0 = mi[2 * g], w1 = mi[2 * g + 1];
                    Fm += lds_at<real>(fb, lo16(w0));
                    Fm1 += lds_at<real>(fb, hi16(w0));
                    Fm += lds_at<real>(fb, lo16(w1));
                    Fm1 += lds_at<real>(fb, hi16(w1));
                }
            }
            Fp += Fp1;
            Fm += Fm1;
        }
        if (nbs > 0) {
            real acc[8];
            const unsigned char* fc = reinterpret_cast<const unsigned char*>(fcol);
#pragma unroll
            for (int b = 0; b < 8; ++b) {
                acc[b] = 0;
                if (b < 2 * kMaxBig) {
                    const int wmax = (wrb >> (4 * b)) & 15u;
#pragma unroll
                    for (int q = 0; q < kinnet::kFastRowCap; q += 2) {
                        if (q < wmax) {
                            const uint32_t s0 = nib(rb[b], q);
                            const uint32_t s1 = nib(rb[b], q + 1);
                            acc[b] += lds_at<real>(fc, s0 * col_stride);
                            acc[b] += lds_at<real>(fc, s1 * col_stride);
                        }
                    }
                }
            }
            const real tot = warp_sum_rows8(acc, lane);
            if ((lane & 3) == 0) red[warp * kRedStride + (lane >> 2)] = tot;
        }
        // ---- S5: dt candidates of the small species ---------------------------------
        if (MODE == kAdaptive) {
            double c = INFINITY;
            if (own >= 0 && !is_big) {
                real a = Fp - Fm;
                a = a < 0 ? -a : a;
                if (a > Tiny<real>::v())
                    c = static_cast<double>(eps_y * (y > y_floor ? y : y_floor) * rcp_pos(a));
            }
            c = warp_min_pos(c);
            if (lane == 0) redmin[warp] = c;
            if (is_big) ybig[tid - W] = static_cast<double>(y);
        }
        __syncthreads();

        // ---- finalize: big species sums, zone-wide dt ---------------------------------
        real bFp = 0, bFm = 0;
        double cand = INFINITY;
        if (lane >= W && lane < W + nbs) {
            const int s = lane - W;
            for (int w = 0; w < W; ++w) {
                bFp += red[w * kRedStride + 2 * s];
                bFm += red[w * kRedStride + 2 * s + 1];
            }
            if (MODE == kAdaptive) {
                const real yb = static_cast<real>(ybig[s]);
                real a = bFp - bFm;
                a = a < 0 ? -a : a;
                if (a > Tiny<real>::v())
                    cand = static_cast<double>(eps_y * (yb > y_floor ? yb : y_floor) * rcp_pos(a));
            }
        } else if (MODE == kAdaptive && lane < W) {
            cand = redmin[lane];
        }
        if (is_big) {
            Fp = bFp;
            Fm = bFm;
        }
        if (MODE == kRhs) {
            if (own >= 0) {
                reinterpret_cast<real*>(p.Fplus)[(size_t)z * N + own] = Fp;
                reinterpret_cast<real*>(p.Fminus)[(size_t)z * N + own] = Fm;
            }
            return;
        }

        double dts;
        bool last;
        if (MODE == kAdaptive) {
            const double cmin = warp_min_pos(cand);
            double dt_ctrl = growth * dt_prev;
            if (cmin < dt_ctrl) dt_ctrl = cmin;
            const double rem = t_hydro - t;
            if (dt_ctrl >= rem * (1.0 - 1e-12)) {
                dts = rem;
                last = true;
            } else {
                dts = dt_ctrl;
                last = false;
            }
            dt_prev = dt_ctrl;
        } else {
            dts = p.dt_fixed;
            last = (steps + 1 >= max_steps);
        }

        // ---- S4: update -------------------------------------------------------------------
        if (own >= 0) {
            const real h = static_cast<real>(dts);
            const real hFm = h * Fm;
            if (y > 0 && hFm >= kappa * y) {  // k dt >= kappa with k = F-/Y
                const real den = y + hFm;      // Eq. (3) as Y (Y + dt F+) / (Y + dt F-)
                if (den > Tiny<real>::v() && y > Tiny<real>::v())
                    y = (y + h * Fp) * (y * rcp_pos(den));
                else
                    y = (y + h * Fp) / (static_cast<real>(1) + (Fm / y) * h);
            } else {
                y = y + h * (Fp - Fm);
            }
            Ybuf[own] = y;
        }
        t = last ? t_hydro : t + dts;
        ++steps;
        if (last) run = false;
        else if (MODE == kAdaptive && steps >= max_steps) {
            status |= NET_STATUS_MAX_STEPS;
            run = false;
        }
        __syncthreads();
    }

    const int bad = (own >= 0) && !isfinite(static_cast<double>(y));
    if (__syncthreads_or(bad)) status |= NET_STATUS_NONFINITE;
    for (int i = tid; i < N; i += T) Yg[i] = Ybuf[i];
    if (tid == 0) {
        if (MODE == kAdaptive && p.dt) p.dt[z] = dt_prev;
        if (p.n_steps) p.n_steps[z] = steps;
        if (p.status) p.status[z] = status;
    }
}

struct DeviceTables {
    int32_t* flux_rxn = nullptr;
    ushort4* flux_react = nullptr;
    double* coef = nullptr;
    int32_t* owner = nullptr;
    uint16_t* small_plus = nullptr;
    uint16_t* small_minus = nullptr;
    uint16_t* small_src = nullptr;
    uint8_t* big_cnt = nullptr;
    uint8_t* big_slot = nullptr;
    uint32_t* fx_pack = nullptr;
    uint32_t* fxc_pack = nullptr;
    uint32_t* plus_pack = nullptr;
    uint32_t* minus_pack = nullptr;
    uint32_t* rb_pack = nullptr;
    uint32_t* cnt_pack = nullptr;
    uint32_t* rbcnt_pack = nullptr;
};

}  // namespace

struct net {
    Schedule S;
    net_params_t P;
    bool has_device = false;
    bool force_generic = false;  // params.kernel == 1: keep the table-driven kernel (A/B tests)
    int device = -1;
    int zones_per_sm = 0;
    DeviceTables D;
    // scratch of net_integrate_host
    cudaStream_t host_stream = nullptr;
    int scratch_zones = 0;
    double *sT9 = nullptr, *srho = nullptr, *sdt = nullptr;
    void* sY = nullptr;
    int *ssteps = nullptr, *sstatus = nullptr;
};

namespace {

template <typename T>
int upload(T** dst, const void* src, size_t count) {
    CUDA_TRY(cudaMalloc(reinterpret_cast<void**>(dst), std::max<size_t>(count, 1) * sizeof(T)));
    if (count) CUDA_TRY(cudaMemcpy(*dst, src, count * sizeof(T), cudaMemcpyHostToDevice));
    return NET_OK;
}

typedef void (*kernel_fn)(const KParams);

template <typename real, int MODE>
kernel_fn pick_block(int T) {
    if (T <= 256) return zone_kernel<real, MODE, 256>;
    if (T <= 512) return zone_kernel<real, MODE, 512>;
    return zone_kernel<real, MODE, 1024>;
}

// register-resident kernel: block-size classes with the residency the register
// file allows (65536 / (TB * MINB) registers per thread)
template <typename real, int MODE>
kernel_fn pick_block_reg(int T) {
    if (T <= 64) return zone_kernel_reg<real, MODE, 64, 8>;
    if (T <= 160) return zone_kernel_reg<real, MODE, 160, 3>;
    if (T <= 256) return zone_kernel_reg<real, MODE, 256, 2>;
    if (T <= 512) return zone_kernel_reg<real, MODE, 512, 1>;
    return nullptr;
}

bool use_reg_kernel(const net* n);

template <int MODE>
kernel_fn pick_kernel(const net* n) {
    if constexpr (MODE == kRates) return pick_block<double, MODE>(n->S.T);
    else if (use_reg_kernel(n)) {
        kernel_fn f = n->P.precision == 32 ? pick_block_reg<float, MODE>(n->S.T)
                                           : pick_block_reg<double, MODE>(n->S.T);
        if (f) return f;
    }
    return n->P.precision == 32 ? pick_block<float, MODE>(n->S.T) : pick_block<double, MODE>(n->S.T);
}

bool use_reg_kernel(const net* n) { return n->S.fast_ok && !n->force_generic; }

size_t net_smem(const net* n) {
    if (use_reg_kernel(n))
        return n->P.precision == 32 ? smem_bytes_reg<float>(n->S) : smem_bytes_reg<double>(n->S);
    return n->P.precision == 32 ? smem_bytes<float>(n->S) : smem_bytes<double>(n->S);
}

int prepare_kernels(net* n) {
    const size_t smem = net_smem(n);
    kernel_fn fns[4] = {pick_kernel<kAdaptive>(n), pick_kernel<kFixed>(n), pick_kernel<kRhs>(n),
                        pick_kernel<kRates>(n)};
    for (kernel_fn f : fns) {
        const size_t need = (f == fns[3]) ? smem_bytes<double>(n->S) : smem;
        CUDA_TRY(cudaFuncSetAttribute(reinterpret_cast<const void*>(f),
                                      cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      static_cast<int>(need)));
    }
    int nb = 0;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(
        &nb, reinterpret_cast<const void*>(fns[0]), n->S.T, smem));
    n->zones_per_sm = nb;
    return NET_OK;
}

void fill_params(const net* n, KParams& k) {
    const Schedule& S = n->S;
    std::memset(&k, 0, sizeof(k));
    k.N = S.N; k.M = S.M; k.T = S.T; k.W = S.W; k.rs = S.rs; k.j2 = S.j2; k.j3 = S.j3;
    k.nbs = S.nbs;
    for (int s = 0; s < S.nbs; ++s) k.big_species[s] = S.big_species[s];
    k.flux_rxn = n->D.flux_rxn;
    k.flux_react = n->D.flux_react;
    k.coef = n->D.coef;
    k.owner = n->D.owner;
    k.small_plus = n->D.small_plus;
    k.small_minus = n->D.small_minus;
    k.small_src = n->D.small_src;
    k.big_cnt = n->D.big_cnt;
    k.big_slot = n->D.big_slot;
    k.fx_pack = n->D.fx_pack;
    k.fxc_pack = n->D.fxc_pack;
    k.plus_pack = n->D.plus_pack;
    k.minus_pack = n->D.minus_pack;
    k.rb_pack = n->D.rb_pack;
    k.cnt_pack = n->D.cnt_pack;
    k.rbcnt_pack = n->D.rbcnt_pack;
    k.kappa = n->P.kappa; k.eps_y = n->P.eps_y; k.y_floor = n->P.y_floor;
    k.growth = n->P.growth; k.max_steps = n->P.max_steps;
}

template <int MODE>
int launch(net* n, int zones, KParams& k, void* stream) {
    if (!n) return fail(NET_EINVAL, "null net");
    if (!n->has_device) return fail(NET_ECUDA, "net has no device copy (net_create_host)");
    if (zones < 0) return fail(NET_EINVAL, "zones < 0");
    if (zones == 0) return NET_OK;
    if (!k.T9 || !k.rho) return fail(NET_EINVAL, "null T9/rho");
    const size_t smem = (MODE == kRates) ? smem_bytes<double>(n->S) : net_smem(n);
    kernel_fn f = pick_kernel<MODE>(n);
    f<<<zones, n->S.T, smem, static_cast<cudaStream_t>(stream)>>>(k);
    CUDA_TRY(cudaGetLastError());
    return NET_OK;
}

int create_common(net_t** out, int N, const int* A, int M, const int* n_react, const int* react,
                  const int* n_prod, const int* prod, const double* coef,
                  const net_params_t* params, bool device) {
    if (!out) return fail(NET_EINVAL, "null out pointer");
    *out = nullptr;
    net* n = new (std::nothrow) net();
    if (!n) return fail(NET_ENOMEM, "out of host memory");
    if (params) n->P = *params; else net_default_params(&n->P);
    if (n->P.precision == 0) n->P.precision = 64;
    n->force_generic = (n->P.kernel == 1);
    if (n->P.precision != 64 && n->P.precision != 32) {
        delete n;
        return fail(NET_EINVAL, "precision must be 64 or 32");
    }
    if (!(n->P.kappa > 0) || !(n->P.eps_y > 0) || !(n->P.y_floor > 0) || !(n->P.growth > 1) ||
        n->P.max_steps < 1 || n->P.max_steps > 2000000000LL) {
        delete n;
        return fail(NET_EINVAL, "bad integrator parameter");
    }
    std::string err;
    int rc;
    try {
        rc = kinnet::build_schedule(N, A, M, n_react, react, n_prod, prod, coef, n->S, err);
    } catch (const std::bad_alloc&) {
        delete n;
        return fail(NET_ENOMEM, "out of host memory");
    }
    if (rc != NET_OK) {
        delete n;
        return fail(rc, err);
    }
    if (n->S.fast_ok) kinnet::pack_fast_tables(n->S, n->P.precision == 32 ? 4 : 8);
    if (net_smem(n) > 227 * 1024) {
        delete n;
        return fail(NET_EINVAL, "network too large for one CTA's shared memory");
    }
    if (device) {
        const Schedule& S = n->S;
        rc = NET_OK;
        if (cudaGetDevice(&n->device) != cudaSuccess) rc = fail(NET_ECUDA, "no CUDA device");
        if (rc == NET_OK) rc = upload(&n->D.flux_rxn, S.flux_rxn.data(), S.flux_rxn.size());
        if (rc == NET_OK)
            rc = upload(&n->D.flux_react, S.flux_react.data(), S.flux_react.size() / 4);
        if (rc == NET_OK) rc = upload(&n->D.coef, S.coef.data(), S.coef.size());
        if (rc == NET_OK) rc = upload(&n->D.owner, S.owner.data(), S.owner.size());
        if (rc == NET_OK) rc = upload(&n->D.small_plus, S.small_plus.data(), S.small_plus.size());
        if (rc == NET_OK) rc = upload(&n->D.small_minus, S.small_minus.data(), S.small_minus.size());
        if (rc == NET_OK) rc = upload(&n->D.small_src, S.small_src.data(), S.small_src.size());
        if (rc == NET_OK) rc = upload(&n->D.big_cnt, S.big_cnt.data(), S.big_cnt.size());
        if (rc == NET_OK) rc = upload(&n->D.big_slot, S.big_slot.data(), S.big_slot.size());
        if (rc == NET_OK && S.fast_ok) {
            rc = upload(&n->D.fx_pack, S.fx_pack.data(), S.fx_pack.size());
            if (rc == NET_OK) rc = upload(&n->D.fxc_pack, S.fxc_pack.data(), S.fxc_pack.size());
            if (rc == NET_OK) rc = upload(&n->D.plus_pack, S.plus_pack.data(), S.plus_pack.size());
            if (rc == NET_OK) rc = upload(&n->D.minus_pack, S.minus_pack.data(), S.minus_pack.size());
            if (rc == NET_OK) rc = upload(&n->D.rb_pack, S.rb_pack.data(), S.rb_pack.size());
            if (rc == NET_OK) rc = upload(&n->D.cnt_pack, S.cnt_pack.data(), S.cnt_pack.size());
            if (rc == NET_OK) rc = upload(&n->D.rbcnt_pack, S.rbcnt_pack.data(), S.rbcnt_pack.size());
        }
        if (rc == NET_OK) {
            n->has_device = true;
            rc = prepare_kernels(n);
        }
        if (rc != NET_OK) {
            std::string keep = g_last_error;
            net_destroy(n);
            g_last_error = keep;
            return rc;
        }
    }
    *out = n;
    return NET_OK;
}

}  // namespace

extern "C" {

int net_default_params(net_params_t* p) {
    if (!p) return fail(NET_EINVAL, "null params");
    p->kappa = 1.0;
    p->eps_y = 0.05;
    p->y_floor = 1e-10;
    p->growth = 2.0;
    p->max_steps = 10000000LL;
    p->precision = 64;
    p->kernel = 0;
    return NET_OK;
}

int net_create(net_t** out, int n_species, const int* A, int n_reactions, const int* n_react,
               const int* react, const int* n_prod, const int* prod, const double* coef,
               const net_params_t* params) {
    return create_common(out, n_species, A, n_reactions, n_react, react, n_prod, prod, coef,
                         params, true);
}

int net_create_host(net_t** out, int n_species, const int* A, int n_reactions,
                    const int* n_react, const int* react, const int* n_prod, const int* prod,
                    const double* coef, const net_params_t* params) {
    return create_common(out, n_species, A, n_reactions, n_react, react, n_prod, prod, coef,
                         params, false);
}

void net_destroy(net_t* n) {
    if (!n) return;
    if (n->has_device) {
        cudaFree(n->D.flux_rxn); cudaFree(n->D.flux_react); cudaFree(n->D.coef);
        cudaFree(n->D.owner); cudaFree(n->D.small_plus); cudaFree(n->D.small_minus);
        cudaFree(n->D.small_src); cudaFree(n->D.big_cnt); cudaFree(n->D.big_slot);
        cudaFree(n->D.fx_pack); cudaFree(n->D.fxc_pack); cudaFree(n->D.plus_pack); cudaFree(n->D.minus_pack);
        cudaFree(n->D.rb_pack); cudaFree(n->D.cnt_pack); cudaFree(n->D.rbcnt_pack);
        cudaFree(n->sT9); cudaFree(n->srho); cudaFree(n->sdt); cudaFree(n->sY);
        cudaFree(n->ssteps); cudaFree(n->sstatus);
        if (n->host_stream) cudaStreamDestroy(n->host_stream);
    }
    delete n;
}

int net_integrate(net_t* n, int zones, const double* T9, const double* rho, void* Y,
                  double t_hydro, double* dt, int* n_steps, int* status, void* stream) {
    if (!n) return fail(NET_EINVAL, "null net");
    if (zones > 0 && !Y) return fail(NET_EINVAL, "null Y");
    if (!(t_hydro == t_hydro)) return fail(NET_EINVAL, "t_hydro is NaN");
    KParams k;
    fill_params(n, k);
    k.T9 = T9; k.rho = rho; k.Y = Y; k.dt = dt; k.n_steps = n_steps; k.status = status;
    k.t_hydro = t_hydro;
    return launch<kAdaptive>(n, zones, k, stream);
}

int net_integrate_fixed(net_t* n, int zones, const double* T9, const double* rho, void* Y,
                        double dt_fixed, long long n_steps, void* stream) {
    if (!n) return fail(NET_EINVAL, "null net");
    if (zones > 0 && !Y) return fail(NET_EINVAL, "null Y");
    if (n_steps < 0 || n_steps > 2000000000LL) return fail(NET_EINVAL, "n_steps out of range [0, 2e9]");
    KParams k;
    fill_params(n, k);
    k.T9 = T9; k.rho = rho; k.Y = Y;
    k.dt_fixed = dt_fixed; k.n_fixed = n_steps;
    return launch<kFixed>(n, zones, k, stream);
}

int net_rates(net_t* n, int zones, const double* T9, const double* rho, double* R, void* stream) {
    if (!n) return fail(NET_EINVAL, "null net");
    if (zones > 0 && !R) return fail(NET_EINVAL, "null R");
    KParams k;
    fill_params(n, k);
    k.T9 = T9; k.rho = rho; k.Rout = R;
    return launch<kRates>(n, zones, k, stream);
}

int net_rhs(net_t* n, int zones, const double* T9, const double* rho, const void* Y, void* Fplus,
            void* Fminus, void* stream) {
    if (!n) return fail(NET_EINVAL, "null net");
    if (zones > 0 && (!Y || !Fplus || !Fminus)) return fail(NET_EINVAL, "null Y/Fplus/Fminus");
    KParams k;
    fill_params(n, k);
    k.T9 = T9; k.rho = rho; k.Y = const_cast<void*>(Y); k.Fplus = Fplus; k.Fminus = Fminus;
    return launch<kRhs>(n, zones, k, stream);
}

int net_integrate_host(net_t* n, int zones, const double* T9, const double* rho, void* Y,
                       double t_hydro, double* dt, int* n_steps, int* status) {
    if (!n) return fail(NET_EINVAL, "null net");
    if (!n->has_device) return fail(NET_ECUDA, "net has no device copy (net_create_host)");
    if (zones < 0) return fail(NET_EINVAL, "zones < 0");
    if (zones == 0) return NET_OK;
    if (!T9 || !rho || !Y) return fail(NET_EINVAL, "null T9/rho/Y");
    const size_t ysz = (n->P.precision == 32 ? sizeof(float) : sizeof(double)) * (size_t)n->S.N;
    if (!n->host_stream) CUDA_TRY(cudaStreamCreateWithFlags(&n->host_stream, cudaStreamNonBlocking));
    if (zones > n->scratch_zones) {
        cudaFree(n->sT9); cudaFree(n->srho); cudaFree(n->sdt); cudaFree(n->sY);
        cudaFree(n->ssteps); cudaFree(n->sstatus);
        n->sT9 = n->srho = n->sdt = nullptr; n->sY = nullptr; n->ssteps = n->sstatus = nullptr;
        n->scratch_zones = 0;
        CUDA_TRY(cudaMalloc(reinterpret_cast<void**>(&n->sT9), sizeof(double) * zones));
        CUDA_TRY(cudaMalloc(reinterpret_cast<void**>(&n->srho), sizeof(double) * zones));
        CUDA_TRY(cudaMalloc(reinterpret_cast<void**>(&n->sdt), sizeof(double) * zones));
        CUDA_TRY(cudaMalloc(&n->sY, ysz * zones));
        CUDA_TRY(cudaMalloc(reinterpret_cast<void**>(&n->ssteps), sizeof(int) * zones));
        CUDA_TRY(cudaMalloc(reinterpret_cast<void**>(&n->sstatus), sizeof(int) * zones));
        n->scratch_zones = zones;
    }
    cudaStream_t s = n->host_stream;
    CUDA_TRY(cudaMemcpyAsync(n->sT9, T9, sizeof(double) * zones, cudaMemcpyHostToDevice, s));
    CUDA_TRY(cudaMemcpyAsync(n->srho, rho, sizeof(double) * zones, cudaMemcpyHostToDevice, s));
    CUDA_TRY(cudaMemcpyAsync(n->sY, Y, ysz * zones, cudaMemcpyHostToDevice, s));
    if (dt) CUDA_TRY(cudaMemcpyAsync(n->sdt, dt, sizeof(double) * zones, cudaMemcpyHostToDevice, s));
    else CUDA_TRY(cudaMemsetAsync(n->sdt, 0, sizeof(double) * zones, s));
    int rc = net_integrate(n, zones, n->sT9, n->srho, n->sY, t_hydro, n->sdt, n->ssteps,
                           n->sstatus, s);
    if (rc != NET_OK) return rc;
    CUDA_TRY(cudaMemcpyAsync(Y, n->sY, ysz * zones, cudaMemcpyDeviceToHost, s));
    if (dt) CUDA_TRY(cudaMemcpyAsync(dt, n->sdt, sizeof(double) * zones, cudaMemcpyDeviceToHost, s));
    if (n_steps)
        CUDA_TRY(cudaMemcpyAsync(n_steps, n->ssteps, sizeof(int) * zones, cudaMemcpyDeviceToHost, s));
    if (status)
        CUDA_TRY(cudaMemcpyAsync(status, n->sstatus, sizeof(int) * zones, cudaMemcpyDeviceToHost, s));
    CUDA_TRY(cudaStreamSynchronize(s));
    return NET_OK;
}

int net_schedule_info(const net_t* n, net_schedule_info_t* info) {
    if (!n || !info) return fail(NET_EINVAL, "null argument");
    const Schedule& S = n->S;
    info->n_species = S.N;
    info->n_reactions = S.M;
    info->threads = S.T;
    info->flux_slots = S.rs;
    info->slots_2body = S.j2;
    info->slots_3body = S.j3;
    info->n_entries = S.n_entries;
    info->n_big_species = S.nbs;
    info->n_entries_big = S.n_entries_big;
    info->small_max = S.small_max;
    info->readback_max = S.readback_max;
    info->smem_bytes = static_cast<int>(net_smem(n));
    info->zones_per_sm = n->zones_per_sm;
    return NET_OK;
}

int net_schedule_table(const net_t* n, const char* name, int* out, int cap) {
    if (!n || !name) return fail(NET_EINVAL, "null argument");
    const Schedule& S = n->S;
    const std::string key(name);
    int count = -1;
    auto emit = [&](auto const& vec, size_t stride, size_t take) {
        // copies `take` of every `stride` elements
        const size_t groups = stride ? vec.size() / stride : 0;
        count = static_cast<int>(groups * take);
        if (out && cap >= count)
            for (size_t g = 0, o = 0; g < groups; ++g)
                for (size_t q = 0; q < take; ++q) out[o++] = static_cast<int>(vec[g * stride + q]);
    };
    if (key == "flux_rxn") emit(S.flux_rxn, 1, 1);
    else if (key == "flux_react") emit(S.flux_react, 4, 3);
    else if (key == "owner") emit(S.owner, 1, 1);
    else if (key == "small_plus") emit(S.small_plus, 1, 1);
    else if (key == "small_minus") emit(S.small_minus, 1, 1);
    else if (key == "small_src") {
        if (S.small_max == 0) count = 0; else emit(S.small_src, 1, 1);
    } else if (key == "big_species") emit(S.big_species, 1, 1);
    else if (key == "big_cnt") {
        if (S.nbs == 0) count = 0; else emit(S.big_cnt, 1, 1);
    } else if (key == "big_slot") {
        if (S.readback_max == 0) count = 0; else emit(S.big_slot, 1, 1);
    } else return fail(NET_EINVAL, "unknown schedule table '" + key + "'");
    if (out && cap < count) return fail(NET_EINVAL, "output buffer too small");
    return count;
}

const char* net_last_error(void) { return g_last_error.c_str(); }

}  // extern "C"
