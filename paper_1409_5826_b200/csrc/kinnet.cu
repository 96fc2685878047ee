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
#include <cstdlib>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/kinnet.h"
#include "device_util.cuh"
#include "schedule.h"
#include "zone_pull.cuh"
#include "zone_pull2.cuh"

namespace {

using kinnet::KPull;
using kinnet::Schedule;
using kinnet::kAdaptive;
using kinnet::kFixed;
using kinnet::kRates;
using kinnet::kRhs;
using kinnet::pull_fn;
using kinnet::pull_smem_bytes;
using kinnet::warp_min_pos;
using kinnet::warp_sum;

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
    // zones
    const double* T9;
    const double* rho;
    const int* order;  // [zones] launch order (zone of CTA b), NULL = identity
    void* Y;
    double* dt;
    int* n_steps;
    int* status;
    const double* bind;
    double* energy;
    void* Fplus;
    void* Fminus;
    double* Rout;
    double t_hydro, dt_fixed;
    long long n_fixed;
    // integrator parameters
    double kappa, eps_y, y_floor, growth;
    long long max_steps;
    int method;  // 0 = asymptotic / Euler, 1 = QSS variant
};


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
    const int z = p.order ? p.order[blockIdx.x] : blockIdx.x;

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
            if (p.method == 1) {  // QSS variant (reading Q20)
                const real num = ((kdt + static_cast<real>(11)) * kdt + static_cast<real>(60)) * kdt + static_cast<real>(180);
                const real den = ((kdt + static_cast<real>(12)) * kdt + static_cast<real>(60)) * kdt + static_cast<real>(360);
                y = y + h * (Fp - Fm) / (static_cast<real>(1) + num / den * kdt);
            } else if (kdt >= kappa)
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
    if (p.energy) {  // uniform; Yg still holds the start-of-call abundances
        double e = 0.0;
        for (int i = tid; i < N; i += T)
            e += p.bind[i] * (static_cast<double>(Ybuf[i]) - static_cast<double>(Yg[i]));
        kinnet::zone_energy_out(e, redmin, p.energy + z);
    }
    for (int i = tid; i < N; i += T) Yg[i] = Ybuf[i];
    if (tid == 0) {
        if (MODE == kAdaptive && p.dt) p.dt[z] = dt_prev;
        if (p.n_steps) p.n_steps[z] = static_cast<int>(steps);
        if (p.status) p.status[z] = status;
    }
}


// Launch order of the zones: hottest first.  The number of sub-steps a zone needs over
// one hydro step grows steeply with its temperature (rates are exponential in T9; on
// configs[3] 12 .. 7900 sub-steps, rank correlation with T9 0.99), and the block scheduler
// hands out CTAs in index order, so in caller order the long zones that happen to start
// late run alone on their SMs at the end.  Longest-processing-time-first on the T9 proxy
// removes that tail (PAPER.md L200 leaves the load balance of unequal networks open).  A
// counting sort on T9 quantised to 1/64: a histogram kernel and a scatter kernel, both over
// as many CTAs as the batch needs, on a 2 x 1024-int workspace zeroed by a memset node in
// front of them (three stream operations, all legal under stream capture).  The order
// inside a bucket is whatever the atomics give -- it only moves WHEN a zone runs, never
// what it computes.
constexpr int kOrderBuckets = 1024;
constexpr int kOrderMinZones = 1024;
constexpr int kOrderThreads = 256;
constexpr int kOrderZonesPerCta = 4096;

__device__ __forceinline__ int order_bucket(double t9) {
    // descending temperature -> ascending bucket; NaN and <= 0 last
    const double k = t9 * 64.0;
    const int b = (k > 0.0) ? (k < 1023.0 ? static_cast<int>(k) : 1023) : 0;
    return kOrderBuckets - 1 - b;
}

__global__ void __launch_bounds__(kOrderThreads) zone_hist_kernel(const double* T9, int zones, int* hist) {
    __shared__ int h[kOrderBuckets];
    for (int i = threadIdx.x; i < kOrderBuckets; i += kOrderThreads) h[i] = 0;
    __syncthreads();
    const int lo = blockIdx.x * kOrderZonesPerCta, hi = min(zones, lo + kOrderZonesPerCta);
    for (int z = lo + threadIdx.x; z < hi; z += kOrderThreads) atomicAdd(&h[order_bucket(T9[z])], 1);
    __syncthreads();
    for (int i = threadIdx.x; i < kOrderBuckets; i += kOrderThreads)
        if (h[i]) atomicAdd(&hist[i], h[i]);
}

// Every CTA scans the 1024 counts for itself (cheaper than a fourth launch), then places its
// slice of the zones: position = start of the bucket + a ticket from the bucket's cursor.
__global__ void __launch_bounds__(kOrderThreads) zone_scatter_kernel(const double* T9, int zones, const int* hist,
                                                                    int* cursor, int* order) {
    __shared__ int start[kOrderBuckets];
    __shared__ int warp_tot[kOrderThreads / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int PER = kOrderBuckets / kOrderThreads;  // consecutive buckets per thread
    int c[PER], run = 0;
#pragma unroll
    for (int q = 0; q < PER; ++q) {
        c[q] = hist[tid * PER + q];
        run += c[q];
    }
    int incl = run;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int up = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += up;
    }
    if (lane == 31) warp_tot[warp] = incl;
    __syncthreads();
    int base = incl - run;
    for (int w = 0; w < warp; ++w) base += warp_tot[w];
#pragma unroll
    for (int q = 0; q < PER; ++q) {
        start[tid * PER + q] = base;
        base += c[q];
    }
    __syncthreads();
    const int lo = blockIdx.x * kOrderZonesPerCta, hi = min(zones, lo + kOrderZonesPerCta);
    for (int z = lo + tid; z < hi; z += kOrderThreads) {
        const int b = order_bucket(T9[z]);
        order[start[b] + atomicAdd(&cursor[b], 1)] = z;
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
    // pull kernel
    double* coef_rxn = nullptr;
    int32_t* p_owner = nullptr;
    uint32_t* p_cnt = nullptr;
    int32_t* p_slot_rxn = nullptr;
    uint32_t* p_f1 = nullptr;
    uint32_t* p_f2 = nullptr;
    uint16_t* p_agg_ptr = nullptr;
    int32_t* p_agg_ent = nullptr;
    double* bind = nullptr;  // [N] binding energies (net_set_binding_energy)
};

}  // namespace

// Launch-order workspaces ("lanes"): one per stream that has a sorted launch in flight on
// this net_t, and one per stream capture (a graph may replay at any time, beside anything).
// [0, 1024) bucket counts, [1024, 2048) bucket cursors, then the order itself.
constexpr int kLanes = 16;
constexpr int kLaneHeader = 2 * kOrderBuckets;
constexpr int kDefaultReserve = 65536;  // zones per lane allocated by net_create
constexpr int kHostStreams = 3;         // internal streams of net_integrate_host_async
constexpr int kHostMinChunk = 16384;    // zones; a staged chunk is max(this, zones / kHostMaxChunks)
constexpr int kHostMaxChunks = 16;

struct net {
    Schedule S;
    kinnet::PullSchedule PS;
    net_params_t P;
    bool has_device = false;
    bool force_generic = false;  // params.kernel == 1: keep the table-driven kernel (A/B tests)
    bool pull2 = false;          // PS is compiled for virtual threads: two species per thread
    int pull2_stair = 0;         // its schedule's staircase class (zone_pull2.cuh: pull2_stair_class)
    int pull2_spill = 0;         // side-a slot rates kept in shared memory by that kernel
    int device = -1;
    int zones_per_sm = 0;
    DeviceTables D;
    // launch-order lanes (net_create / net_reserve allocate; net_integrate only picks one)
    std::mutex mu;
    int lane_cap = 0;
    int* lane_buf[kLanes] = {};
    cudaStream_t lane_stream[kLanes] = {};
    bool lane_used[kLanes] = {};
    bool lane_captured[kLanes] = {};              // handed to a stream capture: that graph's for good
    unsigned long long lane_capture[kLanes] = {}; // ... the capture's id
    cudaEvent_t lane_done[kLanes] = {};           // recorded behind the last eager zone kernel on the lane
    unsigned long long lane_tick[kLanes] = {};    // value of `tick` at the lane's last use
    unsigned long long tick = 0;
    long long sorted_calls = 0, unsorted_calls = 0;  // calls of >= kOrderMinZones zones with / without a lane
    bool host_in_flight = false;                  // net_integrate_host_async without its net_wait
    // device scratch and streams of net_integrate_host_async
    cudaStream_t host_stream[kHostStreams] = {};
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


bool use_pull_kernel(const net* n) { return n->PS.ok && !n->force_generic; }

int pull_block(const net* n) { return n->pull2 ? n->PS.T / 2 : n->PS.T; }

pull_fn pick_pull(const net* n, bool adaptive) {
    if (n->pull2) {
        if (adaptive)
            return n->P.precision == 32 ? kinnet::pull2_kernel_f32_adaptive(n->PS, n->P.method)
                                        : kinnet::pull2_kernel_f64_adaptive(n->PS, n->P.method);
        return n->P.precision == 32 ? kinnet::pull2_kernel_f32_fixed(n->PS, n->P.method)
                                    : kinnet::pull2_kernel_f64_fixed(n->PS, n->P.method);
    }
    if (adaptive)
        return n->P.precision == 32 ? kinnet::pull_kernel_f32_adaptive(n->PS, n->P.method)
                                    : kinnet::pull_kernel_f64_adaptive(n->PS, n->P.method);
    return n->P.precision == 32 ? kinnet::pull_kernel_f32_fixed(n->PS, n->P.method)
                                : kinnet::pull_kernel_f64_fixed(n->PS, n->P.method);
}

int pull2_store_of(const net* n) { return kinnet::pull2_store(n->PS.T / 2, n->PS.nslots); }

size_t pull_smem(const net* n) {
    if (n->pull2)
        return n->P.precision == 32
                   ? kinnet::pull2_smem_bytes<float>(n->PS.T / 2, n->S.M, n->pull2_spill, pull2_store_of(n))
                   : kinnet::pull2_smem_bytes<double>(n->PS.T / 2, n->S.M, n->pull2_spill, pull2_store_of(n));
    return n->P.precision == 32 ? pull_smem_bytes<float>(n->PS.T, n->PS.W, n->S.M)
                                : pull_smem_bytes<double>(n->PS.T, n->PS.W, n->S.M);
}

template <int MODE>
kernel_fn pick_kernel(const net* n) {
    if constexpr (MODE == kRates) return pick_block<double, MODE>(n->S.T);
    return n->P.precision == 32 ? pick_block<float, MODE>(n->S.T) : pick_block<double, MODE>(n->S.T);
}

size_t net_smem(const net* n) {
    if (use_pull_kernel(n)) return pull_smem(n);
    return n->P.precision == 32 ? smem_bytes<float>(n->S) : smem_bytes<double>(n->S);
}

constexpr size_t kMaxSmem = 227 * 1024;
constexpr size_t kRatesSmem = 64 * sizeof(double);  // MODE kRates touches only the fixed header

size_t generic_smem(const net* n) {
    return n->P.precision == 32 ? smem_bytes<float>(n->S) : smem_bytes<double>(n->S);
}

int prepare_kernels(net* n) {
    // the generic kernels are prepared only where they can be launched: a network on the pull
    // path may have a flux array that does not fit (net_rates needs none of it)
    const size_t smem = generic_smem(n);
    if (smem <= kMaxSmem) {
        kernel_fn fns[3] = {pick_kernel<kAdaptive>(n), pick_kernel<kFixed>(n), pick_kernel<kRhs>(n)};
        for (kernel_fn f : fns)
            CUDA_TRY(cudaFuncSetAttribute(reinterpret_cast<const void*>(f),
                                          cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          static_cast<int>(smem)));
    }
    int nb = 0;
    if (use_pull_kernel(n)) {
        const void* f = reinterpret_cast<const void*>(pick_pull(n, true));
        const void* f2 = reinterpret_cast<const void*>(pick_pull(n, false));
        CUDA_TRY(cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      static_cast<int>(pull_smem(n))));
        CUDA_TRY(cudaFuncSetAttribute(f2, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      static_cast<int>(pull_smem(n))));
        CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, f, pull_block(n), pull_smem(n)));
        if (n->pull2 && pull2_store_of(n) != kinnet::kStoreSmem) {
            // the occupancy calculator answers 1 for a kernel that allocates tensor memory; the
            // residency is the smallest of the register, shared-memory and tensor-memory limits
            cudaFuncAttributes fa;
            CUDA_TRY(cudaFuncGetAttributes(&fa, f));
            const int warps = pull_block(n) / 32, regs = (fa.numRegs + 7) / 8 * 8;
            const int by_regs = 4 * (16384 / (32 * regs)) / warps;
            const int by_smem = static_cast<int>((228 * 1024) / (pull_smem(n) + fa.sharedSizeBytes + 1024));
            const int by_tmem = 512 / kinnet::pull2_tmem_cols(pull2_store_of(n), pull_block(n),
                                                              n->P.precision == 32 ? 4 : 8, n->pull2_spill);
            nb = std::min(by_regs, std::min(by_smem, by_tmem));
        }
    } else {
        CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(
            &nb, reinterpret_cast<const void*>(pick_kernel<kAdaptive>(n)), n->S.T, smem));
    }
    n->zones_per_sm = nb;
    return NET_OK;
}

int alloc_lanes(net* n, int cap) {
    for (int l = 0; l < kLanes; ++l) {
        if (n->lane_buf[l]) cudaFree(n->lane_buf[l]);
        n->lane_buf[l] = nullptr;
    }
    n->lane_cap = 0;
    for (int l = 0; l < kLanes; ++l) {
        CUDA_TRY(cudaMalloc(reinterpret_cast<void**>(&n->lane_buf[l]),
                            sizeof(int) * (static_cast<size_t>(kLaneHeader) + cap)));
        if (!n->lane_done[l]) CUDA_TRY(cudaEventCreateWithFlags(&n->lane_done[l], cudaEventDisableTiming));
    }
    n->lane_cap = cap;
    return NET_OK;
}

// Index of the lane this call may use, or -1 (the launch then runs in caller order: same bits).
// Called with n->mu held.  The rule that keeps concurrency off a lane:
//   * an eager call reuses the lane its stream used last (stream order serialises the two),
//     else takes a lane nobody holds, else steals the least recently used eager lane whose
//     last zone kernel has finished (lane_done, recorded by release_lane);
//   * a call under stream capture gets a lane of its own per (capture, stream): the graph keeps
//     pointers into it and may replay at any time, beside eager calls on the stream it was
//     captured on and beside any other graph, so the lane is never handed out again.  No event
//     query here: cudaEventQuery is not legal while a capture is under way.
int pick_lane(net* n, cudaStream_t stream, int zones) {
    if (zones > n->lane_cap) return -1;
    cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
    unsigned long long id = 0;
    if (cudaStreamGetCaptureInfo(stream, &st, &id) != cudaSuccess) {
        (void)cudaGetLastError();
        return -1;
    }
    if (st == cudaStreamCaptureStatusInvalidated) return -1;
    const bool capturing = (st == cudaStreamCaptureStatusActive);
    int pick = -1;
    for (int l = 0; l < kLanes && pick < 0; ++l)
        if (n->lane_used[l] && n->lane_stream[l] == stream && n->lane_captured[l] == capturing &&
            (!capturing || n->lane_capture[l] == id))
            pick = l;
    for (int l = 0; l < kLanes && pick < 0; ++l)
        if (!n->lane_used[l]) pick = l;
    if (pick < 0 && !capturing) {
        for (int l = 0; l < kLanes; ++l) {
            if (n->lane_captured[l] || (pick >= 0 && n->lane_tick[l] >= n->lane_tick[pick])) continue;
            if (cudaEventQuery(n->lane_done[l]) == cudaSuccess) pick = l;
            else (void)cudaGetLastError();  // cudaErrorNotReady: still running
        }
    }
    if (pick < 0) return -1;
    n->lane_used[pick] = true;
    n->lane_stream[pick] = stream;
    n->lane_captured[pick] = capturing;
    n->lane_capture[pick] = id;
    n->lane_tick[pick] = ++n->tick;
    return pick;
}

// Enqueue the counting sort of the zones by falling T9; returns the order (device) or NULL,
// and the lane it lives in (-1 = none).  Called with n->mu held from the first operation on the
// lane to release_lane behind the zone kernel, so that no other host thread can steal or share
// the lane in between.
int enqueue_order(net* n, int zones, const double* T9, cudaStream_t stream, const int** order, int* lane_out) {
    *order = nullptr;
    *lane_out = -1;
    if (zones < kOrderMinZones) return NET_OK;  // fewer zones than a couple of waves
    const int l = pick_lane(n, stream, zones);
    if (l < 0) {
        ++n->unsorted_calls;
        return NET_OK;
    }
    int* lane = n->lane_buf[l];
    const int ctas = (zones + kOrderZonesPerCta - 1) / kOrderZonesPerCta;
    CUDA_TRY(cudaMemsetAsync(lane, 0, sizeof(int) * kLaneHeader, stream));
    zone_hist_kernel<<<ctas, kOrderThreads, 0, stream>>>(T9, zones, lane);
    zone_scatter_kernel<<<ctas, kOrderThreads, 0, stream>>>(T9, zones, lane, lane + kOrderBuckets,
                                                           lane + kLaneHeader);
    CUDA_TRY(cudaGetLastError());
    ++n->sorted_calls;
    *order = lane + kLaneHeader;
    *lane_out = l;
    return NET_OK;
}

// Behind the zone kernel that read the lane: an eager lane becomes stealable once this event
// has completed.  A captured lane stays with its graph (and an event record would only add a
// node to it).
void release_lane(net* n, int l, cudaStream_t stream) {
    if (l < 0 || n->lane_captured[l]) return;
    if (cudaEventRecord(n->lane_done[l], stream) != cudaSuccess) (void)cudaGetLastError();
}

// Entry-point checks shared by everything that launches.
int check_net(const net* n) {
    if (!n) return fail(NET_EINVAL, "null net");
    if (!n->has_device) return fail(NET_ECUDA, "net has no device copy (net_create_host)");
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != n->device)
        return fail(NET_EINVAL, "the net_t lives on device " + std::to_string(n->device) +
                                    " but the calling thread's current device is " + std::to_string(dev));
    return NET_OK;
}

void fill_pull(const net* n, KPull& k) {
    const kinnet::PullSchedule& P = n->PS;
    std::memset(&k, 0, sizeof(k));
    k.N = n->S.N; k.M = n->S.M; k.nbs = P.nbs;
    for (int h = 0; h < kinnet::kPullHubs; ++h) k.hub[h] = P.hub[h];
    k.coef = n->D.coef_rxn;
    k.owner = n->D.p_owner;
    k.cnt = n->D.p_cnt;
    k.slot_rxn = n->D.p_slot_rxn;
    k.f1_pack = n->D.p_f1;
    k.f2_pack = n->D.p_f2;
    k.stair = n->pull2 ? n->pull2_stair : 0;
    k.agg_ptr = n->D.p_agg_ptr;
    k.agg_ent = n->D.p_agg_ent;
    k.kappa = n->P.kappa; k.eps_y = n->P.eps_y; k.y_floor = n->P.y_floor;
    k.growth = n->P.growth; k.max_steps = static_cast<int>(n->P.max_steps);
    k.method = n->P.method;
}

int launch_pull(net* n, int zones, KPull& k, void* stream) {
    pull_fn f = pick_pull(n, k.mode == kAdaptive);
    f<<<zones, pull_block(n), pull_smem(n), static_cast<cudaStream_t>(stream)>>>(k);
    CUDA_TRY(cudaGetLastError());
    return NET_OK;
}

// Device copies of the pull schedule.  Offsets are BYTE offsets into the YP
// table for elements of `elem` bytes; rows are padded to the largest kernel
// instantiation so every instantiation may read its full capacity.
int upload_pull(net* n) {
    const kinnet::PullSchedule& P = n->PS;
    const Schedule& S = n->S;
    const int T = P.T, M = S.M;
    const uint32_t elem = n->P.precision == 32 ? 4u : 8u;
    const int slots = S.rs * S.T;
    std::vector<double> coef(static_cast<size_t>(kinnet::kCoefRows) * M);
    for (int idx = 0; idx < slots; ++idx) {
        const int r = S.flux_rxn[idx];
        if (r < 0) continue;
        for (int c = 0; c < kinnet::kCoefRows; ++c)
            coef[static_cast<size_t>(c) * M + r] = S.coef[static_cast<size_t>(c) * slots + idx];
    }
    const uint32_t one_off = static_cast<uint32_t>(4 * T) * elem;
    // P-slot rows up to the largest capacity, then the N-slot rows
    constexpr int kRows = kinnet::kPullMaxSlots + kinnet::kPullNSlots;
    std::vector<uint32_t> cnt(T), f1(static_cast<size_t>(kRows / 2) * T),
        f2(static_cast<size_t>(kinnet::kPullMaxSlots2 / 2) * T);
    std::vector<int32_t> rxn(static_cast<size_t>(kRows) * T, -1);
    for (int t = 0; t < T; ++t) {
        cnt[t] = P.n_slots[t] | static_cast<uint32_t>(P.n_slots2[t]) << 8 |
                 static_cast<uint32_t>(P.n_nslots[t]) << 16;
        for (int e = 0; e < kinnet::kPullNSlots; ++e) {
            const int row = kinnet::kPullMaxSlots + e;
            rxn[static_cast<size_t>(row) * T + t] = P.nslot_rxn[static_cast<size_t>(e) * T + t];
            f1[static_cast<size_t>(row / 2) * T + t] |=
                (P.nslot_f1[static_cast<size_t>(e) * T + t] * elem) << (16 * (row & 1));
        }
        for (int e = 0; e < kinnet::kPullMaxSlots; ++e) {
            uint32_t off = one_off;
            if (e < P.slots) {
                off = P.slot_f1[static_cast<size_t>(e) * T + t] * elem;
                rxn[static_cast<size_t>(e) * T + t] = P.slot_rxn[static_cast<size_t>(e) * T + t];
            }
            f1[static_cast<size_t>(e / 2) * T + t] |= off << (16 * (e & 1));
        }
        for (int e = 0; e < kinnet::kPullMaxSlots2; ++e) {
            const uint32_t off =
                e < P.slots2 ? P.slot_f2[static_cast<size_t>(e) * T + t] * elem : one_off + 3 * elem;
            f2[static_cast<size_t>(e / 2) * T + t] |= off << (16 * (e & 1));
        }
    }
    int rc = upload(&n->D.coef_rxn, coef.data(), coef.size());
    if (rc == NET_OK) rc = upload(&n->D.p_owner, P.owner.data(), P.owner.size());
    if (rc == NET_OK) rc = upload(&n->D.p_cnt, cnt.data(), cnt.size());
    if (rc == NET_OK) rc = upload(&n->D.p_slot_rxn, rxn.data(), rxn.size());
    if (rc == NET_OK) rc = upload(&n->D.p_f1, f1.data(), f1.size());
    if (rc == NET_OK) rc = upload(&n->D.p_f2, f2.data(), f2.size());
    if (rc == NET_OK) rc = upload(&n->D.p_agg_ptr, P.agg_ptr.data(), P.agg_ptr.size());
    if (rc == NET_OK) rc = upload(&n->D.p_agg_ent, P.agg_ent.data(), P.agg_ent.size());
    return rc;
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
    k.kappa = n->P.kappa; k.eps_y = n->P.eps_y; k.y_floor = n->P.y_floor;
    k.growth = n->P.growth; k.max_steps = n->P.max_steps;
    k.method = n->P.method;
}

template <int MODE>
int launch(net* n, int zones, KParams& k, void* stream) {
    if (int rc = check_net(n)) return rc;
    if (zones < 0) return fail(NET_EINVAL, "zones < 0");
    if (zones == 0) return NET_OK;
    if (!k.T9 || !k.rho) return fail(NET_EINVAL, "null T9/rho");
    const size_t smem = (MODE == kRates) ? kRatesSmem : generic_smem(n);
    if (smem > kMaxSmem)
        return fail(NET_EINVAL, "the generic kernel's flux array does not fit one CTA's shared memory");
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
    if (n->P.method != 0 && n->P.method != 1) {
        delete n;
        return fail(NET_EINVAL, "method must be 0 (asymptotic) or 1 (QSS)");
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
    try {
        kinnet::build_pull_schedule(N, M, n_react, react, n_prod, prod, n->P.precision == 32 ? 4 : 8,
                                    n->PS);
    } catch (const std::bad_alloc&) {
        delete n;
        return fail(NET_ENOMEM, "out of host memory");
    }
    // two species per thread, when an instantiation covers it; up to 32 species one warp with
    // one species per lane is the better fit (0.57 against 0.82 ns per zone-substep at N = 32)
    if (n->P.kernel == 0 && n->PS.ok && N > 32) {
        kinnet::PullSchedule P2;
        try {
            kinnet::build_pull_schedule(N, M, n_react, react, n_prod, prod,
                                        n->P.precision == 32 ? 4 : 8, P2, (N + 63) / 64 * 64);
        } catch (const std::bad_alloc&) {
            delete n;
            return fail(NET_ENOMEM, "out of host memory");
        }
        int spill = 0;
        if (P2.ok && kinnet::pull2_supported(P2, &spill)) {
            n->PS = P2;
            n->pull2 = true;
            n->pull2_spill = spill;
            n->pull2_stair = kinnet::pull2_stair_class(P2);
        }
    }
    if (n->PS.ok && n->PS.nslots > 0 && !n->pull2) {
        n->PS.ok = false;  // only the two-species kernel is instantiated with N-slots
        n->PS.why = "reactions with two non-hub reactants need the two-species-per-thread kernel";
    }
    if (net_smem(n) > kMaxSmem) {
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
        if (rc == NET_OK && n->PS.ok) rc = upload_pull(n);
        if (rc == NET_OK) {
            n->has_device = true;
            rc = prepare_kernels(n);
        }
        if (rc == NET_OK) rc = alloc_lanes(n, kDefaultReserve);
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

// Device alias of a pinned (page-locked, mapped) host buffer, or NULL for anything else.
void* mapped_alias(const void* host) {
    if (!host) return nullptr;
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, host) != cudaSuccess) {
        cudaGetLastError();
        return nullptr;
    }
    return a.type == cudaMemoryTypeHost ? a.devicePointer : nullptr;
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
    p->host_chunk = 0;
    p->method = 0;
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
        cudaFree(n->D.coef_rxn); cudaFree(n->D.p_owner); cudaFree(n->D.p_cnt);
        cudaFree(n->D.p_slot_rxn); cudaFree(n->D.p_f1); cudaFree(n->D.p_f2);
        cudaFree(n->D.p_agg_ptr); cudaFree(n->D.p_agg_ent); cudaFree(n->D.bind);
        cudaFree(n->sT9); cudaFree(n->srho); cudaFree(n->sdt); cudaFree(n->sY);
        cudaFree(n->ssteps); cudaFree(n->sstatus);
        for (int l = 0; l < kLanes; ++l) {
            cudaFree(n->lane_buf[l]);
            if (n->lane_done[l]) cudaEventDestroy(n->lane_done[l]);
        }
        for (cudaStream_t s : n->host_stream)
            if (s) cudaStreamDestroy(s);
    }
    delete n;
}

int net_reserve(net_t* n, int max_zones) {
    if (int rc = check_net(n)) return rc;
    if (max_zones < 0) return fail(NET_EINVAL, "max_zones < 0");
    std::lock_guard<std::mutex> lock(n->mu);
    if (max_zones <= n->lane_cap) return NET_OK;
    for (int l = 0; l < kLanes; ++l)
        if (n->lane_captured[l])
            return fail(NET_EINVAL,
                        "net_reserve after a stream capture of net_integrate on this net_t: the captured "
                        "graph holds pointers into the launch-order workspaces that would be freed; "
                        "reserve before capturing");
    CUDA_TRY(cudaDeviceSynchronize());  // nothing in flight may still read the old workspaces
    return alloc_lanes(n, max_zones);
}

int net_launch_stats(net_t* n, long long* sorted_calls, long long* unsorted_calls, int* lanes_pinned) {
    if (!n) return fail(NET_EINVAL, "null net");
    std::lock_guard<std::mutex> lock(n->mu);
    if (sorted_calls) *sorted_calls = n->sorted_calls;
    if (unsorted_calls) *unsorted_calls = n->unsorted_calls;
    if (lanes_pinned) {
        *lanes_pinned = 0;
        for (int l = 0; l < kLanes; ++l) *lanes_pinned += n->lane_captured[l] ? 1 : 0;
    }
    return NET_OK;
}

int net_set_binding_energy(net_t* n, const double* B) {
    if (int rc = check_net(n)) return rc;
    if (!B) return fail(NET_EINVAL, "null argument");
    for (int i = 0; i < n->S.N; ++i)
        if (!std::isfinite(B[i])) return fail(NET_EINVAL, "non-finite binding energy");
    if (!n->D.bind) CUDA_TRY(cudaMalloc(reinterpret_cast<void**>(&n->D.bind), sizeof(double) * n->S.N));
    CUDA_TRY(cudaDeviceSynchronize());  // a launch in flight may still read the old table
    CUDA_TRY(cudaMemcpy(n->D.bind, B, sizeof(double) * n->S.N, cudaMemcpyHostToDevice));
    return NET_OK;
}

int net_integrate(net_t* n, int zones, const double* T9, const double* rho, void* Y,
                  double t_hydro, double* dt, int* n_steps, int* status, void* stream) {
    return net_integrate_energy(n, zones, T9, rho, Y, t_hydro, dt, n_steps, status, nullptr, stream);
}

int net_integrate_energy(net_t* n, int zones, const double* T9, const double* rho, void* Y,
                         double t_hydro, double* dt, int* n_steps, int* status, double* energy,
                         void* stream) {
    if (int rc = check_net(n)) return rc;
    if (energy && !n->D.bind)
        return fail(NET_EINVAL, "energy asked for before net_set_binding_energy");
    if (zones < 0) return fail(NET_EINVAL, "zones < 0");
    if (zones == 0) return NET_OK;
    if (!Y) return fail(NET_EINVAL, "null Y");
    if (!T9 || !rho) return fail(NET_EINVAL, "null T9/rho");
    if (!std::isfinite(t_hydro)) return fail(NET_EINVAL, "t_hydro is not finite");
    // sorted launches: lane choice, order kernels, zone kernel and the lane's event are one
    // host-side critical section per net_t (a few launches; nothing in it waits for the GPU)
    std::unique_lock<std::mutex> lock(n->mu, std::defer_lock);
    if (zones >= kOrderMinZones) lock.lock();
    const int* order = nullptr;
    int lane = -1;
    if (int rc = enqueue_order(n, zones, T9, static_cast<cudaStream_t>(stream), &order, &lane)) return rc;
    int rc;
    if (use_pull_kernel(n)) {
        KPull q;
        fill_pull(n, q);
        q.mode = kAdaptive;
        q.T9 = T9; q.rho = rho; q.Y = Y; q.dt = dt; q.n_steps = n_steps; q.status = status;
        q.t_hydro = t_hydro;
        q.bind = n->D.bind; q.energy = energy;
        q.order = order;
        rc = launch_pull(n, zones, q, stream);
    } else {
        KParams k;
        fill_params(n, k);
        k.T9 = T9; k.rho = rho; k.Y = Y; k.dt = dt; k.n_steps = n_steps; k.status = status;
        k.t_hydro = t_hydro;
        k.bind = n->D.bind; k.energy = energy;
        k.order = order;
        rc = launch<kAdaptive>(n, zones, k, stream);
    }
    release_lane(n, lane, static_cast<cudaStream_t>(stream));
    return rc;
}

// ---------------------------------------------------------------------------------------
// net_integrate_static (include/kinnet.h): net_integrate for hosts that may not allocate once
// they are running -- codes whose own pool owns all of HBM, time loops inside a capture or
// another region where cudaMalloc is illegal, drivers that must account for every byte up
// front.  The launch-order workspace (the only scratch of the adaptive path) is this array in
// the library image rather than a cudaMalloc'ed lane: [0, 1024) bucket counts, [1024, 2048)
// bucket cursors, then the order of up to NET_STATIC_MAX_ZONES zones; 264 KB on every GPU
// that loads the module, until the process exits.
//
// In HOST code the name g_static_order is only the host-side shadow of the symbol: it is not
// a device address, and a kernel handed `g_static_order` directly would fault or, on a system
// where the GPU can reach host memory, quietly scribble on the shadow.  Host code therefore
// asks the runtime for the device address once per device (static_order_ptr below) and
// passes that pointer to the kernels.
static __device__ __align__(256) int g_static_order[kLaneHeader + NET_STATIC_MAX_ZONES];

namespace {

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
int* g_static_ptr[kStaticMaxDevices] = {};  // device address of g_static_order, per device ordinal

// Device address of the array on `device`, which must be the calling thread's current device
// (check_net has verified that).  The first call per device does the lookup; later calls
// read the cache.
int static_order_ptr(int device, int** out) {
    *out = nullptr;
    if (device < 0 || device >= kStaticMaxDevices)
        return fail(NET_EINVAL, "net_integrate_static supports device ordinals 0.." +
                                    std::to_string(kStaticMaxDevices - 1));
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_order);
        if (e != cudaSuccess || !p) {
            (void)cudaGetLastError();
            return fail(NET_ECUDA, std::string("cudaGetSymbolAddress(static launch-order array): ") +
                                       (e != cudaSuccess ? cudaGetErrorString(e) : "null address"));
        }
        g_static_ptr[device] = static_cast<int*>(p);
    }
    *out = g_static_ptr[device];
    return NET_OK;
}

}  // namespace

int net_integrate_static(net_t* n, int zones, const double* T9, const double* rho, void* Y,
                         double t_hydro, double* dt, int* n_steps, int* status, void* stream) {
    if (int rc = check_net(n)) return rc;
    if (zones < 0) return fail(NET_EINVAL, "zones < 0");
    if (zones > NET_STATIC_MAX_ZONES)
        return fail(NET_EINVAL, "net_integrate_static: " + std::to_string(zones) +
                                    " zones exceed the static launch-order array (NET_STATIC_MAX_ZONES = " +
                                    std::to_string(NET_STATIC_MAX_ZONES) +
                                    "); split the batch into several calls on one stream");
    int* ws = nullptr;  // set-up on the first call per device, also for zones == 0
    if (int rc = static_order_ptr(n->device, &ws)) return rc;
    if (zones == 0) return NET_OK;
    if (!Y) return fail(NET_EINVAL, "null Y");
    if (!T9 || !rho) return fail(NET_EINVAL, "null T9/rho");
    if (!std::isfinite(t_hydro)) return fail(NET_EINVAL, "t_hydro is not finite");
    // hottest-first order of this batch in the static array: counts and cursors start at zero,
    // the scatter then writes every one of order[0, zones) -- nothing of the last call is read
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int ctas = (zones + kOrderZonesPerCta - 1) / kOrderZonesPerCta;
    CUDA_TRY(cudaMemsetAsync(ws, 0, sizeof(int) * kLaneHeader, s));
    zone_hist_kernel<<<ctas, kOrderThreads, 0, s>>>(T9, zones, ws);
    zone_scatter_kernel<<<ctas, kOrderThreads, 0, s>>>(T9, zones, ws, ws + kOrderBuckets, ws + kLaneHeader);
    CUDA_TRY(cudaGetLastError());
    if (use_pull_kernel(n)) {
        KPull q;
        fill_pull(n, q);
        q.mode = kAdaptive;
        q.T9 = T9; q.rho = rho; q.Y = Y; q.dt = dt; q.n_steps = n_steps; q.status = status;
        q.t_hydro = t_hydro;
        q.order = ws + kLaneHeader;
        return launch_pull(n, zones, q, stream);
    }
    KParams k;
    fill_params(n, k);
    k.T9 = T9; k.rho = rho; k.Y = Y; k.dt = dt; k.n_steps = n_steps; k.status = status;
    k.t_hydro = t_hydro;
    k.order = ws + kLaneHeader;
    return launch<kAdaptive>(n, zones, k, stream);
}

int net_integrate_fixed(net_t* n, int zones, const double* T9, const double* rho, void* Y,
                        double dt_fixed, long long n_steps, void* stream) {
    if (int rc = check_net(n)) return rc;
    if (zones > 0 && !Y) return fail(NET_EINVAL, "null Y");
    if (n_steps < 0 || n_steps > 2000000000LL) return fail(NET_EINVAL, "n_steps out of range [0, 2e9]");
    if (!std::isfinite(dt_fixed) || !(dt_fixed > 0.0))
        return fail(NET_EINVAL, "dt_fixed must be finite and > 0");
    if (use_pull_kernel(n)) {
        if (zones < 0) return fail(NET_EINVAL, "zones < 0");
        if (zones == 0) return NET_OK;
        if (!T9 || !rho) return fail(NET_EINVAL, "null T9/rho");
        KPull q;
        fill_pull(n, q);
        q.mode = kFixed;
        q.T9 = T9; q.rho = rho; q.Y = Y;
        q.dt_fixed = dt_fixed; q.n_fixed = static_cast<int>(n_steps);
        return launch_pull(n, zones, q, stream);
    }
    KParams k;
    fill_params(n, k);
    k.T9 = T9; k.rho = rho; k.Y = Y;
    k.dt_fixed = dt_fixed; k.n_fixed = n_steps;
    return launch<kFixed>(n, zones, k, stream);
}

int net_rates(net_t* n, int zones, const double* T9, const double* rho, double* R, void* stream) {
    if (int rc = check_net(n)) return rc;
    if (zones > 0 && !R) return fail(NET_EINVAL, "null R");
    KParams k;
    fill_params(n, k);
    k.T9 = T9; k.rho = rho; k.Rout = R;
    return launch<kRates>(n, zones, k, stream);
}

int net_rhs(net_t* n, int zones, const double* T9, const double* rho, const void* Y, void* Fplus,
            void* Fminus, void* stream) {
    if (int rc = check_net(n)) return rc;
    if (zones > 0 && (!Y || !Fplus || !Fminus)) return fail(NET_EINVAL, "null Y/Fplus/Fminus");
    if (use_pull_kernel(n)) {
        if (zones < 0) return fail(NET_EINVAL, "zones < 0");
        if (zones == 0) return NET_OK;
        if (!T9 || !rho) return fail(NET_EINVAL, "null T9/rho");
        KPull q;
        fill_pull(n, q);
        q.mode = kRhs;
        q.T9 = T9; q.rho = rho; q.Y = const_cast<void*>(Y); q.Fplus = Fplus; q.Fminus = Fminus;
        return launch_pull(n, zones, q, stream);
    }
    KParams k;
    fill_params(n, k);
    k.T9 = T9; k.rho = rho; k.Y = const_cast<void*>(Y); k.Fplus = Fplus; k.Fminus = Fminus;
    return launch<kRhs>(n, zones, k, stream);
}

// Host-buffer path (what crosses the link per network, and
// what the CPU and the link do while the GPU integrates).
//   * Pinned buffers: ZERO-COPY.  The zone kernel itself reads a zone's T9, rho, dt and
//     abundances from the mapped host buffers when the zone starts (S6 in) and writes them back
//     when it ends (S6 out): one launch over the whole batch in the global hottest-first order,
//     every transfer overlapped with the integration of the other zones, no staging copy.
//   * Anything else (pageable memory): staged through net-owned device scratch in chunks over
//     three internal streams; the launch order then applies within a chunk.  A copy between
//     pageable memory and the device is not asynchronous to the host: the upload returns once
//     the data sit in the driver's staging buffer, the download only when it has finished.  So
//     the loop enqueues the upload and the kernels of chunk c BEFORE the download of chunk
//     c-1: while the host thread sits in that download, the GPU already integrates chunk c, and
//     the download of c-1 overlaps it.  (In the opposite order every chunk ran alone: upload,
//     kernels, download, GPU idle during the copies.)  The call returns when all but the last
//     download have finished, i.e. it is asynchronous only for pinned buffers.
int net_integrate_host_async(net_t* n, int zones, const double* T9, const double* rho, void* Y,
                             double t_hydro, double* dt, int* n_steps, int* status) {
    if (int rc = check_net(n)) return rc;
    if (zones < 0) return fail(NET_EINVAL, "zones < 0");
    if (zones == 0) return NET_OK;
    if (!T9 || !rho || !Y) return fail(NET_EINVAL, "null T9/rho/Y");
    {
        std::lock_guard<std::mutex> lock(n->mu);
        if (n->host_in_flight)
            return fail(NET_EINVAL, "net_integrate_host_async: a batch is in flight on this net_t "
                                    "(its scratch and streams are shared): call net_wait first");
        n->host_in_flight = true;  // until net_wait, also when this call fails half-way
    }
    for (cudaStream_t& s : n->host_stream)
        if (!s) CUDA_TRY(cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking));
    if (n->P.host_chunk >= 0) {  // < 0 forces the staged path
        void* aT9 = mapped_alias(T9);
        void* arho = mapped_alias(rho);
        void* aY = mapped_alias(Y);
        void* adt = mapped_alias(dt);
        void* asteps = mapped_alias(n_steps);
        void* astatus = mapped_alias(status);
        if (aT9 && arho && aY && (adt || !dt) && (asteps || !n_steps) && (astatus || !status))
            return net_integrate(n, zones, static_cast<const double*>(aT9), static_cast<const double*>(arho),
                                 aY, t_hydro, static_cast<double*>(adt), static_cast<int*>(asteps),
                                 static_cast<int*>(astatus), n->host_stream[0]);
    }
    const size_t ysz = (n->P.precision == 32 ? sizeof(float) : sizeof(double)) * (size_t)n->S.N;
    if (zones > n->scratch_zones) {
        for (cudaStream_t s : n->host_stream) CUDA_TRY(cudaStreamSynchronize(s));
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
    const int chunk = n->P.host_chunk != 0
                          ? std::abs(n->P.host_chunk)
                          : std::max(kHostMinChunk, (zones + kHostMaxChunks - 1) / kHostMaxChunks);
    auto download = [&](int lo, int m, cudaStream_t s) -> int {
        char* Yh = static_cast<char*>(Y) + ysz * lo;
        char* Yd = static_cast<char*>(n->sY) + ysz * lo;
        CUDA_TRY(cudaMemcpyAsync(Yh, Yd, ysz * m, cudaMemcpyDeviceToHost, s));
        if (dt) CUDA_TRY(cudaMemcpyAsync(dt + lo, n->sdt + lo, sizeof(double) * m, cudaMemcpyDeviceToHost, s));
        if (n_steps)
            CUDA_TRY(cudaMemcpyAsync(n_steps + lo, n->ssteps + lo, sizeof(int) * m, cudaMemcpyDeviceToHost, s));
        if (status)
            CUDA_TRY(cudaMemcpyAsync(status + lo, n->sstatus + lo, sizeof(int) * m, cudaMemcpyDeviceToHost, s));
        return NET_OK;
    };
    int c = 0, prev_lo = -1, prev_m = 0;
    cudaStream_t prev_s = nullptr;
    for (int lo = 0; lo < zones; lo += chunk, ++c) {
        const int m = std::min(chunk, zones - lo);
        cudaStream_t s = n->host_stream[c % kHostStreams];
        char* Yh = static_cast<char*>(Y) + ysz * lo;
        char* Yd = static_cast<char*>(n->sY) + ysz * lo;
        CUDA_TRY(cudaMemcpyAsync(n->sT9 + lo, T9 + lo, sizeof(double) * m, cudaMemcpyHostToDevice, s));
        CUDA_TRY(cudaMemcpyAsync(n->srho + lo, rho + lo, sizeof(double) * m, cudaMemcpyHostToDevice, s));
        CUDA_TRY(cudaMemcpyAsync(Yd, Yh, ysz * m, cudaMemcpyHostToDevice, s));
        if (dt) CUDA_TRY(cudaMemcpyAsync(n->sdt + lo, dt + lo, sizeof(double) * m, cudaMemcpyHostToDevice, s));
        else CUDA_TRY(cudaMemsetAsync(n->sdt + lo, 0, sizeof(double) * m, s));
        if (int rc = net_integrate(n, m, n->sT9 + lo, n->srho + lo, Yd, t_hydro, n->sdt + lo,
                                   n->ssteps + lo, n->sstatus + lo, s))
            return rc;
        // chunk c is queued: now the download of chunk c-1 (which blocks the host for pageable
        // buffers) cannot leave the GPU idle
        if (prev_lo >= 0)
            if (int rc = download(prev_lo, prev_m, prev_s)) return rc;
        prev_lo = lo; prev_m = m; prev_s = s;
    }
    if (prev_lo >= 0)
        if (int rc = download(prev_lo, prev_m, prev_s)) return rc;
    return NET_OK;
}

int net_wait(net_t* n) {
    if (int rc = check_net(n)) return rc;
    cudaError_t first = cudaSuccess;
    for (cudaStream_t s : n->host_stream)
        if (s) {
            const cudaError_t e = cudaStreamSynchronize(s);
            if (first == cudaSuccess) first = e;
        }
    {
        std::lock_guard<std::mutex> lock(n->mu);
        n->host_in_flight = false;
    }
    if (first != cudaSuccess) return fail(NET_ECUDA, std::string("net_wait: ") + cudaGetErrorString(first));
    return NET_OK;
}

int net_integrate_host(net_t* n, int zones, const double* T9, const double* rho, void* Y,
                       double t_hydro, double* dt, int* n_steps, int* status) {
    if (int rc = net_integrate_host_async(n, zones, T9, rho, Y, t_hydro, dt, n_steps, status)) {
        const std::string keep = g_last_error;  // drain what was enqueued, report the first error
        if (n && n->has_device && keep.find("a batch is in flight") == std::string::npos) net_wait(n);
        g_last_error = keep;
        return rc;
    }
    return net_wait(n);
}

int net_schedule_info(const net_t* n, net_schedule_info_t* info) {
    if (!n || !info) return fail(NET_EINVAL, "null argument");
    const Schedule& S = n->S;
    info->n_species = S.N;
    info->n_reactions = S.M;
    info->threads = use_pull_kernel(n) ? pull_block(n) : S.T;
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
    info->kernel = use_pull_kernel(n) ? (n->pull2 ? 2 : 1) : 0;
    info->pull_ok = n->PS.ok ? 1 : 0;
    info->pull_hubs = n->PS.nbs;
    info->pull_slots = n->PS.slots;
    info->pull_slots2 = n->PS.slots2;
    info->pull_agg_max = n->PS.agg_max;
    info->pull_wavefronts = static_cast<int>(n->PS.conflict_wavefronts);
    info->pull_wavefronts_ideal = static_cast<int>(n->PS.ideal_wavefronts);
    info->pull_threads = n->PS.ok ? n->PS.T : 0;
    info->pull_nslots = n->PS.ok ? n->PS.nslots : 0;
    info->pull_stair = n->pull2 ? n->pull2_stair : 0;
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
    } else if (key.rfind("pull_", 0) == 0) {
        const kinnet::PullSchedule& P = n->PS;
        if (!P.ok) return fail(NET_EINVAL, "no pull schedule for this network: " + P.why);
        if (key == "pull_hub") {
            const std::vector<int32_t> hubs(P.hub, P.hub + P.nbs);
            emit(hubs, 1, 1);
        } else if (key == "pull_owner") emit(P.owner, 1, 1);
        else if (key == "pull_n_slots") emit(P.n_slots, 1, 1);
        else if (key == "pull_n_slots2") emit(P.n_slots2, 1, 1);
        else if (key == "pull_slot_rxn") emit(P.slot_rxn, 1, 1);
        else if (key == "pull_slot_f1") emit(P.slot_f1, 1, 1);
        else if (key == "pull_slot_f2") emit(P.slot_f2, 1, 1);
        else if (key == "pull_n_nslots") emit(P.n_nslots, 1, 1);
        else if (key == "pull_nslot_rxn") emit(P.nslot_rxn, 1, 1);
        else if (key == "pull_nslot_f1") emit(P.nslot_f1, 1, 1);
        else if (key == "pull_agg_ptr") emit(P.agg_ptr, 1, 1);
        else if (key == "pull_agg_ent") emit(P.agg_ent, 1, 1);
        else return fail(NET_EINVAL, "unknown schedule table '" + key + "'");
    } else return fail(NET_EINVAL, "unknown schedule table '" + key + "'");
    if (out && cap < count) return fail(NET_EINVAL, "output buffer too small");
    return count;
}

const char* net_last_error(void) { return g_last_error.c_str(); }

}  // extern "C"
