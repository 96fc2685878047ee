// zone_pull2.cuh -- the pull kernel with TWO species per thread (internal).
//
// Same method, tables and shared-memory protocol as zone_pull.cuh; what changes is
// the mapping: the pull schedule is compiled for 2*TB "virtual threads" and physical
// thread (warp w, lane l) plays the virtual threads (w, l) -- side a, the rows with
// many incoming reactions -- and (2*NW-1-w, l) -- side b, the short rows.  Why: one
// sub-step is a chain of dependent FP64 operations at 8 clk each (profiles/r01d),
// and a warp issues in order, so with one species per thread most issue slots of a
// warp wait on its own previous instruction.  Two species per thread are two
// independent chains in every phase (rate sums, gathers, update), the hub-row
// shares of the two are added before ONE butterfly, and the redundant finalize runs
// in NW = TB/32 warps instead of twice as many.
#pragma once
#include <type_traits>

#include "zone_pull.cuh"

namespace kinnet {

// The G coefficients (hub F+ rows, C[10..18]) of both species live in shared memory: read
// once per sub-step, conflict-free, they would otherwise hold 36 registers of the 168
// that let four CTAs share an SM (16 K registers per scheduler: 3 warps of <= 168).
constexpr int kPull2SmemCoefs = 9;

// Where a thread keeps what it re-reads every sub-step (the loop-invariant coefficients):
//   kStoreSmem    G and the spilled slot rates in shared memory, K in registers (block sizes < 96: up to
//                 12 CTAs per SM are too many for the tensor-memory columns)
//   kStoreTmemK   K, G and up to 12 spilled rates in tensor memory (128 columns per lane group): no
//                 coefficient in shared memory, none in registers beyond 20 slot rates.  With N-slots too
//   kStoreTmemKs  160-thread blocks, three per SM, whose two lane groups leave each thread 64 columns:
//                 G and 12 rates in tensor memory, K in shared memory (128 registers)
//   kStoreTmem    ... and with N-slots K in registers (168 registers; the 128-register build spills)
enum Pull2Store { kStoreSmem = 0, kStoreTmem = 1, kStoreTmemKs = 2, kStoreTmemK = 3 };
__host__ __device__ constexpr int pull2_store(int TB, int nslots) {
    return TB < 96 ? kStoreSmem : TB == 160 ? (nslots > 0 ? kStoreTmem : kStoreTmemKs) : kStoreTmemK;
}
// Tensor memory (TMEM, 512 columns x 128 lanes x 32 bit per SM) as a LANE-PRIVATE store: tcgen05.ld
// reaches a warp's own 32 lanes in ~12 cycles and does not touch the shared-memory pipe, which was this
// kernel's busiest unit (measured: a saturated LDS stream loses nothing to a concurrent tcgen05.ld
// stream).  Layout of a thread's columns under kStoreTmemK, in values of `real`, chunks of 8 values = one
// tcgen05.ld each, ordered so that every chunk completes sub-expressions of the rate sums:
//   [ 0.. 8)  K of side a: C0 C1 C4 C5 C6 C2 C7 C3     [ 8..16)  C8 C9, then G0 G3 G1 G5 G2 G7 of side a
//   [16..32)  the same of side b                      [32..38)  G4 G6 G8 of side a, of side b; [38..40) unused
//   [40..)    spilled slot rates
// The first two chunks of the NEXT sub-step are issued right after barrier B and land during the finalize.
constexpr int kPull2TmemRateBase = 40;
// spilled slot rates per thread that tensor memory takes (the rest stay in shared memory)
__host__ __device__ constexpr int pull2_tmem_rates(int store, int TB, int real_bytes, int spill) {
    (void)TB, (void)real_bytes;
    const int cap = store == kStoreSmem ? 0 : 12;
    return spill < cap ? spill : cap;
}
// columns per thread (32-bit words), and what one CTA allocates
__host__ __device__ constexpr int pull2_tmem_words(int store, int TB, int real_bytes, int spill) {
    const int nrt = pull2_tmem_rates(store, TB, real_bytes, spill);
    return (real_bytes / 4) * (store == kStoreTmemK ? kPull2TmemRateBase + nrt : 2 * kPull2SmemCoefs + nrt);
}
__host__ __device__ constexpr int pull2_tmem_cols(int store, int TB, int real_bytes, int spill) {
    const int need = pull2_tmem_words(store, TB, real_bytes, spill) * ((TB / 32 + 3) / 4);
    int cols = 32;
    while (cols < need) cols *= 2;
    return cols;
}

// spill = slot rates of both sides kept out of registers
template <typename real>
__host__ __device__ inline size_t pull2_smem_bytes(int TB, int M, int spill, int store) {
    const int nrt = pull2_tmem_rates(store, TB, static_cast<int>(sizeof(real)), spill);
    const size_t coef = static_cast<size_t>(spill - nrt) * TB +
                        (store == kStoreSmem     ? static_cast<size_t>(kPull2SmemCoefs) * 2 * TB
                         : store == kStoreTmemKs ? static_cast<size_t>(kPullCoefs - kPull2SmemCoefs) * 2 * TB
                                                 : 0);
    return 32 * sizeof(double) + sizeof(real) * (static_cast<size_t>(TB / 32) * 8 + 8 * TB + 4 + coef) +
           sizeof(double) * static_cast<size_t>(M);
}

// Staircase of live slots (branch-free block sizes): species are dealt to the virtual threads by falling
// in-degree, so warp w's side a (virtual warp w) needs fewer slots the larger w, its side b (virtual warp
// 2 NW - 1 - w) more.  When the compiled schedule fits under
//   side a: max(cap_a - 4 w, 12)        side b: max(cap_b - 4 (NW - 1 - w), 4)
// (hub150: 20 + 4, 16 + 8, 12 + 12 live slots in its three warps, against 20 + 12 in every warp), each warp
// runs its own copy of the sub-step loop with those compile-time capacities (KPull.stair).
__host__ __device__ constexpr int pull2_stair_a(int cap_a, int w) { return cap_a - 4 * w > 12 ? cap_a - 4 * w : 12; }
__host__ __device__ constexpr int pull2_stair_b(int cap_b, int nw, int w) {
    return cap_b - 4 * (nw - 1 - w) > 4 ? cap_b - 4 * (nw - 1 - w) : 4;
}
// KPull.stair: 0 = side a does not fit (every warp runs the instantiation's capacities); else bit 0 set, bit 1 =
// warp 0 plays no species on side b (N <= 32 (2 NW - 1)): its copy of the loop then has none of that side's
// work (capacity 0); bit 8 + w = warp w's side b does not fit its step and runs the full capacity
int pull2_stair_class(const PullSchedule& P);
// method = net_params_t.method (1 = the QSS instantiations)
pull_fn pull2_kernel_f64_adaptive(const PullSchedule& P, int method);
pull_fn pull2_kernel_f64_fixed(const PullSchedule& P, int method);
pull_fn pull2_kernel_f32_adaptive(const PullSchedule& P, int method);
pull_fn pull2_kernel_f32_fixed(const PullSchedule& P, int method);
// slots of the two sides of a schedule compiled for virtual threads; false when no
// instantiation covers it (the caller then compiles the one-species schedule)
bool pull2_supported(const PullSchedule& P, int* spill);

#ifdef KINNET_PULL_INSTANTIATE

// ---- tcgen05.ld / st on the calling warp's own lanes (32x32b: lane i <-> thread i of the warp)
#define KINNET_TM_LD(N, OUTS, ...)                                                                   \
    __device__ __forceinline__ void tm_ld(uint32_t (&r)[N], uint32_t a) {                           \
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x" #N ".b32 {" OUTS "}, [%" #N "];" : __VA_ARGS__ : "r"(a)); \
    }                                                                                               \
    /* the wait names the registers so that no use of them can be scheduled above it */            \
    __device__ __forceinline__ void tm_wait(uint32_t (&r)[N]) {                                     \
        asm volatile("tcgen05.wait::ld.sync.aligned;" : KINNET_TM_INOUT##N(r)::"memory");           \
    }                                                                                               \
    __device__ __forceinline__ void tm_touch(uint32_t (&r)[N]) { asm volatile("" : KINNET_TM_INOUT##N(r)); }
#define KINNET_TM_INOUT1(r) "+r"(r[0])
#define KINNET_TM_INOUT2(r) KINNET_TM_INOUT1(r), "+r"(r[1])
#define KINNET_TM_INOUT4(r) KINNET_TM_INOUT2(r), "+r"(r[2]), "+r"(r[3])
#define KINNET_TM_INOUT8(r) KINNET_TM_INOUT4(r), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7])
#define KINNET_TM_INOUT16(r)                                                                         \
    KINNET_TM_INOUT8(r), "+r"(r[8]), "+r"(r[9]), "+r"(r[10]), "+r"(r[11]), "+r"(r[12]), "+r"(r[13]), "+r"(r[14]), "+r"(r[15])
KINNET_TM_LD(1, "%0", "=r"(r[0]))
KINNET_TM_LD(2, "%0,%1", "=r"(r[0]), "=r"(r[1]))
KINNET_TM_LD(4, "%0,%1,%2,%3", "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]))
KINNET_TM_LD(8, "%0,%1,%2,%3,%4,%5,%6,%7", "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]),
             "=r"(r[6]), "=r"(r[7]))
KINNET_TM_LD(16, "%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15", "=r"(r[0]), "=r"(r[1]), "=r"(r[2]),
             "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]),
             "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]))
#undef KINNET_TM_LD

__device__ __forceinline__ void tm_st(uint32_t a, double v) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1,%2};" ::"r"(a), "r"(__double2loint(v)),
                 "r"(__double2hiint(v))
                 : "memory");
}
__device__ __forceinline__ void tm_st(uint32_t a, float v) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(a), "r"(__float_as_uint(v)) : "memory");
}
__device__ __forceinline__ double tm_val(uint32_t lo, uint32_t hi) {
    return __hiloint2double(static_cast<int>(hi), static_cast<int>(lo));
}
// the nine G coefficients of both sides of a thread: columns [0, 9 W) and [9 W, 18 W), W words per value
__device__ __forceinline__ void tm_load_g(double (&Ga)[9], double (&Gb)[9], uint32_t a) {
    uint32_t u[16], v[16], w[4];
    tm_ld(u, a);
    tm_ld(v, a + 16);
    tm_ld(w, a + 32);
    tm_wait(u);
    tm_touch(v);
    tm_touch(w);
#pragma unroll
    for (int j = 0; j < 8; ++j) Ga[j] = tm_val(u[2 * j], u[2 * j + 1]);
    Ga[8] = tm_val(v[0], v[1]);
#pragma unroll
    for (int j = 0; j < 7; ++j) Gb[j] = tm_val(v[2 + 2 * j], v[3 + 2 * j]);
    Gb[7] = tm_val(w[0], w[1]);
    Gb[8] = tm_val(w[2], w[3]);
}
__device__ __forceinline__ void tm_load_g(float (&Ga)[9], float (&Gb)[9], uint32_t a) {
    uint32_t u[16], v[2];
    tm_ld(u, a);
    tm_ld(v, a + 16);
    tm_wait(u);
    tm_touch(v);
#pragma unroll
    for (int j = 0; j < 9; ++j) Ga[j] = __uint_as_float(u[j]);
#pragma unroll
    for (int j = 0; j < 7; ++j) Gb[j] = __uint_as_float(u[9 + j]);
    Gb[7] = __uint_as_float(v[0]);
    Gb[8] = __uint_as_float(v[1]);
}
// four consecutive spilled rates
__device__ __forceinline__ void tm_load4(double (&x)[4], uint32_t a) {
    uint32_t u[8];
    tm_ld(u, a);
    tm_wait(u);
#pragma unroll
    for (int j = 0; j < 4; ++j) x[j] = tm_val(u[2 * j], u[2 * j + 1]);
}
__device__ __forceinline__ void tm_load4(float (&x)[4], uint32_t a) {
    uint32_t u[4];
    tm_ld(u, a);
    tm_wait(u);
#pragma unroll
    for (int j = 0; j < 4; ++j) x[j] = __uint_as_float(u[j]);
}
// eight values whose tcgen05.ld was issued earlier into u, v (the sub-step's first two chunks)
__device__ __forceinline__ void tm_take8x2(double (&x)[8], double (&y)[8], uint32_t (&u)[16], uint32_t (&v)[16]) {
    tm_wait(u);
    tm_touch(v);
#pragma unroll
    for (int j = 0; j < 8; ++j) x[j] = tm_val(u[2 * j], u[2 * j + 1]), y[j] = tm_val(v[2 * j], v[2 * j + 1]);
}
__device__ __forceinline__ void tm_take8x2(float (&x)[8], float (&y)[8], uint32_t (&u)[8], uint32_t (&v)[8]) {
    tm_wait(u);
    tm_touch(v);
#pragma unroll
    for (int j = 0; j < 8; ++j) x[j] = __uint_as_float(u[j]), y[j] = __uint_as_float(v[j]);
}
// eight consecutive values
__device__ __forceinline__ void tm_load8(double (&x)[8], uint32_t a) {
    uint32_t u[16];
    tm_ld(u, a);
    tm_wait(u);
#pragma unroll
    for (int j = 0; j < 8; ++j) x[j] = tm_val(u[2 * j], u[2 * j + 1]);
}
__device__ __forceinline__ void tm_load8(float (&x)[8], uint32_t a) {
    uint32_t u[8];
    tm_ld(u, a);
    tm_wait(u);
#pragma unroll
    for (int j = 0; j < 8; ++j) x[j] = __uint_as_float(u[j]);
}

// One side (one species) of a thread: everything that is loop invariant.
template <typename real, int CP, int CPR, int J2, int NS>
struct PullSide {
    real R[CPR > 0 ? CPR : 1];
    real C[kPullCoefs - kPull2SmemCoefs];  // K by class; G0, Gx are in shared memory
    uint32_t f1[(CP + NS) / 2], f2[J2 / 2];  // P-slot offsets, then the N-slot offsets
    int wn, wn2, wnn, own;
    uint32_t s_pub;
};

// k = F-/y and the six hub-row shares of one species (see zone_pull.cuh)
template <typename real>
__device__ __forceinline__ void pull_rate_sums(const real (&C)[kPullCoefs - kPull2SmemCoefs],
                                               const real (&G)[kPull2SmemCoefs], real y, real p1, real p2,
                                               real p3, real yh0, real yh1, real yh2, real& k,
                                               real (&share)[6]) {
    real e0 = fma(C[4], yh0, C[1]);
    e0 = fma(C[5], yh1, e0);
    e0 = fma(C[6], yh2, e0);
    real e1 = fma(C[7], yh1, C[2]);
    e1 = fma(C[8], yh2, e1);
    const real e2 = fma(C[9], yh2, C[3]);
    k = fma(yh0, e0, C[0]);
    k = fma(yh1, e1, k);
    k = fma(yh2, e2, k);
    const real m0 = fma(C[4], yh0, e0);
    real m1 = fma(C[5], yh0, e1);
    m1 = fma(C[7], yh1, m1);
    real m2 = fma(C[6], yh0, e2);
    m2 = fma(C[8], yh1, m2);
    m2 = fma(C[9], yh2, m2);
    real g0 = fma(G[3], yh1, G[0]);
    g0 = fma(G[4], yh2, g0);
    real g1 = fma(G[5], yh0, G[1]);
    g1 = fma(G[6], yh2, g1);
    real g2 = fma(G[7], yh0, G[2]);
    g2 = fma(G[8], yh1, g2);
    share[0] = y * g0;
    share[1] = y * g1;
    share[2] = y * g2;
    share[3] = p1 * m0;
    share[4] = p2 * m1;
    share[5] = p3 * m2;
}

// warp w runs f with its step of the staircase as compile-time capacities
template <int NW, int CPA, int CPB, int W = 0, typename F>
__device__ __forceinline__ bool stair_dispatch(int warp, int cls, F& f) {
    if constexpr (W + 1 < NW) {
        if (warp != W) return stair_dispatch<NW, CPA, CPB, W + 1>(warp, cls, f);
    }
    if constexpr (W == 0) {
        if (cls & 2) return f(std::integral_constant<int, pull2_stair_a(CPA, 0)>{}, std::integral_constant<int, 0>{});
    }
    if constexpr (pull2_stair_b(CPB, NW, W) < CPB) {
        if (cls >> (8 + W) & 1) return f(std::integral_constant<int, pull2_stair_a(CPA, W)>{}, std::integral_constant<int, CPB>{});
    }
    return f(std::integral_constant<int, pull2_stair_a(CPA, W)>{}, std::integral_constant<int, pull2_stair_b(CPB, NW, W)>{});
}

// Twelve warps per SM -- three per scheduler, whose 16 K registers then give each thread
// 168 (ptxas derives exactly that from the launch bounds): four 96-thread CTAs, three 128-thread,
// two 192-thread ones.  Five 96-thread CTAs at 128 registers run as fast on a full batch (252k
// zone-networks/s on configs[3] either way, profiles/r02b), but the 168-register build does not spill, and
// its sub-step is 17 % shorter in a lone CTA (0.72 us against 0.87 us): every batch that does not fill
// the SMs gains.  160-thread blocks, whose K stays in shared memory, run three CTAs at 128 registers.
// With fp32 state the rates take half the registers: 128 registers, four warps per scheduler, five
// 96-thread CTAs (318k zone-networks/s on configs[3] at that commit, 365k with the branch-free loop).
// NS = 4 compiles the N-slots in (networks with heavy + heavy reactions, schedule.h): four more
// gathers per side into k, skipped by the warps none of whose species has one, and the hub
// owners' own P-slot sums (heavy + heavy reactions that emit a hub) joined to their rows.
// QSS compiles the quasi-steady-state variant of the update in (net_params_t.method = 1); a
// run-time switch costs the default kernel 6 % (registers), so it is an instantiation.
// ST: where the coefficients live (Pull2Store; = pull2_store(TB, NS)).
template <typename real, int TB, int CPA, int SPA, int CPB, int SPB, int J2, int NS, bool ADAPT, bool QSS, int ST>
__global__ void __launch_bounds__(TB, (sizeof(real) == 4 || ST == kStoreTmemKs ? 480 : 384) / TB)
    zone_kernel_pull2(const KPull p) {
    static_assert(ST == pull2_store(TB, NS), "store mode");
    constexpr bool TM = ST != kStoreSmem;   // tensor memory in use
    constexpr bool KT = ST == kStoreTmemK;  // ... for K too
    constexpr bool BRF = TB <= 128;         // branch-free gathers (see KINNET_LOADS)
    static_assert(CPA % 4 == 0 && CPB % 4 == 0 && SPA % 4 == 0 && SPA < CPA && SPB % 4 == 0 && SPB < CPB,
                  "slot capacities");
    static_assert(NS == 0 || NS == kPullNSlots, "N-slot capacity");
    constexpr int T = TB, NW = TB / 32, TV = 2 * TB;  // physical threads, warps; virtual threads
    constexpr int CPRA = CPA - SPA, CPRB = CPB - SPB;  // slots whose rate stays in a register
    constexpr uint32_t SZ = sizeof(real);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int N = p.N, M = p.M, nbs = p.nbs;
    const int z = p.order ? p.order[blockIdx.x] : blockIdx.x;
    const int va = tid, vb = (2 * NW - 1 - warp) * 32 + lane;  // the two virtual threads played here

    double* redq = reinterpret_cast<double*>(smem_raw);       // [32] per-warp q maxima, [16..18] own terms
    real* red = reinterpret_cast<real*>(redq + 32);           // [NW][8] per-warp hub-row sums
    real* YP = red + NW * 8;                                  // [4][TV] published products, then 1
    constexpr int NRX = SPA + SPB + 2 * NS;                   // slot rates kept out of registers, per thread
    real* Rx = YP + 4 * TV + 4;                               // [NRX - NRT][T] spilled slot rates, N-slot rates
    constexpr int NRT = pull2_tmem_rates(ST, TB, sizeof(real), NRX);  // rate rows in tensor memory
    real* Gs = Rx + (NRX - NRT) * T;                          // [9][TV] G0, Gx of every virtual thread      (not TM)
    constexpr int NK = kPullCoefs - kPull2SmemCoefs;          // K coefficients per species
    constexpr bool KS = ST == kStoreTmemKs;                   // K in shared memory instead of registers
    real* Ks = Gs;                                            // [NK][TV] K of every virtual thread          (KS)
    double* Rbuf = reinterpret_cast<double*>(Gs + (TM ? (KS ? NK * TV : 0) : kPull2SmemCoefs * TV));  // [M] rates, set-up only
    // tensor-memory columns of a thread (TM): G of side a, G of side b, then the NRT rates; KT: see
    // pull2_store
    constexpr uint32_t RW = sizeof(real) / 4, TMC = pull2_tmem_words(ST, TB, sizeof(real), NRX);
    constexpr uint32_t TM_COLS = pull2_tmem_cols(ST, TB, sizeof(real), NRX);  // what the CTA allocates
    constexpr uint32_t TM_RATE0 = RW * (KT ? kPull2TmemRateBase : 2 * kPull2SmemCoefs);  // first rate column
    __shared__ uint32_t tm_slot;
    uint32_t s_redq;
    asm volatile("mov.u32 %0, %1;"
                 : "=r"(s_redq)
                 : "r"(static_cast<uint32_t>(__cvta_generic_to_shared(smem_raw))));
    const uint32_t s_red = s_redq + 32 * 8;
    const uint32_t s_YP = s_red + NW * 8 * SZ;
    const uint32_t s_Rx = s_YP + (4 * TV + 4) * SZ + tid * SZ;
    const uint32_t s_own = s_redq + 16 * 8;   // [3] own-consumption terms of the hub owners
    const uint32_t s_ownp = s_redq + 20 * 8;  // [3] their own P-slot sums (NS > 0)
    const uint32_t s_G = s_YP + (4 * TV + 4 + (NRX - NRT) * T) * SZ;
    if (s_YP + (4 * TV + 4) * SZ > 0xffffu) __trap();  // the packed gather addresses are 16-bit
    if (TM && warp == 0) {  // one warp allocates this CTA's columns; the address arrives through shared memory
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(
                         static_cast<uint32_t>(__cvta_generic_to_shared(&tm_slot))),
                     "n"(TM_COLS)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }

    PullSide<real, CPA, CPRA, J2, NS> A;
    PullSide<real, CPB, CPRB, J2, NS> B;
#pragma unroll
    for (int e = 0; e < CPA / 2; ++e) A.f1[e] = p.f1_pack[e * TV + va] + s_YP * 0x10001u;
#pragma unroll
    for (int e = 0; e < CPB / 2; ++e) B.f1[e] = p.f1_pack[e * TV + vb] + s_YP * 0x10001u;
#pragma unroll
    for (int e = 0; e < J2 / 2; ++e) {
        A.f2[e] = p.f2_pack[e * TV + va] + s_YP * 0x10001u;
        B.f2[e] = p.f2_pack[e * TV + vb] + s_YP * 0x10001u;
    }
#pragma unroll
    for (int e = 0; e < NS / 2; ++e) {  // N-slots: the rows after the largest P-slot capacity
        A.f1[CPA / 2 + e] = p.f1_pack[(kPullMaxSlots / 2 + e) * TV + va] + s_YP * 0x10001u;
        B.f1[CPB / 2 + e] = p.f1_pack[(kPullMaxSlots / 2 + e) * TV + vb] + s_YP * 0x10001u;
    }
    {
        const uint32_t ca = p.cnt[va], cb = p.cnt[vb];
        A.wnn = __reduce_max_sync(0xffffffffu, (ca >> 16) & 255u);
        B.wnn = __reduce_max_sync(0xffffffffu, (cb >> 16) & 255u);
        A.wn = __reduce_max_sync(0xffffffffu, ca & 255u);  // warp-wide trip counts
        A.wn2 = __reduce_max_sync(0xffffffffu, (ca >> 8) & 255u);
        B.wn = __reduce_max_sync(0xffffffffu, cb & 255u);
        B.wn2 = __reduce_max_sync(0xffffffffu, (cb >> 8) & 255u);
    }
    A.s_pub = s_YP + va * SZ;
    B.s_pub = s_YP + vb * SZ;

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
    if (tid < 4) YP[4 * TV + tid] = static_cast<real>(1);
    if (TM) asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    uint32_t tm_base = 0;  // this thread's lane quarter and first column
    if (TM) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        tm_base = *reinterpret_cast<volatile uint32_t*>(&tm_slot) + (static_cast<uint32_t>(warp & 3) << 21) +
                  static_cast<uint32_t>(warp >> 2) * TMC;
    }
    // tensor-memory address of this thread's column c
    auto tm_at = [&](uint32_t c) -> uint32_t { return tm_base + c; };
    auto tm_free = [&]() {  // by the allocating warp (warp 0: lane quarter 0, lane group 0)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tm_base & 0xffffu), "n"(TM_COLS));
    };
    // spilled rate `row` (0 .. NRX) of this thread: shared memory, or tensor memory
    auto put_rate = [&](int row, real r) {
        if (row < NRT) tm_st(tm_at(TM_RATE0 + RW * row), r);
        else Rx[(row - NRT) * T + tid] = r;
    };

    auto slot_rate = [&](int e, int v) -> real {
        const int32_t w = p.slot_rxn[e * TV + v];
        return w < 0 ? static_cast<real>(0)
                     : static_cast<real>(static_cast<double>(w >> 24) * Rbuf[w & 0xffffff]);
    };
#pragma unroll
    for (int e = 0; e < CPA; ++e) {
        const real r = slot_rate(e, va);
        if (e < CPRA) A.R[e] = r;
        else put_rate(e - CPRA, r);
    }
#pragma unroll
    for (int e = 0; e < CPB; ++e) {
        const real r = slot_rate(e, vb);
        if (e < CPRB) B.R[e] = r;
        else put_rate(SPA + e - CPRB, r);
    }
#pragma unroll
    for (int e = 0; e < NS; ++e) {
        put_rate(SPA + SPB + e, slot_rate(kPullMaxSlots + e, va));
        put_rate(SPA + SPB + NS + e, slot_rate(kPullMaxSlots + e, vb));
    }
    auto rate_sums = [&](real (&C)[kPullCoefs - kPull2SmemCoefs], int v, int side) {
        int q = p.agg_ptr[v];
#pragma unroll
        for (int s = 0; s < kPullCoefs; ++s) {
            const int qe = p.agg_ptr[(s + 1) * TV + v];
            double acc = 0.0;
            for (; q < qe; ++q) {  // fixed (reaction) order
                const int32_t w = p.agg_ent[(size_t)q * TV + v];
                acc += static_cast<double>(w >> 24) * Rbuf[w & 0xffffff];
            }
            if (KT) {  // value positions of a side: pull2_store; side b's K/G chunk pair follows side a's
                constexpr int pos[kPullCoefs] = {0, 1, 5, 7, 2, 3, 4, 6, 8, 9, 10, 12, 14, 11, 32, 13, 33, 15, 34};
                tm_st(tm_at(RW * (pos[s] < 32 ? pos[s] + 16 * side : pos[s] + 3 * side)), static_cast<real>(acc));
            } else if (s < kPullCoefs - kPull2SmemCoefs) C[s] = static_cast<real>(acc);
            else if (TM) tm_st(tm_at(RW * (side * kPull2SmemCoefs + s - (kPullCoefs - kPull2SmemCoefs))), static_cast<real>(acc));
            else Gs[(s - (kPullCoefs - kPull2SmemCoefs)) * TV + v] = static_cast<real>(acc);
        }
    };
    rate_sums(A.C, va, 0);
    rate_sums(B.C, vb, 1);
    if (TM) asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    if (KS) {
#pragma unroll
        for (int j = 0; j < NK; ++j) {
            Ks[j * TV + va] = A.C[j];
            Ks[j * TV + vb] = B.C[j];
        }
    }
    const uint32_t s_K = s_G;  // Ks sits where Gs would

    // ---- S6: zone state in ---------------------------------------------------------
    real* Yg = reinterpret_cast<real*>(p.Y) + (size_t)z * N;
    A.own = p.owner[va];
    B.own = p.owner[vb];
    const bool hub_owner = tid < nbs;  // hub h is owned by virtual thread h = side a of thread h
    const bool plain_a = A.own >= 0 && !hub_owner, plain_b = B.own >= 0;
    real ya = (A.own >= 0) ? Yg[A.own] : static_cast<real>(0);
    real yb = (B.own >= 0) ? Yg[B.own] : static_cast<real>(0);
    real yh0 = nbs > 0 ? Yg[p.hub[0]] : static_cast<real>(0);
    real yh1 = nbs > 1 ? Yg[p.hub[1]] : static_cast<real>(0);
    real yh2 = nbs > 2 ? Yg[p.hub[2]] : static_cast<real>(0);

    const real kappa = static_cast<real>(p.kappa);
    const real eps_y = static_cast<real>(p.eps_y);
    const real y_floor = static_cast<real>(p.y_floor);
    const real yfl_eps = eps_y * y_floor;
    const double growth = p.growth, t_hydro = p.t_hydro;
    const bool rhs_only = p.mode == kRhs;
    constexpr bool qss = QSS;

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

    // the hub abundance this lane updates in finalize (lane h: hub h), carried beside yh0..2: selecting
    // it from the three warp-uniform values costs a divergent branch per sub-step
    real yme = lane == 0 ? yh0 : (lane == 1 ? yh1 : (lane == 2 ? yh2 : static_cast<real>(0)));
    uint32_t pf0[8 * RW], pf1[8 * RW];  // K and most of G of side a, read ahead (KT)
    if (KT) {
        tm_ld(pf0, tm_at(0));
        tm_ld(pf1, tm_at(8 * RW));
    }
    // The sub-step loop, compiled for CAW / CBW live slots on side a / b of the calling warp (the
    // instantiation's capacities, or this warp's step of the staircase).  Returns true when the kernel is done
    // (mode kRhs).
    auto substeps = [&](auto caw_, auto cbw_) -> bool {
    constexpr int CAW = decltype(caw_)::value, CBW = decltype(cbw_)::value;
    constexpr bool HB = CBW > 0;  // this warp plays species on side b at all (else: none of that side's work)
    while (run) {
        // ---- publish y x {1, hubs}, both species -------------------------------------------
        const real pa1 = ya * yh0, pa2 = ya * yh1, pa3 = ya * yh2;
        const real pb1 = yb * yh0, pb2 = yb * yh1, pb3 = yb * yh2;
        sts(A.s_pub, ya);
        if (HB) sts(B.s_pub, yb);
        sts(A.s_pub + TV * SZ, pa1);
        if (HB) sts(B.s_pub + TV * SZ, pb1);
        sts(A.s_pub + 2 * TV * SZ, pa2);
        if (HB) sts(B.s_pub + 2 * TV * SZ, pb2);
        sts(A.s_pub + 3 * TV * SZ, pa3);
        if (HB) sts(B.s_pub + 3 * TV * SZ, pb3);

        // barrier A, right behind the publishes: what follows up to barrier B (rate sums, gathers, butterfly)
        // needs no further hand-shake, so the warps' skews over it add up once, at B, instead of being
        // waited out twice
        cta_barrier();
        // ---- rate sums: k = F-/y (Eq. (1)) and the hub-row shares, added over the two ----------
        real ka, kb = 0, share[6];
        {
            real sb[6] = {}, Ga[kPull2SmemCoefs], Gb[kPull2SmemCoefs] = {};
            if (KT) {
                // five chunks of 8 values: K and most of G of side a, of side b, the three last G of both
                // (the first two were issued after the last barrier B, or before the loop)
                real Ka[NK], Kb[NK], x[8], x1[8];
                tm_take8x2(x, x1, pf0, pf1);
                Ka[0] = x[0], Ka[1] = x[1], Ka[4] = x[2], Ka[5] = x[3], Ka[6] = x[4], Ka[2] = x[5], Ka[7] = x[6], Ka[3] = x[7];
#pragma unroll
                for (int j = 0; j < 8; ++j) x[j] = x1[j];
                Ka[8] = x[0], Ka[9] = x[1], Ga[0] = x[2], Ga[3] = x[3], Ga[1] = x[4], Ga[5] = x[5], Ga[2] = x[6], Ga[7] = x[7];
                if (HB) {
                    tm_load8(x, tm_at(16 * RW));
                    Kb[0] = x[0], Kb[1] = x[1], Kb[4] = x[2], Kb[5] = x[3], Kb[6] = x[4], Kb[2] = x[5], Kb[7] = x[6], Kb[3] = x[7];
                    tm_load8(x, tm_at(24 * RW));
                    Kb[8] = x[0], Kb[9] = x[1], Gb[0] = x[2], Gb[3] = x[3], Gb[1] = x[4], Gb[5] = x[5], Gb[2] = x[6], Gb[7] = x[7];
                }
                tm_load8(x, tm_at(32 * RW));
                Ga[4] = x[0], Ga[6] = x[1], Ga[8] = x[2], Gb[4] = x[3], Gb[6] = x[4], Gb[8] = x[5];
                pull_rate_sums<real>(Ka, Ga, ya, pa1, pa2, pa3, yh0, yh1, yh2, ka, share);
                if (HB) pull_rate_sums<real>(Kb, Gb, yb, pb1, pb2, pb3, yh0, yh1, yh2, kb, sb);
            } else if (TM) {
                tm_load_g(Ga, Gb, tm_at(0));
            } else {
#pragma unroll
                for (int j = 0; j < kPull2SmemCoefs; ++j) {
                    Ga[j] = lds_at<real>(s_G + (j * TV + va) * SZ);
                    Gb[j] = lds_at<real>(s_G + (j * TV + vb) * SZ);
                }
            }
            if (KT) {
            } else if (KS) {
                real Ka[NK], Kb[NK];
#pragma unroll
                for (int j = 0; j < NK; ++j) {
                    Ka[j] = lds_at<real>(s_K + (j * TV + va) * SZ);
                    Kb[j] = lds_at<real>(s_K + (j * TV + vb) * SZ);
                }
                pull_rate_sums<real>(Ka, Ga, ya, pa1, pa2, pa3, yh0, yh1, yh2, ka, share);
                if (HB) pull_rate_sums<real>(Kb, Gb, yb, pb1, pb2, pb3, yh0, yh1, yh2, kb, sb);
            } else {
                pull_rate_sums<real>(A.C, Ga, ya, pa1, pa2, pa3, yh0, yh1, yh2, ka, share);
                if (HB) pull_rate_sums<real>(B.C, Gb, yb, pb1, pb2, pb3, yh0, yh1, yh2, kb, sb);
            }
            if (HB) {
#pragma unroll
                for (int i = 0; i < 6; ++i) share[i] += sb[i];
            }
        }
        // own consumption of a hub owner in a hub-only reaction, read in finalize.  Stored between
        // the barriers: B orders it before this step's reads, the next A orders those reads
        // before the next store.
        if (hub_owner) sts(s_own + tid * SZ, ka * ya);

        // ---- S2+S3: P-slot gathers of both species, interleaved with the hub-row butterfly -----
        real Fpa, Fpb;
        {
            real sa0, sa1, sa2, sa3, a0, a1, a2, a3;
            real sb0 = 0, sb1 = 0, sb2 = 0, sb3 = 0, b0, b1, b2, b3;
// BRF: no branch inside the gathers.  Every group of four slots up to the instantiation's capacity is
// live in every warp; the groups a warp does not use (warp-uniform trip counts wn, wn2) hold rate 0 and the
// address of the constant 1 (one broadcast wavefront), so they add exact zeros.  Branching around them costs
// far more than their issue slots: it cuts the sub-step into basic blocks that ptxas cannot schedule across
// (hub150: 486 -> 448 instructions in the loop although all 20 + 12 slots of every warp are live, 255k ->
// 265k zone-networks/s on configs[3], a lone CTA 0.72 -> 0.53 us per sub-step).  With five or six warps the
// padding outweighs it (hub365, caps 24 + 12 against 16 + 12 in four of its six warps: 4.94 -> 5.22 ns per
// zone-substep), so those block sizes keep the branches.
#define KINNET_LOADS(S, CP_, CW_, g, x0, x1, x2, x3)                                            \
    if ((4 * (g) < CW_) && ((g) == 0 || (BRF || 4 * (g) < S.wn))) {                                 \
        const uint32_t w0 = S.f1[(2 * (g)) % (CP_ / 2)], w1 = S.f1[(2 * (g) + 1) % (CP_ / 2)]; \
        x0 = lds_at<real>(lo16(w0));                                                       \
        x1 = lds_at<real>(hi16(w0));                                                       \
        x2 = lds_at<real>(lo16(w1));                                                       \
        x3 = lds_at<real>(hi16(w1));                                                       \
        if (4 * (g) < J2 && (BRF || 4 * (g) < S.wn2)) { /* second factors (three-body reactions) */ \
            const uint32_t v0 = S.f2[(2 * (g)) % (J2 / 2)], v1 = S.f2[(2 * (g) + 1) % (J2 / 2)]; \
            const real z0 = lds_at<real>(lo16(v0)), z1 = lds_at<real>(hi16(v0));           \
            const real z2 = lds_at<real>(lo16(v1)), z3 = lds_at<real>(hi16(v1));           \
            x0 *= z0;                                                                      \
            x1 *= z1;                                                                      \
            x2 *= z2;                                                                      \
            x3 *= z3;                                                                      \
        }                                                                                  \
    }
#define KINNET_FMAS_A(g)                                                        \
    if ((g) == 0) {                                                             \
        sa0 = A.R[0] * a0;                                                      \
        sa1 = A.R[1] * a1;                                                      \
        sa2 = A.R[2] * a2;                                                      \
        sa3 = A.R[3] * a3;                                                      \
    } else if (4 * (g) < CPRA && 4 * (g) < CAW && (BRF || 4 * (g) < A.wn)) {                              \
        sa0 = fma(A.R[(4 * (g)) % CPRA], a0, sa0);                              \
        sa1 = fma(A.R[(4 * (g) + 1) % CPRA], a1, sa1);                          \
        sa2 = fma(A.R[(4 * (g) + 2) % CPRA], a2, sa2);                          \
        sa3 = fma(A.R[(4 * (g) + 3) % CPRA], a3, sa3);                          \
    } else if (4 * (g) < CAW && (BRF || 4 * (g) < A.wn)) {                               \
        real xr[4];                                                             \
        rates4(xr, (4 * (g) >= CPRA ? 4 * (g) - CPRA : 0));                     \
        sa0 = fma(xr[0], a0, sa0);                                              \
        sa1 = fma(xr[1], a1, sa1);                                              \
        sa2 = fma(xr[2], a2, sa2);                                              \
        sa3 = fma(xr[3], a3, sa3);                                              \
    }
#define KINNET_FMAS_B(g)                                                        \
    if (4 * (g) < CPRB && 4 * (g) < CBW && ((g) == 0 || (BRF || 4 * (g) < B.wn))) {                       \
        sb0 = fma(B.R[(4 * (g)) % CPRB], b0, sb0);                              \
        sb1 = fma(B.R[(4 * (g) + 1) % CPRB], b1, sb1);                          \
        sb2 = fma(B.R[(4 * (g) + 2) % CPRB], b2, sb2);                          \
        sb3 = fma(B.R[(4 * (g) + 3) % CPRB], b3, sb3);                          \
    } else if (4 * (g) < CBW && (BRF || 4 * (g) < B.wn)) {                               \
        real xr[4];                                                             \
        rates4(xr, SPA + (4 * (g) >= CPRB ? 4 * (g) - CPRB : 0));               \
        sb0 = fma(xr[0], b0, sb0);                                              \
        sb1 = fma(xr[1], b1, sb1);                                              \
        sb2 = fma(xr[2], b2, sb2);                                              \
        sb3 = fma(xr[3], b3, sb3);                                              \
    }
#define KINNET_STAGE(g)                               \
    KINNET_LOADS(A, CPA, CAW, g, a0, a1, a2, a3)      \
    KINNET_LOADS(B, CPB, CBW, g, b0, b1, b2, b3)
#define KINNET_FMAS(g) \
    KINNET_FMAS_A(g)   \
    KINNET_FMAS_B(g)
            static_assert(CPRA >= 4 && CPRB >= 4, "group 0 reads its rates from registers");
            // four consecutive spilled rates of this thread, rows row .. row + 3
            auto rates4 = [&](real (&x)[4], int row) {
                if (row < NRT) {
                    tm_load4(x, tm_at(TM_RATE0 + RW * row));
                } else {
#pragma unroll
                    for (int j = 0; j < 4; ++j) x[j] = lds_at<real>(s_Rx + (row - NRT + j) * T * SZ);
                }
            };
            const bool up16 = lane & 16, up8 = lane & 8, up4 = lane & 4;
            // level 16 of the butterfly (rows 0..2 = F+ shares of the hubs, 3..5 = F- shares)
            real r0 = __shfl_xor_sync(0xffffffffu, up16 ? share[0] : share[3], 16);
            real r1 = __shfl_xor_sync(0xffffffffu, up16 ? share[1] : share[4], 16);
            real r2 = __shfl_xor_sync(0xffffffffu, up16 ? share[2] : share[5], 16);
            KINNET_STAGE(0)
            const real b0_ = (up16 ? share[3] : share[0]) + r0;
            const real b1_ = (up16 ? share[4] : share[1]) + r1;
            const real b2_ = (up16 ? share[5] : share[2]) + r2;
            r0 = __shfl_xor_sync(0xffffffffu, up8 ? b0_ : b1_, 8);  // level 8
            r1 = __shfl_xor_sync(0xffffffffu, b2_, 8);
            KINNET_FMAS(0)
            KINNET_STAGE(1)
            const real c0_ = (up8 ? b1_ : b0_) + r0;
            const real c1_ = b2_ + r1;
            r0 = __shfl_xor_sync(0xffffffffu, up4 ? c0_ : c1_, 4);  // level 4
            KINNET_FMAS(1)
            KINNET_STAGE(2)
            real tot = (up4 ? c1_ : c0_) + r0;
            r0 = __shfl_xor_sync(0xffffffffu, tot, 2);
            KINNET_FMAS(2)
            KINNET_STAGE(3)
            tot += r0;
            r0 = __shfl_xor_sync(0xffffffffu, tot, 1);
            KINNET_FMAS(3)
            KINNET_STAGE(4)
            tot += r0;
            KINNET_FMAS(4)
            KINNET_STAGE(5)
            KINNET_FMAS(5)
#undef KINNET_STAGE
#undef KINNET_FMAS
#undef KINNET_FMAS_A
#undef KINNET_FMAS_B
#undef KINNET_LOADS
            // lanes 0, 8, 4, 16, 24, 20 hold the warp totals of rows 0, 1, 2, 3, 4, 5
            const int row = 3 * (lane >> 4) + ((lane & 4) ? 2 : ((lane >> 3) & 1));
            if ((lane & 3) == 0 && (lane & 12) != 12) sts(s_red + (warp * 8 + row) * SZ, tot);
            Fpa = (sa0 + sa1) + (sa2 + sa3);
            Fpb = (sb0 + sb1) + (sb2 + sb3);
        }
        if (NS > 0) {  // N-slots: k += sum nu R Y_partner, F- of the reactants of heavy + heavy reactions
            auto nrates4 = [&](real (&x)[4], int row) {
                if (row < NRT) {
                    tm_load4(x, tm_at(TM_RATE0 + RW * row));
                } else {
#pragma unroll
                    for (int j = 0; j < 4; ++j) x[j] = lds_at<real>(s_Rx + (row - NRT + j) * T * SZ);
                }
            };
            if (A.wnn > 0) {  // warp-uniform: the schedule keeps these species in one warp
                const uint32_t w0 = A.f1[CPA / 2], w1 = A.f1[(CPA + NS) / 2 - 1];
                const real n0 = lds_at<real>(lo16(w0)), n1 = lds_at<real>(hi16(w0));
                const real n2 = lds_at<real>(lo16(w1)), n3 = lds_at<real>(hi16(w1));
                real x[4];
                nrates4(x, SPA + SPB);
                ka += fma(x[2], n2, x[0] * n0) + fma(x[3], n3, x[1] * n1);
            }
            if (B.wnn > 0) {
                const uint32_t w0 = B.f1[CPB / 2], w1 = B.f1[(CPB + NS) / 2 - 1];
                const real n0 = lds_at<real>(lo16(w0)), n1 = lds_at<real>(hi16(w0));
                const real n2 = lds_at<real>(lo16(w1)), n3 = lds_at<real>(hi16(w1));
                real x[4];
                nrates4(x, SPA + SPB + NS);
                kb += fma(x[2], n2, x[0] * n0) + fma(x[3], n3, x[1] * n1);
            }
            // a hub made by heavy + heavy reactions gathers those fluxes on its own thread
            if (hub_owner) sts(s_ownp + tid * SZ, Fpa);
        }

        // ---- S5: q candidates of the non-hub species: |F+ - F-| / (eps max(y, floor)) ------
        real inva = 0, invb = 0;  // reciprocal factors of the dt candidates, off the critical path
        if (ADAPT) {
            inva = rcp_pos(ya > y_floor ? eps_y * ya : yfl_eps);
            if (HB) invb = rcp_pos(yb > y_floor ? eps_y * yb : yfl_eps);
            if (!plain_a) inva = 0;  // hub owners are judged on their full rows in finalize
            if (!plain_b) invb = 0;
        }
        const real cha = fma(-ka, ya, Fpa), chb = fma(-kb, yb, Fpb);
        if (ADAPT) {
            const real qa = abs_of(cha) * inva, qb = abs_of(chb) * invb;
            const double c = warp_max_pos(static_cast<double>(qa > qb ? qa : qb));
            if (lane == 0) sts(s_redq + warp * 8, c);
        }
        cta_barrier();
        if (KT) {  // the next sub-step's first two coefficient chunks: in flight during the finalize
            tm_ld(pf0, tm_at(0));
            tm_ld(pf1, tm_at(8 * RW));
        }

        // ---- finalize (every warp redundantly): hub rows over warps, zone-wide dt -----------
        real invh = 0;
        double q_rem = 0.0, rem = 0.0;
        if (ADAPT) {  // these depend on nothing the barrier waited for: they run beside the loads
            invh = rcp_pos(yme > y_floor ? eps_y * yme : yfl_eps);
            rem = t_hydro - t;
            q_rem = rcp_pos(rem);
        }
        real hFp, hFm;
        {   // lanes 0..nbs-1 only (one wavefront per load instead of two); predicated loads, not a
            // branch: the divergence bookkeeping costs more than the adds the idle lanes then do on zeros
            const bool act = lane < nbs;
            real vp[NW], vm[NW];
#pragma unroll
            for (int w = 0; w < NW; ++w) {
                vp[w] = lds_if<real>(act, s_red + (w * 8 + lane) * SZ);
                vm[w] = lds_if<real>(act, s_red + (w * 8 + 3 + lane) * SZ);
            }
            const real own_term = lds_if<real>(act, s_own + lane * SZ);
#pragma unroll
            for (int s = 1; s < NW; s *= 2)  // fixed pairwise order over warps (log depth)
#pragma unroll
                for (int w = 0; w + s < NW; w += 2 * s) {
                    vp[w] += vp[w + s];
                    vm[w] += vm[w + s];
                }
            hFp = vp[0];
            hFm = vm[0] + own_term;
            if (NS > 0) hFp += lds_if<real>(act, s_ownp + lane * SZ);
        }
        if (!ADAPT && rhs_only) {
            real* Fpo = reinterpret_cast<real*>(p.Fplus) + (size_t)z * N;
            real* Fmo = reinterpret_cast<real*>(p.Fminus) + (size_t)z * N;
            if (hub_owner) {
                Fpo[A.own] = hFp;
                Fmo[A.own] = hFm;
            } else if (A.own >= 0) {
                Fpo[A.own] = Fpa;
                Fmo[A.own] = ka * ya;
            }
            if (B.own >= 0) {
                Fpo[B.own] = Fpb;
                Fmo[B.own] = kb * yb;
            }
            if (TM) {  // give the columns back (every warp is past its last tcgen05.ld)
                if (KT) {
                    tm_wait(pf0);
                    tm_touch(pf1);
                }
                cta_barrier();
                if (warp == 0)
                    tm_free();
            }
            return true;
        }

        double q, hd;
        bool last;
        if (ADAPT) {
            double cand = 0.0;
            if (lane >= 8 && lane < 8 + NW) cand = lds_at<double>(s_redq + (lane - 8) * 8);
            const double qh = static_cast<double>(abs_of(hFp - hFm) * invh);
            if (lane < nbs) cand = qh;
            const double qmax = warp_max_pos(cand);
            const double qg = q_prev * ginv;                 // growth cap: dt <= g dt_prev
            const double q_ctrl = (qmax > qg) ? qmax : qg;   // a NaN candidate loses
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

        // ---- S4: update (Eq. (3)), Eq. (3) as (y q + F+) / (q + k) -----------
        real yna, ynb = yb;
        {
            const real aa = fma(ya, qr, Fpa) * rcp_pos(qr + ka);
            const real ea = fma(h, cha, ya);
            yna = (ya > 0 && ka * h >= kappa) ? aa : ea;
            if (qss)  // uniform: the QSS variant, one formula for every species
                yna = fma(cha, rcp_pos(qr + qss_alpha_k(ya > 0 ? ka : static_cast<real>(0), h)), ya);
            if (HB) {
                const real ab = fma(yb, qr, Fpb) * rcp_pos(qr + kb);
                const real eb = fma(h, chb, yb);
                ynb = (yb > 0 && kb * h >= kappa) ? ab : eb;
                if (qss) ynb = fma(chb, rcp_pos(qr + qss_alpha_k(yb > 0 ? kb : static_cast<real>(0), h)), yb);
            }
        }
        {  // hub species, on lanes 0..nbs-1 of every warp: Y (Y q + F+) / (Y q + F-)
            const bool pos = yme > Tiny<real>::v();
            const real den = fma(yme, qr, hFm);
            const real as = fma(yme, qr, hFp) * (yme * rcp_pos(pos ? den : static_cast<real>(1)));
            const real es = fma(h, hFp - hFm, yme);
            real hn = (pos && h * hFm >= kappa * yme) ? as : es;
            if (qss) {
                const real kh = pos ? hFm * rcp_pos(pos ? yme : static_cast<real>(1)) : static_cast<real>(0);
                hn = fma(hFp - hFm, rcp_pos(qr + qss_alpha_k(kh, h)), yme);
            }
            if (lane >= nbs) hn = 0;  // a missing hub reads as abundance 0
            yh0 = __shfl_sync(0xffffffffu, hn, 0);
            yh1 = __shfl_sync(0xffffffffu, hn, 1);
            yh2 = __shfl_sync(0xffffffffu, hn, 2);
            yme = hn;
            ya = hub_owner ? hn : yna;  // hub h lives on side a of thread h: warp 0, lane h
            yb = ynb;
        }
        t = last ? t_hydro : t + hd;
        ++steps;
        if (last) run = false;
        else if (ADAPT && steps >= max_steps) {
            status |= NET_STATUS_MAX_STEPS;
            run = false;
        }
    }
    return false;
    };
    {
        bool done;
        if (BRF && NW > 1 && p.stair) {  // warp-uniform
            done = stair_dispatch<NW, CPA, CPB>(warp, p.stair, substeps);
        } else {
            done = substeps(std::integral_constant<int, CPA>{}, std::integral_constant<int, CPB>{});
        }
        if (done) return;
    }
    if (ADAPT && steps > 0) dt_out = 1.0 / q_prev;

    // ---- S6: zone state out ------------------------------------------------------------------
    if (KT) {  // the read-ahead of a sub-step that never came: land it before the barrier below
        tm_wait(pf0);
        tm_touch(pf1);
    }
    const int bad = ((A.own >= 0) && !isfinite(static_cast<double>(ya))) ||
                    ((B.own >= 0) && !isfinite(static_cast<double>(yb)));
    if (__syncthreads_or(bad)) status |= NET_STATUS_NONFINITE;
    if (TM && warp == 0) tm_free();  // every warp is past its last tcgen05.ld: give the columns back
    if (p.energy) {  // uniform; Yg still holds the start-of-call abundances
        double e = 0.0;
        if (A.own >= 0) e = p.bind[A.own] * (static_cast<double>(ya) - static_cast<double>(Yg[A.own]));
        if (B.own >= 0) e += p.bind[B.own] * (static_cast<double>(yb) - static_cast<double>(Yg[B.own]));
        zone_energy_out(e, redq, p.energy + z);
    }
    if (A.own >= 0) Yg[A.own] = ya;
    if (B.own >= 0) Yg[B.own] = yb;
    if (tid == 0) {
        if (ADAPT && p.dt) p.dt[z] = dt_out;
        if (p.n_steps) p.n_steps[z] = steps;
        if (p.status) p.status[z] = status;
    }
}

// Instantiations: physical block size (virtual threads / 2) x slot capacity of side a x
// second-factor capacity.  Twelve side-a and eight side-b slot rates stay in registers,
// the rest in shared memory (measured on configs[3], zone-networks/s: a/b spill 8/4 ->
// 216.7k, 8/8 -> 218.2k, 12/8 -> 206.8k, 4/4 -> 206.2k).  Networks outside these classes
// run on the one-species kernel.
constexpr int kPull2CapB = 12, kPull2SpillB = 4, kPull2RegA = 12;

inline bool pull2_sides(const PullSchedule& P, int& slots_a, int& slots_b, int& slots2) {
    if (!P.ok || P.T % 64 != 0) return false;
    const int nwv = P.T / 32;
    slots_a = slots_b = slots2 = 0;
    for (int t = 0; t < P.T; ++t) {
        int& dst = (t / 32 < nwv / 2) ? slots_a : slots_b;
        dst = dst > P.n_slots[t] ? dst : P.n_slots[t];
        slots2 = slots2 > P.n_slots2[t] ? slots2 : P.n_slots2[t];
    }
    return true;
}
inline int pull2_cap_a(int slots_a) { return slots_a <= 20 ? 20 : 24; }

template <typename real, int TB, int CPA, bool ADAPT>
pull_fn pick_pull2_j2(int s2, int ns, bool qss) {
    // networks with N-slots have two-factor P-slots anyway: one second-factor class for them;
    // the QSS variant is instantiated for the larger second-factor class only
    constexpr int SA = CPA - kPull2RegA, CB = kPull2CapB, SB = kPull2SpillB, NS = kPullNSlots;
    constexpr int S0 = pull2_store(TB, 0), SN = pull2_store(TB, NS);
    if (qss) {
        if (ns > 0) return zone_kernel_pull2<real, TB, CPA, SA, CB, SB, 8, NS, ADAPT, true, SN>;
        return zone_kernel_pull2<real, TB, CPA, SA, CB, SB, 8, 0, ADAPT, true, S0>;
    }
    if (ns > 0) return zone_kernel_pull2<real, TB, CPA, SA, CB, SB, 8, NS, ADAPT, false, SN>;
    if (s2 <= 4) return zone_kernel_pull2<real, TB, CPA, SA, CB, SB, 4, 0, ADAPT, false, S0>;
    return zone_kernel_pull2<real, TB, CPA, SA, CB, SB, 8, 0, ADAPT, false, S0>;
}
// CPA = the side-a capacity this translation unit instantiates (20 or 24; pull2_inst.cu is compiled once per
// capacity so that the two halves build in parallel); nullptr for a schedule of the other capacity
template <typename real, int CPA, bool ADAPT>
pull_fn pick_pull2(const PullSchedule& P, int method = 0) {
    int sa, sb, s2;
    if (!pull2_sides(P, sa, sb, s2)) return nullptr;
    if (sa > 24 || sb > kPull2CapB || s2 > kJ2C || pull2_cap_a(sa) != CPA) return nullptr;
    const bool qss = method == 1;
    switch (P.T / 2) {
        case 32: return pick_pull2_j2<real, 32, CPA, ADAPT>(s2, P.nslots, qss);
        case 64: return pick_pull2_j2<real, 64, CPA, ADAPT>(s2, P.nslots, qss);
        case 96: return pick_pull2_j2<real, 96, CPA, ADAPT>(s2, P.nslots, qss);
        case 128: return pick_pull2_j2<real, 128, CPA, ADAPT>(s2, P.nslots, qss);
        case 160: return pick_pull2_j2<real, 160, CPA, ADAPT>(s2, P.nslots, qss);
        case 192: return pick_pull2_j2<real, 192, CPA, ADAPT>(s2, P.nslots, qss);
        default: return nullptr;
    }
}

#endif  // KINNET_PULL_INSTANTIATE

}  // namespace kinnet
