// schedule.h -- host-side compile of a reaction network into the per-thread
// flux-slot layout and gather schedule used by the sm_100a kernels.
// Internal to the library (the public face is include/kinnet.h).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace kinnet {

constexpr int kMaxReact = 3;
constexpr int kMaxProd = 4;
constexpr int kNCoef = 7;
constexpr int kCoefRows = 8;       // a0+ln p, a1..a6, n_react-1
constexpr int kMaxBigSpecies = 4;  // species whose F+/F- are reduced across the CTA

// One zone is integrated by one CTA of `T` threads.
//
// Flux slots ("fluxes ... highly parallel"): reaction r lives in
// slot j of thread t; its flux is written to shared memory at j*T + t, so every
// thread owns one bank-aligned column of the flux array.
//
// Sums (the F+_i / F-_i sums are the least parallel
// part and badly load-imbalanced, hundreds of terms for n, p, 4He against fewer
// than ten for most isotopes):
//   * small rows: thread `owner^-1(i)` gathers all entries of F+_i then F-_i
//     from shared memory in a fixed order;
//   * big species: every thread sums, from its OWN column (conflict-free), the
//     fluxes that feed each big row, the partial sums are combined by a warp
//     butterfly and a fixed-order sum over warps.
// Both are deterministic; there are no atomics.
struct Schedule {
    int N = 0, M = 0;
    int T = 0, W = 0;        // threads and warps per zone
    int rs = 0;              // flux slots per thread
    int j2 = 0, j3 = 0;      // slots [0,j2) have a 2nd reactant, [0,j3) a 3rd
    int n_entries = 0, n_entries_big = 0;

    std::vector<int32_t> flux_rxn;     // [rs*T]   reaction id or -1
    std::vector<uint16_t> flux_react;  // [rs*T*4] reactant species (N = constant one), 4th unused
    std::vector<double> coef;          // [kCoefRows][rs*T]

    std::vector<int32_t> owner;        // [T] species owned by thread t, or -1
    std::vector<int32_t> thread_of;    // [N]
    std::vector<uint16_t> small_plus;  // [T]
    std::vector<uint16_t> small_minus; // [T]
    int small_max = 0;
    std::vector<uint16_t> small_src;   // [small_max*T] flux index j*T+t of entry e of thread t

    int nbs = 0;                       // big species, pinned to threads W .. W+nbs-1
    std::vector<int32_t> big_species;  // [nbs]
    std::vector<uint8_t> big_cnt;      // [2*nbs][T] readback entries for row 2*s (+) / 2*s+1 (-)
    int readback_max = 0;
    std::vector<uint8_t> big_slot;     // [readback_max*T] own flux slot of readback entry e

};

// Returns 0 or a NET_E* code with a message in err.
int build_schedule(int N, const int* A, int M, const int* n_react, const int* react,
                   const int* n_prod, const int* prod, const double* coef, Schedule& out,
                   std::string& err);

// ---------------------------------------------------------------------------
// Pull schedule: the layout of the fast kernel (zone_kernel_pull).
//
// No flux array.  Thread t owns species owner[t] and keeps its abundance y in a
// register.  Up to three hub species (the n-, p-, alpha-like rows with hundreds
// of terms) are tracked in registers by every thread.  Each
// sub-step every thread publishes  YP[c][t] = y * {1, Y_hub0, Y_hub1, Y_hub2}[c]
// to shared memory; then
//   * F+ of a non-hub species is a gather over its incoming reactions, each flux
//     evaluated at the consumer:  f_r = R_r * YP[c1][t1] (* YP[c2][t2])   ("P-slot");
//   * k = F-/y of a non-hub species and the per-thread partial sums of the six
//     hub rows are polynomials in the hub abundances whose coefficients are sums of
//     rates over the reactions that share their abundance factors, formed once per
//     zone per call (T9 and rho are frozen over the hydro step, PAPER.md L47,
//     L197, L202);
//   * the hub rows are reduced over the CTA in a fixed order (no atomics).
//   * a reaction with TWO non-hub reactants a + b (the 12C+12C, 12C+16O, 16O+16O class of
//     the paper's Type Ia network) has no rate-sum form: its flux needs the
//     abundance of another thread.  Its products -- hubs included, on the hub's own thread --
//     get two-factor P-slots R * YP[0][t_a] * YP[0][t_b]; each reactant gets an "N-slot"
//     k_a += nu R * YP[0][t_b], gathered beside the P-slots (k = F-/y, Eq. (1)).
// A network qualifies (ok) when every reaction has at most two non-hub reactants, those
// with two have no hub co-reactant, reactions with one non-hub reactant and a hub product
// have at most one hub co-reactant different from that product, and the capacities below
// hold; anything else runs on the generic flux-array kernel.
constexpr int kPullHubs = 3;
constexpr int kPullClasses = 10;  // co-reactant classes: {}, {h}, {h,h'} (h <= h')
constexpr int kPullCoefs = 19;    // K[10], G0[3], Gx[3][2]
constexpr int kPullMaxSlots = 24; // P-slots per thread (largest kernel instantiation)
constexpr int kPullMaxSlots2 = 8; // P-slots per thread with a second factor
constexpr int kPullNSlots = 4;    // N-slots per thread (reactions it enters with another non-hub reactant)

struct PullSchedule {
    bool ok = false;
    std::string why;                   // why not, when !ok
    int T = 0, W = 0, nbs = 0;
    int hub[kPullHubs] = {-1, -1, -1}; // hub species; hub h is owned by thread h
    std::vector<int32_t> owner;        // [T] species of thread t or -1
    std::vector<int32_t> thread_of;    // [N]
    int slots = 0;                     // max P-slots of any thread
    int slots2 = 0;                    // max P-slots with a second factor of any thread
    std::vector<uint8_t> n_slots;      // [T]  1 + last used position (positions may have holes)
    std::vector<uint8_t> n_slots2;     // [T]  1 + last position whose slot has a second factor
    std::vector<int32_t> slot_rxn;     // [slots][T] reaction | nu << 24, -1 = hole
    std::vector<uint16_t> slot_f1;     // [slots][T] YP word index c*T + t of the first factor
    std::vector<uint16_t> slot_f2;     // [slots2][T] YP word index of the second factor (4T+3 = one)
    int nslots = 0;                    // max N-slots of any thread (0: no reaction has two non-hub reactants)
    std::vector<uint8_t> n_nslots;     // [T]
    std::vector<int32_t> nslot_rxn;    // [kPullNSlots][T] reaction | nu << 24, -1 = hole
    std::vector<uint16_t> nslot_f1;    // [kPullNSlots][T] YP word index of the partner's abundance
    // rate sums: coefficient s of thread t = sum of nu * R over agg_ent[agg_ptr[s][t] .. agg_ptr[s+1][t])
    int agg_max = 0;
    std::vector<uint16_t> agg_ptr;     // [kPullCoefs + 1][T]
    std::vector<int32_t> agg_ent;      // [agg_max][T] reaction | nu << 24
    long conflict_wavefronts = 0;      // predicted shared-memory wavefronts of the P-slot gathers (fp64)
    long ideal_wavefronts = 0;
};

// coefficient slots of PullSchedule::agg_ptr
//   0..9   K_c   c = 0: {}, 1..3: {hub c-1}, 4..9: {0,0},{0,1},{0,2},{1,1},{1,2},{2,2}
//   10..12 G0_h  reactions of this thread with hub h as a product and no hub co-reactant
//   13..18 Gx_h,j  hub h as a product, one hub co-reactant: the j-th of the other two hubs
// elem_bytes = size of one abundance (8 or 4): it fixes the shared-memory bank of a word.
// force_T > 0 compiles for exactly that many (virtual) threads instead of the first block-size
// class >= N (the two-species-per-thread kernel plays two virtual threads per thread).
void build_pull_schedule(int N, int M, const int* n_react, const int* react, const int* n_prod,
                         const int* prod, int elem_bytes, PullSchedule& out, int force_T = 0);

}  // namespace kinnet
