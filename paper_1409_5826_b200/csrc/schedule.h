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

    // ---- packed copies for the register-resident kernel -------------------
    // fast_ok when the network fits its compile-time capacities (kFast*).
    bool fast_ok = false;
    int plus_max = 0, minus_max = 0, bigrow_max = 0;
    std::vector<uint32_t> fx_pack;     // [rs][T]   byte offsets of Y[a] | Y[b] << 16
    std::vector<uint32_t> fxc_pack;    // [kFastSlots3][T] byte offset of Y[c] for slot rows < j3
    std::vector<uint32_t> plus_pack;   // [kFastPlus/2][T]  two 16-bit flux byte offsets per word
    std::vector<uint32_t> minus_pack;  // [kFastMinus/2][T]
    std::vector<uint32_t> rb_pack;     // [2*kMaxBigSpecies][T] eight 4-bit own-slot ids per row
    std::vector<uint32_t> cnt_pack;    // [T] plus | minus << 8
    std::vector<uint32_t> rbcnt_pack;  // [T] eight 4-bit readback counts, one per big row
};

constexpr int kFastSlots = 12;   // flux slots per thread held in registers
constexpr int kFastPlus = 24;    // F+ small-row entries per thread
constexpr int kFastMinus = 24;   // F- small-row entries per thread
constexpr int kFastRowCap = 8;   // readback entries per thread and big row
constexpr int kFastSlots3 = 2;   // slot rows that may hold three-body reactions

void pack_fast_tables(Schedule& S, int elem_bytes);

// Returns 0 or a NET_E* code with a message in err.
int build_schedule(int N, const int* A, int M, const int* n_react, const int* react,
                   const int* n_prod, const int* prod, const double* coef, Schedule& out,
                   std::string& err);

}  // namespace kinnet
