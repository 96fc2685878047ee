// schedule.cpp -- see schedule.h.  Pure host C++; no CUDA.
#include "schedule.h"

#include <algorithm>
#include <cmath>
#include <limits>
#include <numeric>

#include "../../include/kinnet.h"

namespace kinnet {

namespace {

double ln_factorial(int m) {
    double s = 0.0;
    for (int q = 2; q <= m; ++q) s += std::log(static_cast<double>(q));
    return s;
}

}  // namespace

int build_schedule(int N, const int* A, int M, const int* n_react, const int* react,
                   const int* n_prod, const int* prod, const double* coef, Schedule& S,
                   std::string& err) {
    if (!A || !n_react || !react || !n_prod || !prod || !coef) {
        err = "null table pointer";
        return NET_EINVAL;
    }
    if (N < 1 || N > NET_MAX_SPECIES) {
        err = "n_species out of range [1, " + std::to_string(NET_MAX_SPECIES) + "]";
        return NET_EINVAL;
    }
    if (M < 1 || M > NET_MAX_REACTIONS) {
        err = "n_reactions out of range [1, " + std::to_string(NET_MAX_REACTIONS) + "]";
        return NET_EINVAL;
    }
    for (int r = 0; r < M; ++r) {
        if (n_react[r] < 1 || n_react[r] > kMaxReact) {
            err = "reaction " + std::to_string(r) + ": n_react not in 1..3";
            return NET_EINVAL;
        }
        if (n_prod[r] < 1 || n_prod[r] > kMaxProd) {
            err = "reaction " + std::to_string(r) + ": n_prod not in 1..4";
            return NET_EINVAL;
        }
        long bal = 0;
        for (int q = 0; q < n_react[r]; ++q) {
            int s = react[r * kMaxReact + q];
            if (s < 0 || s >= N) {
                err = "reaction " + std::to_string(r) + ": reactant index out of range";
                return NET_EINVAL;
            }
            bal += A[s];
        }
        for (int q = 0; q < n_prod[r]; ++q) {
            int s = prod[r * kMaxProd + q];
            if (s < 0 || s >= N) {
                err = "reaction " + std::to_string(r) + ": product index out of range";
                return NET_EINVAL;
            }
            bal -= A[s];
        }
        if (bal != 0) {
            err = "reaction " + std::to_string(r) + " does not conserve nucleon number";
            return NET_EINVAL;
        }
        for (int c = 0; c < kNCoef; ++c)
            if (!std::isfinite(coef[r * kNCoef + c])) {
                err = "reaction " + std::to_string(r) + ": non-finite coefficient";
                return NET_EINVAL;
            }
    }

    S = Schedule();
    S.N = N;
    S.M = M;
    S.T = std::max(32, (N + 31) / 32 * 32);
    S.W = S.T / 32;
    const int T = S.T;
    S.rs = (M + T - 1) / T;
    if (S.rs > 255) {
        err = "too many reactions per species for the slot layout (flux slots > 255)";
        return NET_EINVAL;
    }

    // ---- entry counts per (species, sign) and the big species ------------
    std::vector<int> cnt_plus(N, 0), cnt_minus(N, 0);
    for (int r = 0; r < M; ++r) {
        for (int q = 0; q < n_react[r]; ++q) ++cnt_minus[react[r * kMaxReact + q]];
        for (int q = 0; q < n_prod[r]; ++q) ++cnt_plus[prod[r * kMaxProd + q]];
    }
    S.n_entries = std::accumulate(cnt_plus.begin(), cnt_plus.end(), 0) +
                  std::accumulate(cnt_minus.begin(), cnt_minus.end(), 0);
    {
        const int threshold = std::max(48, T / 2);
        std::vector<int> cand;
        for (int i = 0; i < N; ++i)
            if (std::max(cnt_plus[i], cnt_minus[i]) >= threshold) cand.push_back(i);
        std::stable_sort(cand.begin(), cand.end(), [&](int a, int b) {
            return cnt_plus[a] + cnt_minus[a] > cnt_plus[b] + cnt_minus[b];
        });
        int cap = std::min(kMaxBigSpecies, 32 - S.W);
        if (cap < 0) cap = 0;
        if (static_cast<int>(cand.size()) > cap) cand.resize(cap);
        std::sort(cand.begin(), cand.end());
        S.big_species.assign(cand.begin(), cand.end());
        S.nbs = static_cast<int>(cand.size());
    }
    std::vector<int> big_index(N, -1);
    for (int s = 0; s < S.nbs; ++s) big_index[S.big_species[s]] = s;

    // ---- reactions -> (thread, slot): arity-sorted round-robin deal ------
    // Sorting by arity makes the 2nd/3rd reactant multiply uniform per slot row;
    // sorting by big-row signature inside an arity class spreads the reactions
    // that feed each big row evenly over the threads (readback balance).
    auto signature = [&](int r) {
        unsigned sig = 0;
        for (int q = 0; q < n_react[r]; ++q) {
            int b = big_index[react[r * kMaxReact + q]];
            if (b >= 0) sig += 1u << (4 * (2 * b + 1) % 32);
        }
        for (int q = 0; q < n_prod[r]; ++q) {
            int b = big_index[prod[r * kMaxProd + q]];
            if (b >= 0) sig += 1u << (4 * (2 * b) % 32);
        }
        return sig;
    };
    std::vector<int> order(M);
    std::iota(order.begin(), order.end(), 0);
    std::vector<unsigned> sig(M);
    for (int r = 0; r < M; ++r) sig[r] = signature(r);
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) {
        if (n_react[a] != n_react[b]) return n_react[a] > n_react[b];
        return sig[a] < sig[b];
    });
    int n3 = 0, n2 = 0;
    for (int r = 0; r < M; ++r) {
        n3 += n_react[r] == 3;
        n2 += n_react[r] >= 2;
    }
    S.j3 = (n3 + T - 1) / T;
    S.j2 = (n2 + T - 1) / T;

    const int slots = S.rs * T;
    S.flux_rxn.assign(slots, -1);
    S.flux_react.assign(static_cast<size_t>(slots) * 4, static_cast<uint16_t>(N));
    S.coef.assign(static_cast<size_t>(kCoefRows) * slots, 0.0);
    for (int idx = 0; idx < slots; ++idx)
        S.coef[idx] = -std::numeric_limits<double>::infinity();  // empty slot: R = exp(-inf) = 0
    std::vector<int> slot_of(M);  // flux index j*T + t of reaction r
    for (int k = 0; k < M; ++k) {
        const int r = order[k];
        const int idx = k;  // j = k / T, t = k % T  ->  j*T + t = k
        slot_of[r] = idx;
        S.flux_rxn[idx] = r;
        double lnp = 0.0;
        for (int q = 0; q < n_react[r]; ++q) {
            const int s = react[r * kMaxReact + q];
            S.flux_react[static_cast<size_t>(idx) * 4 + q] = static_cast<uint16_t>(s);
            bool first = true;
            int m = 0;
            for (int u = 0; u < q; ++u) first = first && react[r * kMaxReact + u] != s;
            if (!first) continue;
            for (int u = 0; u < n_react[r]; ++u) m += react[r * kMaxReact + u] == s;
            lnp -= ln_factorial(m);  // statistical factor 1/prod(m!)
        }
        S.coef[0 * static_cast<size_t>(slots) + idx] = coef[r * kNCoef + 0] + lnp;
        for (int c = 1; c < kNCoef; ++c)
            S.coef[c * static_cast<size_t>(slots) + idx] = coef[r * kNCoef + c];
        S.coef[7 * static_cast<size_t>(slots) + idx] = static_cast<double>(n_react[r] - 1);
    }

    // ---- species -> owner thread -------------------------------------------
    S.owner.assign(T, -1);
    S.thread_of.assign(N, -1);
    for (int s = 0; s < S.nbs; ++s) {
        S.owner[S.W + s] = S.big_species[s];
        S.thread_of[S.big_species[s]] = S.W + s;
    }
    {
        std::vector<int> rest;
        for (int i = 0; i < N; ++i)
            if (big_index[i] < 0) rest.push_back(i);
        // longest rows first: threads of one warp then run similar trip counts
        std::stable_sort(rest.begin(), rest.end(), [&](int a, int b) {
            return cnt_plus[a] + cnt_minus[a] > cnt_plus[b] + cnt_minus[b];
        });
        int t = 0;
        for (int i : rest) {
            while (t < T && S.owner[t] >= 0) ++t;
            if (t >= T) {
                err = "internal: no thread left for a species";
                return NET_EINVAL;
            }
            S.owner[t] = i;
            S.thread_of[i] = t;
        }
    }

    // ---- small rows and big-row readback lists -----------------------------
    std::vector<std::vector<uint16_t>> plus(T), minus(T);
    std::vector<std::vector<std::vector<uint8_t>>> rb(
        T, std::vector<std::vector<uint8_t>>(2 * std::max(1, S.nbs)));
    if (slots > 65535) {
        err = "flux array too large for 16-bit gather indices";
        return NET_EINVAL;
    }
    for (int r = 0; r < M; ++r) {  // reaction order = fixed, documented summation order
        const int idx = slot_of[r];
        const int t_src = idx % T, j_src = idx / T;
        for (int q = 0; q < n_react[r]; ++q) {
            const int s = react[r * kMaxReact + q];
            if (big_index[s] >= 0) {
                rb[t_src][2 * big_index[s] + 1].push_back(static_cast<uint8_t>(j_src));
                ++S.n_entries_big;
            } else {
                minus[S.thread_of[s]].push_back(static_cast<uint16_t>(idx));
            }
        }
        for (int q = 0; q < n_prod[r]; ++q) {
            const int s = prod[r * kMaxProd + q];
            if (big_index[s] >= 0) {
                rb[t_src][2 * big_index[s]].push_back(static_cast<uint8_t>(j_src));
                ++S.n_entries_big;
            } else {
                plus[S.thread_of[s]].push_back(static_cast<uint16_t>(idx));
            }
        }
    }
    S.small_plus.assign(T, 0);
    S.small_minus.assign(T, 0);
    S.small_max = 0;
    for (int t = 0; t < T; ++t) {
        if (plus[t].size() + minus[t].size() > 65535) {
            err = "small row too long";
            return NET_EINVAL;
        }
        S.small_plus[t] = static_cast<uint16_t>(plus[t].size());
        S.small_minus[t] = static_cast<uint16_t>(minus[t].size());
        S.small_max = std::max<int>(S.small_max, plus[t].size() + minus[t].size());
    }
    S.small_src.assign(static_cast<size_t>(std::max(1, S.small_max)) * T, 0);
    for (int t = 0; t < T; ++t) {
        int e = 0;
        for (uint16_t v : plus[t]) S.small_src[static_cast<size_t>(e++) * T + t] = v;
        for (uint16_t v : minus[t]) S.small_src[static_cast<size_t>(e++) * T + t] = v;
    }
    S.big_cnt.assign(static_cast<size_t>(2 * std::max(1, S.nbs)) * T, 0);
    S.readback_max = 0;
    for (int t = 0; t < T; ++t) {
        int total = 0;
        for (int b = 0; b < 2 * S.nbs; ++b) {
            if (rb[t][b].size() > 255) {
                err = "readback list too long";
                return NET_EINVAL;
            }
            S.big_cnt[static_cast<size_t>(b) * T + t] = static_cast<uint8_t>(rb[t][b].size());
            total += static_cast<int>(rb[t][b].size());
        }
        S.readback_max = std::max(S.readback_max, total);
    }
    S.big_slot.assign(static_cast<size_t>(std::max(1, S.readback_max)) * T, 0);
    for (int t = 0; t < T; ++t) {
        int e = 0;
        for (int b = 0; b < 2 * S.nbs; ++b)
            for (uint8_t v : rb[t][b]) S.big_slot[static_cast<size_t>(e++) * T + t] = v;
    }

    return NET_OK;
}

namespace {

// Shared-memory wavefronts of the P-slot gathers.  One wavefront serves 128 bytes:
// a warp's LDS.64 goes out as two half-warps, an LDS.32 as one piece.  Within a
// piece, lanes that read different words of the same bank (word index modulo the
// piece size) are serialised; equal words are broadcast.
int piece_wavefronts(const uint16_t* words, int lanes) {
    int worst = 1;
    for (int b = 0; b < lanes; ++b) {
        int distinct = 0;
        uint16_t seen[32];
        for (int l = 0; l < lanes; ++l) {
            const uint16_t w = words[l];
            if (w % lanes != b) continue;
            bool dup = false;
            for (int q = 0; q < distinct; ++q) dup = dup || seen[q] == w;
            if (!dup) seen[distinct++] = w;
        }
        worst = std::max(worst, distinct);
    }
    return worst;
}

void pull_wavefronts(const PullSchedule& P, int elem_bytes, long& actual, long& ideal) {
    actual = ideal = 0;
    const int T = P.T, lanes = 128 / elem_bytes;
    for (int w = 0; w < P.W; ++w) {
        int wmax = 0;
        for (int l = 0; l < 32; ++l) wmax = std::max<int>(wmax, P.n_slots[w * 32 + l]);
        for (int e = 0; e < wmax; ++e)
            for (int piece = 0; piece < 32 / lanes; ++piece) {
                uint16_t words[32];
                for (int l = 0; l < lanes; ++l)
                    words[l] = P.slot_f1[static_cast<size_t>(e) * T + w * 32 + piece * lanes + l];
                actual += piece_wavefronts(words, lanes);
                ideal += 1;
            }
    }
}

// Order the P-slots of every thread so that the lanes served by one wavefront
// read different banks at every position ("memory accesses
// are not yet optimized" is what the paper blames for the cost of the sums).
// The order of a thread's slots is free -- it only fixes the order of its F+ sum
// -- so this is an edge colouring of the bipartite multigraph lanes x banks of
// each piece; a min-conflicts search from a greedy start gets within a few
// wavefronts of the bound max(slots of a lane, slots on a bank).
//   pos[t][p]   slot index of thread t at position p, -1 = hole
//   cap         positions available to the warp (multiple of 4, the kernel's group size)
//   cap2        positions that may hold a slot with a second factor
struct Placement {
    std::vector<std::vector<int>> pos;
};

template <typename SlotT>
void place_piece(const std::vector<std::vector<SlotT>>& slots, int t0, int lanes, int cap, int cap2,
                 std::vector<std::vector<int>>& pos) {
    // cnt[p][b] = lanes of the piece reading bank b at position p
    std::vector<std::vector<int>> cnt(cap, std::vector<int>(lanes, 0));
    auto bank = [&](int t, int s) { return slots[t][s].f1 % lanes; };
    auto cost_at = [&](int p) {
        int worst = 1;
        for (int b = 0; b < lanes; ++b) worst = std::max(worst, cnt[p][b]);
        return worst;
    };
    for (int l = 0; l < lanes; ++l) pos[t0 + l].assign(cap, -1);
    // greedy start: two-factor slots first (fewer legal positions), busiest banks first
    std::vector<int> bank_deg(lanes, 0);
    for (int l = 0; l < lanes; ++l)
        for (size_t s = 0; s < slots[t0 + l].size(); ++s) ++bank_deg[bank(t0 + l, s)];
    struct Item { int t, s; };
    std::vector<Item> items;
    for (int l = 0; l < lanes; ++l)
        for (size_t s = 0; s < slots[t0 + l].size(); ++s) items.push_back({t0 + l, static_cast<int>(s)});
    std::stable_sort(items.begin(), items.end(), [&](const Item& a, const Item& b) {
        const bool ta = slots[a.t][a.s].two, tb = slots[b.t][b.s].two;
        if (ta != tb) return ta;
        return bank_deg[bank(a.t, a.s)] > bank_deg[bank(b.t, b.s)];
    });
    for (const Item& it : items) {
        const int b = bank(it.t, it.s), lim = slots[it.t][it.s].two ? cap2 : cap;
        int best = -1, best_cnt = 1 << 30;
        for (int p = 0; p < lim; ++p)
            if (pos[it.t][p] < 0 && cnt[p][b] < best_cnt) {
                best = p;
                best_cnt = cnt[p][b];
            }
        pos[it.t][best] = it.s;
        ++cnt[best][b];
    }
    // min-conflicts: swap two positions of one lane whenever that lowers the wavefront count
    uint32_t rng = 0x9E3779B9u ^ static_cast<uint32_t>(t0 * 2654435761u);
    auto next = [&]() { rng = rng * 1664525u + 1013904223u; return rng >> 8; };
    for (int pass = 0; pass < 400; ++pass) {
        bool any_conflict = false;
        for (int p = 0; p < cap; ++p) any_conflict = any_conflict || cost_at(p) > 1;
        if (!any_conflict) break;
        for (int l = 0; l < lanes; ++l) {
            const int t = t0 + l;
            for (int p = 0; p < cap; ++p) {
                const int s = pos[t][p];
                if (s < 0 || cnt[p][bank(t, s)] < 2) continue;  // not in conflict
                const int q0 = static_cast<int>(next() % cap);
                for (int dq = 0; dq < cap; ++dq) {
                    const int q = (q0 + dq) % cap;
                    if (q == p) continue;
                    const int s2 = pos[t][q];
                    if (slots[t][s].two && q >= cap2) continue;
                    if (s2 >= 0 && slots[t][s2].two && p >= cap2) continue;
                    const int before = cost_at(p) + cost_at(q);
                    const int b1 = bank(t, s), b2 = s2 >= 0 ? bank(t, s2) : -1;
                    --cnt[p][b1]; ++cnt[q][b1];
                    if (s2 >= 0) { --cnt[q][b2]; ++cnt[p][b2]; }
                    const int after = cost_at(p) + cost_at(q);
                    // accept improvements, and sideways moves that empty the conflict here
                    if (after < before || (after == before && cnt[q][b1] == 1 && (next() & 3) == 0)) {
                        std::swap(pos[t][p], pos[t][q]);
                        break;
                    }
                    ++cnt[p][b1]; --cnt[q][b1];
                    if (s2 >= 0) { ++cnt[q][b2]; --cnt[p][b2]; }
                }
            }
        }
    }
}

}  // namespace

void build_pull_schedule(int N, int M, const int* n_react, const int* react, const int* n_prod,
                         const int* prod, int elem_bytes, PullSchedule& P, int force_T) {
    P = PullSchedule();
    auto reject = [&](const std::string& why) {
        P.ok = false;
        P.why = why;
    };
    // the kernel is instantiated for these block sizes and runs exactly T threads
    int T = 0;
    for (int cls : {32, 64, 160, 256, 384, 512})
        if (T == 0 && N <= cls) T = cls;
    if (force_T > 0) T = (force_T % 32 == 0 && force_T >= N) ? force_T : 0;
    if (T == 0) return reject("more than 512 species (or a bad forced thread count)");
    P.T = T;
    P.W = T / 32;
    if (M > 65535) return reject("more than 65535 reactions");

    // ---- hubs: the rows with hundreds of terms ------------------
    std::vector<int> cnt_plus(N, 0), cnt_minus(N, 0);
    for (int r = 0; r < M; ++r) {
        for (int q = 0; q < n_react[r]; ++q) ++cnt_minus[react[r * kMaxReact + q]];
        for (int q = 0; q < n_prod[r]; ++q) ++cnt_plus[prod[r * kMaxProd + q]];
    }
    {
        const int threshold = std::max(48, T / 2);
        std::vector<int> cand;
        for (int i = 0; i < N; ++i)
            if (std::max(cnt_plus[i], cnt_minus[i]) >= threshold) cand.push_back(i);
        std::stable_sort(cand.begin(), cand.end(), [&](int a, int b) {
            return cnt_plus[a] + cnt_minus[a] > cnt_plus[b] + cnt_minus[b];
        });
        if (static_cast<int>(cand.size()) > kPullHubs) cand.resize(kPullHubs);
        std::sort(cand.begin(), cand.end());
        P.nbs = static_cast<int>(cand.size());
        for (int h = 0; h < P.nbs; ++h) P.hub[h] = cand[h];
    }
    std::vector<int> hub_index(N, -1);
    for (int h = 0; h < P.nbs; ++h) hub_index[P.hub[h]] = h;
    auto pair_class = [](int a, int b) {  // a <= b, hubs 0..2 -> 4..9
        static const int tab[3][3] = {{4, 5, 6}, {-1, 7, 8}, {-1, -1, 9}};
        return tab[a][b];
    };

    // ---- per reaction: owner, co-reactant class, factors ---------------------------
    struct Rx {
        int owner, cls, co[2], nco;
        int hh_a = -1, hh_b = -1;  // the two non-hub reactants of a heavy + heavy reaction
    };
    std::vector<Rx> rx(M);
    for (int r = 0; r < M; ++r) {
        int heavy = -1, heavy0 = -1, nheavy = 0;
        for (int q = 0; q < n_react[r]; ++q) {
            const int s = react[r * kMaxReact + q];
            if (hub_index[s] < 0) {
                if (nheavy == 0) heavy0 = s;
                heavy = s;
                ++nheavy;
            }
        }
        if (nheavy > 2 || (nheavy == 2 && n_react[r] > 2))
            return reject("reaction " + std::to_string(r) +
                          " has two non-hub reactants next to a third reactant");
        Rx& x = rx[r];
        if (nheavy == 2) {  // heavy + heavy: N-slots and two-factor P-slots, no rate-sum class
            x.owner = heavy0;
            x.hh_a = heavy0;
            x.hh_b = heavy;
            x.nco = 0;
            x.cls = -1;
            continue;
        }
        x.owner = nheavy == 1 ? heavy : react[r * kMaxReact];
        x.nco = 0;
        bool skipped = false;
        for (int q = 0; q < n_react[r]; ++q) {
            const int s = react[r * kMaxReact + q];
            if (s == x.owner && !skipped) {
                skipped = true;
                continue;
            }
            x.co[x.nco++] = hub_index[s];
        }
        if (x.nco == 2 && x.co[0] > x.co[1]) std::swap(x.co[0], x.co[1]);
        x.cls = x.nco == 0 ? 0 : x.nco == 1 ? 1 + x.co[0] : pair_class(x.co[0], x.co[1]);
    }

    // ---- species -> thread: hub h on thread h, the rest by falling in-degree ---------
    std::vector<int> indeg(N, 0);  // P-slots = distinct (reaction, non-hub product) pairs
    for (int r = 0; r < M; ++r)
        for (int q = 0; q < n_prod[r]; ++q) {
            const int s = prod[r * kMaxProd + q];
            bool first = true;
            for (int u = 0; u < q; ++u) first = first && prod[r * kMaxProd + u] != s;
            if (first && hub_index[s] < 0) ++indeg[s];
        }
    P.owner.assign(T, -1);
    P.thread_of.assign(N, -1);
    for (int h = 0; h < P.nbs; ++h) {
        P.owner[h] = P.hub[h];
        P.thread_of[P.hub[h]] = h;
    }
    {
        std::vector<int> rest;
        for (int i = 0; i < N; ++i)
            if (hub_index[i] < 0) rest.push_back(i);
        std::stable_sort(rest.begin(), rest.end(), [&](int a, int b) { return indeg[a] > indeg[b]; });
        // Species with N-slots (reactants of heavy + heavy reactions) go next to each other, at
        // the rank of the first of them, shifted so that the block stays inside one warp when
        // it fits: the N-slot gathers are skipped by every warp that has none.
        std::vector<char> special(N, 0);
        for (int r = 0; r < M; ++r)
            if (rx[r].hh_a >= 0) special[rx[r].hh_a] = special[rx[r].hh_b] = 1;
        std::vector<int> sp, ord;
        int first_rank = -1;
        for (size_t k = 0; k < rest.size(); ++k) {
            if (special[rest[k]]) {
                if (first_rank < 0) first_rank = static_cast<int>(ord.size());
                sp.push_back(rest[k]);
            } else {
                ord.push_back(rest[k]);
            }
        }
        if (!sp.empty()) {
            int start = first_rank + P.nbs;  // thread index of the block
            const int ns = static_cast<int>(sp.size());
            if (ns <= 32 && start / 32 != (start + ns - 1) / 32) {
                const int back = (start / 32 + 1) * 32 - ns;  // slide back to end at the warp's last lane
                start = back >= P.nbs ? back : (start / 32 + 1) * 32;
            }
            rest.assign(ord.begin(), ord.begin() + std::min<size_t>(ord.size(), start - P.nbs));
            rest.insert(rest.end(), sp.begin(), sp.end());
            rest.insert(rest.end(), ord.begin() + std::min<size_t>(ord.size(), start - P.nbs), ord.end());
        }
        int t = P.nbs;
        for (int i : rest) {
            P.owner[t] = i;
            P.thread_of[i] = t++;
        }
    }

    // ---- balance the banks: swap species between threads of one warp ---------------------
    // A piece (the lanes one wavefront serves) cannot gather a position in fewer
    // wavefronts than its busiest bank holds words, so spread every piece's sources
    // over the banks before the slots are ordered.  Swaps stay inside a warp: its slot
    // count (the falling in-degree order) is untouched.
    {
        const int lanes = 128 / elem_bytes;
        std::vector<std::vector<int>> srcs(N);  // non-hub species -> owner species of each P-slot
        for (int r = 0; r < M; ++r)
            for (int q = 0; q < n_prod[r]; ++q) {
                const int s = prod[r * kMaxProd + q];
                bool first = true;
                for (int u = 0; u < q; ++u) first = first && prod[r * kMaxProd + u] != s;
                if (first && hub_index[s] < 0) srcs[s].push_back(rx[r].owner);
            }
        const int pieces = T / lanes;
        std::vector<int> cap(pieces, 0);
        for (int pc = 0; pc < pieces; ++pc) {
            int most = 0;
            for (int l = 0; l < 32; ++l) {
                const int sp = P.owner[(pc * lanes / 32) * 32 + l];
                if (sp >= 0) most = std::max<int>(most, srcs[sp].size());
            }
            cap[pc] = (most + 3) / 4 * 4;
        }
        std::vector<int> deg(static_cast<size_t>(pieces) * lanes);
        auto total_cost = [&]() {
            std::fill(deg.begin(), deg.end(), 0);
            for (int t = 0; t < T; ++t) {
                const int sp = P.owner[t];
                if (sp < 0) continue;
                for (int j : srcs[sp]) ++deg[static_cast<size_t>(t / lanes) * lanes + P.thread_of[j] % lanes];
            }
            long cost = 0;
            for (int pc = 0; pc < pieces; ++pc) {
                int worst = cap[pc];
                for (int b = 0; b < lanes; ++b) worst = std::max(worst, deg[static_cast<size_t>(pc) * lanes + b]);
                cost += worst;
                // second term: sum of squares breaks ties towards flatter banks
            }
            return cost;
        };
        uint32_t rng = 0x2545F491u;
        auto next = [&]() { rng = rng * 1664525u + 1013904223u; return rng >> 8; };
        long cost = total_cost();
        long floor_cost = 0;
        for (int pc = 0; pc < pieces; ++pc) floor_cost += cap[pc];
        for (int it = 0; it < 20000 && cost > floor_cost; ++it) {
            const int w = static_cast<int>(next() % P.W);
            const int t1 = w * 32 + static_cast<int>(next() % 32), t2 = w * 32 + static_cast<int>(next() % 32);
            if (t1 == t2 || t1 < P.nbs || t2 < P.nbs) continue;  // hubs stay on threads 0..2
            const int s1 = P.owner[t1], s2 = P.owner[t2];
            if (s1 < 0 && s2 < 0) continue;
            auto put = [&](int sp, int t) {
                P.owner[t] = sp;
                if (sp >= 0) P.thread_of[sp] = t;
            };
            put(s1, t2);
            put(s2, t1);
            const long c2 = total_cost();
            if (c2 <= cost) cost = c2;
            else {
                put(s1, t1);
                put(s2, t2);
            }
        }
    }

    // ---- P-slots and rate-sum lists ---------------------------------------------------
    struct Slot {
        int32_t rxn;
        uint16_t f1, f2;
        bool two;
    };
    struct NSlot {
        int32_t rxn;
        uint16_t f1;
    };
    std::vector<std::vector<Slot>> slots(T);
    std::vector<std::vector<NSlot>> nsl(T);
    std::vector<std::vector<std::vector<int32_t>>> agg(T, std::vector<std::vector<int32_t>>(kPullCoefs));
    // the constant one: YP[4T .. 4T+3]; second factors default to the copy in bank 3,
    // clear of the hub words 0..2 they are gathered next to
    const uint16_t one_word = static_cast<uint16_t>(4 * T);
    const uint16_t one_word2 = static_cast<uint16_t>(4 * T + 3);
    for (int r = 0; r < M; ++r) {  // reaction order = fixed, documented summation order
        const Rx& x = rx[r];
        const int t_own = P.thread_of[x.owner];
        const bool hh = x.hh_a >= 0;
        if (hh) {  // F- of the two reactants: k_a += nu R Y_b (twice the flux over Y_a when a == b)
            const int ta = P.thread_of[x.hh_a], tb = P.thread_of[x.hh_b];
            if (ta == tb) nsl[ta].push_back({r | (2 << 24), static_cast<uint16_t>(ta)});
            else {
                nsl[ta].push_back({r | (1 << 24), static_cast<uint16_t>(tb)});
                nsl[tb].push_back({r | (1 << 24), static_cast<uint16_t>(ta)});
            }
        } else {
            agg[t_own][x.cls].push_back(r | (1 << 24));
        }
        for (int q = 0; q < n_prod[r]; ++q) {
            const int s = prod[r * kMaxProd + q];
            bool first = true;
            int nu = 0;
            for (int u = 0; u < q; ++u) first = first && prod[r * kMaxProd + u] != s;
            if (!first) continue;
            for (int u = 0; u < n_prod[r]; ++u) nu += prod[r * kMaxProd + u] == s;
            const int h = hub_index[s];
            if (hh) {  // any product, a hub's own thread included: R * Y_a * Y_b at the consumer
                Slot sl;
                sl.rxn = r | (nu << 24);
                sl.f1 = static_cast<uint16_t>(P.thread_of[x.hh_a]);
                sl.two = true;
                sl.f2 = static_cast<uint16_t>(P.thread_of[x.hh_b]);
                slots[P.thread_of[s]].push_back(sl);
            } else if (h >= 0) {
                int slot;
                if (x.nco == 0) slot = 10 + h;
                else if (x.nco == 1 && x.co[0] != h) {
                    const int j = x.co[0] - (x.co[0] > h ? 1 : 0);  // index among the other two hubs
                    slot = 13 + 2 * h + j;
                } else
                    return reject("reaction " + std::to_string(r) +
                                  " makes a hub next to two hub co-reactants or to itself");
                agg[t_own][slot].push_back(r | (nu << 24));
            } else {
                Slot sl;
                sl.rxn = r | (nu << 24);
                const int c1 = x.nco == 0 ? 0 : 1 + x.co[0];
                sl.f1 = static_cast<uint16_t>(c1 * T + t_own);
                sl.two = x.nco == 2;
                sl.f2 = sl.two ? static_cast<uint16_t>(P.thread_of[P.hub[x.co[1]]]) : one_word;
                slots[P.thread_of[s]].push_back(sl);
            }
        }
    }
    P.n_slots.assign(T, 0);
    P.n_slots2.assign(T, 0);
    P.agg_max = 0;
    for (int t = 0; t < T; ++t) {
        int n2 = 0;
        for (const Slot& sl : slots[t]) n2 += sl.two;
        P.slots = std::max<int>(P.slots, slots[t].size());
        P.slots2 = std::max(P.slots2, n2);
        int tot = 0;
        for (const auto& v : agg[t]) tot += static_cast<int>(v.size());
        P.agg_max = std::max(P.agg_max, tot);
    }
    if (P.slots > kPullMaxSlots)
        return reject("a non-hub species has more than " + std::to_string(kPullMaxSlots) +
                      " incoming reactions");
    if (P.slots2 > kPullMaxSlots2)
        return reject("a non-hub species has more than " + std::to_string(kPullMaxSlots2) +
                      " incoming three-body reactions");
    if (P.agg_max > 65535) return reject("rate-sum list too long");
    for (int t = 0; t < T; ++t) P.nslots = std::max<int>(P.nslots, nsl[t].size());
    if (P.nslots > kPullNSlots)
        return reject("a species enters more than " + std::to_string(kPullNSlots) +
                      " reactions with another non-hub reactant");

    // ---- positions: bank-conflict-aware order of every thread's slots ------------------
    const int lanes = 128 / elem_bytes;
    std::vector<std::vector<int>> pos(T);
    std::vector<int> warp_cap(P.W, 0);
    for (int w = 0; w < P.W; ++w) {
        int most = 0, most2 = 0;
        for (int l = 0; l < 32; ++l) {
            int n2 = 0;
            for (const Slot& sl : slots[w * 32 + l]) n2 += sl.two;
            most = std::max<int>(most, slots[w * 32 + l].size());
            most2 = std::max(most2, n2);
        }
        const int cap = (most + 3) / 4 * 4, cap2 = std::min(cap, (most2 + 3) / 4 * 4);
        warp_cap[w] = cap;
        for (int piece = 0; piece < 32 / lanes; ++piece)
            place_piece(slots, w * 32 + piece * lanes, lanes, cap, cap2, pos);
    }
    P.slots = P.slots2 = 0;
    for (int t = 0; t < T; ++t)
        for (int p = 0; p < static_cast<int>(pos[t].size()); ++p) {
            if (pos[t][p] < 0) continue;
            P.n_slots[t] = static_cast<uint8_t>(p + 1);
            if (slots[t][pos[t][p]].two) P.n_slots2[t] = static_cast<uint8_t>(p + 1);
        }
    for (int t = 0; t < T; ++t) {
        P.slots = std::max<int>(P.slots, P.n_slots[t]);
        P.slots2 = std::max<int>(P.slots2, P.n_slots2[t]);
    }
    const int ns = std::max(1, P.slots), ns2 = std::max(1, P.slots2);
    P.slot_rxn.assign(static_cast<size_t>(ns) * T, -1);
    P.slot_f1.assign(static_cast<size_t>(ns) * T, one_word);
    P.slot_f2.assign(static_cast<size_t>(ns2) * T, one_word2);
    P.agg_ptr.assign(static_cast<size_t>(kPullCoefs + 1) * T, 0);
    P.agg_ent.assign(static_cast<size_t>(std::max(1, P.agg_max)) * T, 0);
    for (int t = 0; t < T; ++t) {
        for (int p = 0; p < static_cast<int>(pos[t].size()) && p < ns; ++p) {
            const int sidx = pos[t][p];
            if (sidx < 0) continue;
            const Slot& sl = slots[t][sidx];
            P.slot_rxn[static_cast<size_t>(p) * T + t] = sl.rxn;
            P.slot_f1[static_cast<size_t>(p) * T + t] = sl.f1;
            if (sl.two) P.slot_f2[static_cast<size_t>(p) * T + t] = sl.f2;
        }
        int q = 0;
        for (int c = 0; c < kPullCoefs; ++c) {
            P.agg_ptr[static_cast<size_t>(c) * T + t] = static_cast<uint16_t>(q);
            for (int32_t v : agg[t][c]) P.agg_ent[static_cast<size_t>(q++) * T + t] = v;
        }
        P.agg_ptr[static_cast<size_t>(kPullCoefs) * T + t] = static_cast<uint16_t>(q);
    }
    P.n_nslots.assign(T, 0);
    P.nslot_rxn.assign(static_cast<size_t>(kPullNSlots) * T, -1);
    P.nslot_f1.assign(static_cast<size_t>(kPullNSlots) * T, one_word);
    for (int t = 0; t < T; ++t) {
        P.n_nslots[t] = static_cast<uint8_t>(nsl[t].size());
        for (size_t e = 0; e < nsl[t].size(); ++e) {
            P.nslot_rxn[e * T + t] = nsl[t][e].rxn;
            P.nslot_f1[e * T + t] = nsl[t][e].f1;
        }
    }
    // holes (rate 0): read a word some lane of the same piece reads at that position
    // anyway, so that the hole costs no wavefront of its own
    for (int t0 = 0; t0 < T; t0 += lanes)
        for (int p = 0; p < ns; ++p) {
            int donor = -1;
            for (int l = 0; l < lanes && donor < 0; ++l)
                if (P.slot_rxn[static_cast<size_t>(p) * T + t0 + l] >= 0) donor = t0 + l;
            if (donor < 0) continue;
            for (int l = 0; l < lanes; ++l)
                if (P.slot_rxn[static_cast<size_t>(p) * T + t0 + l] < 0)
                    P.slot_f1[static_cast<size_t>(p) * T + t0 + l] =
                        P.slot_f1[static_cast<size_t>(p) * T + donor];
        }
    pull_wavefronts(P, elem_bytes, P.conflict_wavefronts, P.ideal_wavefronts);
    P.ok = true;
}

}  // namespace kinnet