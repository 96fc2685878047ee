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

    // ---- packed tables for the register-resident kernel ---------------------
    S.plus_max = *std::max_element(S.small_plus.begin(), S.small_plus.end());
    S.minus_max = *std::max_element(S.small_minus.begin(), S.small_minus.end());
    S.bigrow_max = 0;
    for (uint8_t c : S.big_cnt) S.bigrow_max = std::max<int>(S.bigrow_max, c);
    S.fast_ok = N <= 1023 && S.rs <= kFastSlots && S.rs <= 15 && S.j3 <= kFastSlots3 &&
                S.plus_max <= kFastPlus && S.minus_max <= kFastMinus &&
                S.bigrow_max <= kFastRowCap && (S.rs + 1) * T * 8 <= 65535;
    return NET_OK;
}

// Packed tables of the register-resident kernel.  Offsets are BYTE offsets for
// elements of `elem` bytes (8: double, 4: float).  Gather lists are padded to
// their capacity with the offset of the thread's own word in the all-zero flux
// row `rs`, readback lists with the slot id `rs`, so the kernel needs no
// per-lane predicates.
void pack_fast_tables(Schedule& S, int elem) {
    const int T = S.T, slots = S.rs * T;
    const uint32_t e32 = static_cast<uint32_t>(elem);
    S.fx_pack.assign(static_cast<size_t>(S.rs) * T, 0);
    S.fxc_pack.assign(static_cast<size_t>(kFastSlots3) * T, 0);
    for (int idx = 0; idx < slots; ++idx) {
        const uint16_t* re = &S.flux_react[static_cast<size_t>(idx) * 4];
        S.fx_pack[idx] = re[0] * e32 | (re[1] * e32) << 16;
        if (idx / T < kFastSlots3) S.fxc_pack[idx] = re[2] * e32;
    }
    S.plus_pack.assign(static_cast<size_t>(kFastPlus / 2) * T, 0);
    S.minus_pack.assign(static_cast<size_t>(kFastMinus / 2) * T, 0);
    S.rb_pack.assign(static_cast<size_t>(2 * kMaxBigSpecies) * T, 0);
    S.cnt_pack.assign(T, 0);
    S.rbcnt_pack.assign(T, 0);
    for (int t = 0; t < T; ++t) {
        const uint32_t zero_off = static_cast<uint32_t>(S.rs * T + t) * e32;
        const int np = S.small_plus[t], nm = S.small_minus[t];
        for (int e = 0; e < kFastPlus; ++e) {
            const uint32_t off = e < np ? S.small_src[static_cast<size_t>(e) * T + t] * e32 : zero_off;
            S.plus_pack[static_cast<size_t>(e / 2) * T + t] |= off << (16 * (e & 1));
        }
        for (int e = 0; e < kFastMinus; ++e) {
            const uint32_t off =
                e < nm ? S.small_src[static_cast<size_t>(np + e) * T + t] * e32 : zero_off;
            S.minus_pack[static_cast<size_t>(e / 2) * T + t] |= off << (16 * (e & 1));
        }
        S.cnt_pack[t] = static_cast<uint32_t>(np) | static_cast<uint32_t>(nm) << 8;
        int e = 0;
        for (int b = 0; b < 2 * kMaxBigSpecies; ++b) {
            const int c = b < 2 * S.nbs ? S.big_cnt[static_cast<size_t>(b) * T + t] : 0;
            for (int q = 0; q < kFastRowCap; ++q) {
                const uint32_t sid = q < c ? S.big_slot[static_cast<size_t>(e + q) * T + t]
                                           : static_cast<uint32_t>(S.rs);
                S.rb_pack[static_cast<size_t>(b) * T + t] |= sid << (4 * q);
            }
            e += c;
            S.rbcnt_pack[t] |= static_cast<uint32_t>(c) << (4 * b);
        }
    }
}

}  // namespace kinnet