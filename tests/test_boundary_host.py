"""CPU-only checks of the C-ABI library: it loads, exports what include/kinnet.h
declares, rejects bad tables, and its compiled schedule (the host half of the
hot path) contains every (species, sign, reaction) entry exactly once."""
import os
import re
from collections import Counter

import numpy as np
import pytest

import paper_1409_5826_b200 as K
from gen import make_toy
from gen.configs import network

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "kinnet.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(net_[a-z_]+)\s*\(", header))
    assert declared == set(K.EXPORTS)
    for name in declared:
        assert hasattr(K.lib, name), name


def test_default_params():
    p = K.net_default_params()
    assert (p.kappa, p.eps_y, p.y_floor, p.growth, p.max_steps, p.precision, p.kernel, p.host_chunk,
            p.method) == (1.0, 0.05, 1e-10, 2.0, 10_000_000, 64, 0, 0, 0)


def test_integrate_without_device_copy_fails_loudly(g16):
    net = K.Net(g16, host_only=True)
    z = np.zeros(1)
    with pytest.raises(K.KinnetError) as e:
        net.net_integrate(1, z, z, np.zeros(16), 1e-6, stream=0)
    assert e.value.code == K.NET_ECUDA and "no device copy" in str(e.value)


def _broken(net, **kw):
    import copy

    bad = copy.deepcopy(net)
    for k, v in kw.items():
        setattr(bad, k, v)
    return bad


def test_invalid_tables_are_rejected(g16):
    re_ = g16.react.copy()
    re_[0, 0] = 99
    with pytest.raises(K.KinnetError) as e:
        K.Net(_broken(g16, react=re_), host_only=True)
    assert e.value.code == K.NET_EINVAL and "reactant index" in str(e.value)
    nr = g16.n_react.copy()
    nr[3] = 4
    with pytest.raises(K.KinnetError):
        K.Net(_broken(g16, n_react=nr), host_only=True)
    npd = g16.n_prod.copy()
    npd[3] = 0
    with pytest.raises(K.KinnetError):
        K.Net(_broken(g16, n_prod=npd), host_only=True)
    A = g16.A.copy()
    A[5] += 1
    with pytest.raises(K.KinnetError) as e:
        K.Net(_broken(g16, A=A), host_only=True)
    assert "conserve" in str(e.value)
    co = g16.coef.copy()
    co[0, 0] = np.nan
    with pytest.raises(K.KinnetError):
        K.Net(_broken(g16, coef=co), host_only=True)
    with pytest.raises(K.KinnetError):
        K.Net(g16, K.NetParams(precision=16), host_only=True)
    with pytest.raises(K.KinnetError):
        K.Net(g16, K.NetParams(kappa=0.0), host_only=True)


def expected_entries(net):
    ent = Counter()
    for r in range(net.n_reactions):
        for s in net.react[r, : net.n_react[r]]:
            ent[(int(s), "-", r)] += 1
        for s in net.prod[r, : net.n_prod[r]]:
            ent[(int(s), "+", r)] += 1
    return ent


def schedule_entries(net, kn):
    info = kn.schedule_info()
    T = info["threads"]
    rxn = kn.schedule_table("flux_rxn")
    owner = kn.schedule_table("owner")
    sp, sm = kn.schedule_table("small_plus"), kn.schedule_table("small_minus")
    src = kn.schedule_table("small_src").reshape(-1, T) if info["small_max"] else None
    ent = Counter()
    for t in range(T):
        for e in range(sp[t] + sm[t]):
            assert owner[t] >= 0
            r = rxn[src[e, t]]
            assert r >= 0
            ent[(int(owner[t]), "+" if e < sp[t] else "-", int(r))] += 1
    nbs = info["n_big_species"]
    if nbs:
        bs = kn.schedule_table("big_species")
        cnt = kn.schedule_table("big_cnt").reshape(2 * nbs, T)
        slot = kn.schedule_table("big_slot").reshape(-1, T)
        for t in range(T):
            e = 0
            for b in range(2 * nbs):
                for _ in range(cnt[b, t]):
                    r = rxn[slot[e, t] * T + t]  # own column only
                    assert r >= 0
                    ent[(int(bs[b // 2]), "+" if b % 2 == 0 else "-", int(r))] += 1
                    e += 1
            assert e <= info["readback_max"]
    return ent, info


@pytest.mark.parametrize("name", ["g16", "hub150", "hub365"])
def test_schedule_round_trip(name):
    net = network(name)
    kn = K.Net(net, K.NetParams(kernel=1), host_only=True)  # the generic schedule
    got, info = schedule_entries(net, kn)
    want = expected_entries(net)
    assert got == want
    assert info["n_entries"] == sum(want.values())
    T, rs = info["threads"], info["flux_slots"]
    assert T % 32 == 0 and T >= net.n_species and rs * T >= net.n_reactions
    # every reaction sits in exactly one flux slot, with its reactants in order
    rxn = kn.schedule_table("flux_rxn")
    assert sorted(r for r in rxn if r >= 0) == list(range(net.n_reactions))
    fr = kn.schedule_table("flux_react").reshape(-1, 3)
    for idx, r in enumerate(rxn):
        j = idx // T
        if r < 0:
            assert (fr[idx] == net.n_species).all()
            continue
        n = net.n_react[r]
        assert list(fr[idx, :n]) == list(net.react[r, :n]) and (fr[idx, n:] == net.n_species).all()
        assert n == 1 or j < info["slots_2body"]
        assert n <= 2 or j < info["slots_3body"]
    # each species has exactly one owner thread; big species sit at W .. W+nbs-1
    owner = kn.schedule_table("owner")
    assert sorted(o for o in owner if o >= 0) == list(range(net.n_species))
    W = T // 32
    if info["n_big_species"]:
        assert list(owner[W: W + info["n_big_species"]]) == list(kn.schedule_table("big_species"))


def test_schedule_hub_rows_are_the_big_ones(hub150):
    """p, n, 4He have hundreds of fluxes, the rest a few tens."""
    kn = K.Net(hub150, K.NetParams(kernel=1), host_only=True)
    info = kn.schedule_info()
    assert list(kn.schedule_table("big_species")) == [0, 1, 2]
    assert info["n_entries_big"] > 0.35 * info["n_entries"]
    assert info["small_max"] <= 40
    # readback lists are balanced: within 2x of the mean
    assert info["readback_max"] <= 2 * info["n_entries_big"] / info["threads"] + 2


def test_three_alpha_multiplicity_in_schedule():
    """3a -> C and back: the alpha rows receive the flux three times (S:Q2)."""
    net = make_toy([4, 12], [((0, 0, 0), (1,)), ((1,), (0, 0, 0))], [7.0, 0.5])
    kn = K.Net(net, K.NetParams(kernel=1), host_only=True)
    got, _ = schedule_entries(net, kn)
    assert got[(0, "-", 0)] == 3 and got[(0, "+", 1)] == 3 and got[(1, "+", 0)] == 1


# ------------------------------------------------------------------ pull schedule
PAIRS = {4: (0, 0), 5: (0, 1), 6: (0, 2), 7: (1, 1), 8: (1, 2), 9: (2, 2)}


def pull_entries(net, kn):
    """Every (species, sign, reaction) term the pull kernel accounts for, rebuilt
    from its tables alone: P-slots give F+ of non-hub species (and of hubs made by
    heavy + heavy reactions); rate-sum coefficient K_c gives the owner's F- and the
    F- of the hubs in class c; G0/Gx give F+ of the hubs; N-slots give F- of the two
    non-hub reactants of a heavy + heavy reaction."""
    info = kn.schedule_info()
    assert info["pull_ok"] == 1
    T = info["pull_threads"]
    assert T == info["threads"] * (2 if info["kernel"] == 2 else 1)
    hub = list(kn.schedule_table("pull_hub"))
    owner = kn.schedule_table("pull_owner")
    ns, ns2 = kn.schedule_table("pull_n_slots"), kn.schedule_table("pull_n_slots2")
    rxn = kn.schedule_table("pull_slot_rxn").reshape(-1, T)
    f1 = kn.schedule_table("pull_slot_f1").reshape(-1, T)
    f2 = kn.schedule_table("pull_slot_f2").reshape(-1, T)
    ptr = kn.schedule_table("pull_agg_ptr").reshape(20, T)
    agg = kn.schedule_table("pull_agg_ent").reshape(-1, T)
    assert sorted(o for o in owner if o >= 0) == list(range(net.n_species))
    assert list(owner[: len(hub)]) == hub  # hub h on thread h
    ent = Counter()
    for t in range(T):
        assert ns2[t] <= ns[t] <= info["pull_slots"]
        for e in range(rxn.shape[0]):
            if rxn[e, t] == -1:  # hole: rate 0, any finite word
                assert f1[e, t] <= 4 * T and (e >= f2.shape[0] or f2[e, t] == 4 * T + 3)
                continue
            assert e < ns[t]
            assert owner[t] >= 0
            r, nu = int(rxn[e, t]) & 0xFFFFFF, int(rxn[e, t]) >> 24
            ent[(int(owner[t]), "+", r)] += nu
            # the factors of the slot reproduce the reactant multiset of the reaction
            c1, t1 = divmod(int(f1[e, t]), T)
            react = [int(owner[t1])] + ([hub[c1 - 1]] if c1 else [])
            if e < f2.shape[0] and f2[e, t] != 4 * T + 3:  # second factor: a species' own word
                assert e < ns2[t] and f2[e, t] < T
                react.append(int(owner[f2[e, t]]))
            assert sorted(react) == sorted(int(s) for s in net.react[r, : net.n_react[r]])
            heavy = [x for x in react if x not in hub]
            # a hub's own thread gathers only what heavy + heavy reactions make of it
            assert owner[t] not in hub or len(heavy) == 2
        for s in range(19):
            for q in range(ptr[s, t], ptr[s + 1, t]):
                r, nu = int(agg[q, t]) & 0xFFFFFF, int(agg[q, t]) >> 24
                if s < 10:
                    assert nu == 1
                    ent[(int(owner[t]), "-", r)] += 1
                    co = [] if s == 0 else [s - 1] if s < 4 else list(PAIRS[s])
                    for h in co:
                        ent[(hub[h], "-", r)] += 1
                    assert sorted([int(owner[t])] + [hub[h] for h in co]) == sorted(
                        int(x) for x in net.react[r, : net.n_react[r]])
                elif s < 13:
                    ent[(hub[s - 10], "+", r)] += nu
                    assert net.n_react[r] == 1
                else:
                    h, j = divmod(s - 13, 2)
                    other = [x for x in range(3) if x != h][j]
                    ent[(hub[h], "+", r)] += nu
                    assert sorted(int(x) for x in net.react[r, :2]) == sorted([int(owner[t]), hub[other]])
    nn = kn.schedule_table("pull_n_nslots")
    nrx = kn.schedule_table("pull_nslot_rxn").reshape(4, T)
    nf1 = kn.schedule_table("pull_nslot_f1").reshape(4, T)
    assert nn.max(initial=0) == info["pull_nslots"]
    for t in range(T):
        for e in range(4):
            if nrx[e, t] == -1:
                assert e >= nn[t] and nf1[e, t] == 4 * T
                continue
            assert e < nn[t] and owner[t] >= 0 and owner[t] not in hub and nf1[e, t] < T
            r, nu = int(nrx[e, t]) & 0xFFFFFF, int(nrx[e, t]) >> 24
            partner = int(owner[nf1[e, t]])
            assert partner not in hub and net.n_react[r] == 2
            assert sorted([int(owner[t]), partner]) == sorted(int(x) for x in net.react[r, :2])
            assert nu == (2 if partner == owner[t] else 1)
            ent[(int(owner[t]), "-", r)] += nu
    return ent, info


def test_pull_schedule_heavy_pairs():
    """hub150hh: 16 reactions with two non-hub reactants (one of them an identical pair) and
    their inverses stay on the two-species pull kernel; every term is still there once."""
    net = network("hub150hh")
    heavy = [r for r in range(net.n_reactions)
             if sum(1 for s in net.react[r, : net.n_react[r]] if s >= 3) == 2]
    assert len(heavy) == 16 and any(net.react[r, 0] == net.react[r, 1] for r in heavy)
    kn = K.Net(net, host_only=True)
    got, info = pull_entries(net, kn)
    assert got == expected_entries(net)
    assert info["kernel"] == 2 and 1 <= info["pull_nslots"] <= 4
    # the one-species kernel is not instantiated with N-slots: generic fallback
    assert K.Net(net, K.NetParams(kernel=2), host_only=True).schedule_info()["kernel"] == 0


@pytest.mark.parametrize("kernel", [0, 2])
@pytest.mark.parametrize("name", ["hub150", "hub365", "hub150+perm"])
def test_pull_schedule_round_trip(name, kernel):
    """kernel = 0 compiles the schedule for virtual threads (two per thread, kernel 2 in
    schedule_info) where an instantiation covers it; kernel = 2 asks for the one-species one."""
    net = network("hub150").permuted(7)[0] if name.endswith("+perm") else network(name)
    kn = K.Net(net, K.NetParams(kernel=kernel), host_only=True)
    got, info = pull_entries(net, kn)
    assert got == expected_entries(net)
    assert info["kernel"] == (2 if kernel == 0 else 1) and info["pull_hubs"] == 3
    assert info["pull_wavefronts"] >= info["pull_wavefronts_ideal"] > 0


def test_pull_schedule_small_and_unsupported_networks(g16):
    # no hubs, one non-hub reactant per reaction: qualifies with zero hubs
    net = make_toy([1, 1, 1], [((0,), (1,)), ((1,), (0,)), ((1,), (2,))], [2.0, 3.0, 0.5])
    kn = K.Net(net, host_only=True)
    got, info = pull_entries(net, kn)
    assert got == expected_entries(net) and info["pull_hubs"] == 0 and info["kernel"] in (1, 2)
    # two non-hub reactants: generic flux-array kernel
    info = K.Net(g16, host_only=True).schedule_info()
    assert info["pull_ok"] == 0 and info["kernel"] == 0
    with pytest.raises(K.KinnetError):
        K.Net(g16, host_only=True).schedule_table("pull_owner")
    # kernel = 1 forces the generic kernel even when the network qualifies
    info = K.Net(network("hub150"), K.NetParams(kernel=1), host_only=True).schedule_info()
    assert info["pull_ok"] == 1 and info["kernel"] == 0


def test_staircase_class_of_the_two_species_schedule():
    """S0 host logic behind KPull.stair (include/kinnet.h, net_schedule_info_t.pull_stair): the class is
    recomputed here from the schedule tables alone.  hub150: every side fits its step and warp 0 plays
    no species on side b; hub150hh: warp 1's side b (up to 10 slots) overflows its step of 8; g16 does
    not run on the two-species kernel at all."""
    from gen.configs import network

    def want(kn, info, cap_b=12):
        n, own = kn.schedule_table("pull_n_slots"), kn.schedule_table("pull_owner")
        nw = info["pull_threads"] // 64
        if info["threads"] > 128:  # 160/192-thread blocks run the branching loop: no per-warp copies
            return 0
        cap_a = 20 if n[: 32 * nw].max() <= 20 else 24
        cls = 1 | 2
        for t, (slots, o) in enumerate(zip(n, own)):
            vw = t // 32
            if vw < nw:
                if slots > max(cap_a - 4 * vw, 12):
                    return 0
            else:
                w = 2 * nw - 1 - vw
                if slots > max(cap_b - 4 * (nw - 1 - w), 4):
                    cls |= 1 << (8 + w)
                if w == 0 and o >= 0:
                    cls &= ~2
        return cls

    seen = {}
    for name in ("hub150", "hub150hh", "hub365"):
        kn = K.Net(network(name), host_only=True)
        info = kn.schedule_info()
        assert info["kernel"] == 2 and info["pull_ok"] == 1
        assert info["pull_stair"] == want(kn, info), name
        seen[name] = info["pull_stair"]
    assert seen["hub150"] == 3                      # fits, warp 0 one-sided
    assert seen["hub150hh"] == 3 | 1 << 9           # warp 1's side b at full capacity
    # hub365 runs 192-thread blocks, which are not compiled with per-warp loop copies: the reported
    # class must say so, whatever its slot counts would allow
    assert seen["hub365"] == 0 and K.Net(network("hub365"), host_only=True).schedule_info()["threads"] == 192
    assert K.Net(network("g16"), host_only=True).schedule_info()["pull_stair"] == 0
    # negative case inside the eligible block sizes: the 250-species network runs 128 threads, but a
    # side-a row overflows its warp's step -> class 0 (recomputed from the tables above)
    from gen import make_hub_network

    kn = K.Net(make_hub_network(250, 2900, seed=250), host_only=True)
    info = kn.schedule_info()
    assert info["kernel"] == 2 and info["threads"] == 128 and info["pull_stair"] == 0 == want(kn, info)
    n = kn.schedule_table("pull_n_slots")
    assert any(n[t] > max(24 - 4 * (t // 32), 12) for t in range(32 * (info["pull_threads"] // 64)))
