"""Seeded synthetic reaction networks with the shapes of the paper's workloads.

The paper's real 150- and 365-isotope networks (§6) are not
available; these generators stand in for them and reproduce their *shape*:
species/reaction counts (150/1604, 365/~4400), three hub species ("n", "p",
"alpha"-like) with hundreds of fluxes each while the rest have a few tens
(§11 item 5), and very stiff rate spreads.  Every reaction
conserves nucleon number, sum(A reactants) == sum(A products).

Only table construction lives here.  The single expression borrowed from the
method is the value of the 7-parameter log-rate at one reference point, needed
to solve a0 so that a reaction's rate hits its drawn target there (recipe in
SURVEY.md §8(d), restated in DESIGN.md).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from math import factorial, log

import numpy as np

MAX_REACT = 3
MAX_PROD = 4
N_COEF = 7


@dataclass
class Network:
    """Plain tables of one network (what ``net_create`` takes).

    A        [N]   int32  mass numbers
    n_react  [M]   int32  reactants per reaction, 1..3
    react    [M,3] int32  reactant species (repeats allowed), pad = -1
    n_prod   [M]   int32  products per reaction, 1..4
    prod     [M,4] int32  product species (repeats allowed), pad = -1
    coef     [M,7] f64    a0..a6 of the 7-parameter rate form
    """

    A: np.ndarray
    n_react: np.ndarray
    react: np.ndarray
    n_prod: np.ndarray
    prod: np.ndarray
    coef: np.ndarray
    name: str = ""
    meta: dict = field(default_factory=dict)

    @property
    def n_species(self) -> int:
        return int(self.A.shape[0])

    @property
    def n_reactions(self) -> int:
        return int(self.n_react.shape[0])

    def check(self) -> None:
        N, M = self.n_species, self.n_reactions
        assert self.react.shape == (M, MAX_REACT) and self.prod.shape == (M, MAX_PROD)
        assert self.coef.shape == (M, N_COEF)
        for r in range(M):
            nr, npd = int(self.n_react[r]), int(self.n_prod[r])
            assert 1 <= nr <= MAX_REACT and 1 <= npd <= MAX_PROD
            re, pr = self.react[r, :nr], self.prod[r, :npd]
            assert (re >= 0).all() and (re < N).all() and (pr >= 0).all() and (pr < N).all()
            assert (self.react[r, nr:] == -1).all() and (self.prod[r, npd:] == -1).all()
            assert self.A[re].sum() == self.A[pr].sum(), f"reaction {r} does not conserve A"

    def permuted(self, seed: int) -> tuple["Network", np.ndarray]:
        """Same network with reactions shuffled and species relabelled.

        Returns (network, sigma) with new species index sigma[i] for old i.
        """
        rng = np.random.default_rng(seed)
        N, M = self.n_species, self.n_reactions
        sigma = rng.permutation(N).astype(np.int32)
        order = rng.permutation(M)
        A = np.empty_like(self.A)
        A[sigma] = self.A

        def relabel(tab):
            out = tab.copy()
            mask = out >= 0
            out[mask] = sigma[out[mask]]
            return out

        net = Network(
            A=A,
            n_react=self.n_react[order].copy(),
            react=relabel(self.react[order]),
            n_prod=self.n_prod[order].copy(),
            prod=relabel(self.prod[order]),
            coef=self.coef[order].copy(),
            name=self.name + f"+perm{seed}",
            meta=dict(self.meta),
        )
        return net, sigma


def _stat_log_prefactor(reactants) -> float:
    """ln(1/prod m_s!) over distinct reactant species."""
    out = 0.0
    for s in set(reactants):
        out -= log(factorial(list(reactants).count(s)))
    return out


def _pack(A, reactions, coefs, name, meta) -> Network:
    M = len(reactions)
    n_react = np.zeros(M, np.int32)
    n_prod = np.zeros(M, np.int32)
    react = -np.ones((M, MAX_REACT), np.int32)
    prod = -np.ones((M, MAX_PROD), np.int32)
    for r, (re, pr) in enumerate(reactions):
        n_react[r], n_prod[r] = len(re), len(pr)
        react[r, : len(re)] = re
        prod[r, : len(pr)] = pr
    net = Network(
        A=np.asarray(A, np.int32),
        n_react=n_react,
        react=react,
        n_prod=n_prod,
        prod=prod,
        coef=np.asarray(coefs, np.float64).reshape(M, N_COEF),
        name=name,
        meta=meta,
    )
    net.check()
    return net


def _draw_coefs(rng, reactions, lo, hi, T9ref, rhoref, charged, a2_all=None):
    """Seven coefficients per reaction (recipe: SURVEY §8(d) "Coefficients").

    a1..a6 are drawn; a0 is solved so that the full rate, including the
    statistical prefactor and rho^(n-1), equals 10^u at (T9ref, rhoref) with
    u ~ U[lo, hi].
    """
    t13 = T9ref ** (1.0 / 3.0)
    coefs = []
    for re, pr in reactions:
        n = len(re)
        u = rng.uniform(lo, hi)
        threshold_like = n == 1 and len(pr) >= 2
        a1 = -rng.uniform(0.0, 40.0) if threshold_like else -rng.uniform(0.0, 5.0)
        if a2_all is not None:
            a2 = -rng.uniform(0.0, a2_all) if n >= 2 else 0.0
        elif n >= 2 and any(s in charged for s in re):
            a2 = -rng.uniform(0.0, 40.0)
        else:
            a2 = 0.0
        a3 = rng.uniform(-2.0, 2.0)
        a4 = rng.uniform(-0.5, 0.5)
        a5 = rng.uniform(-0.05, 0.05)
        a6 = (-1.5, -2.0 / 3.0, 0.0, 1.5)[int(rng.integers(0, 4))]
        rest = (
            a1 / T9ref
            + a2 / t13
            + a3 * t13
            + a4 * T9ref
            + a5 * T9ref ** (5.0 / 3.0)
            + a6 * log(T9ref)
        )
        a0 = u * log(10.0) - rest - _stat_log_prefactor(re) - (n - 1) * log(rhoref)
        coefs.append((a0, a1, a2, a3, a4, a5, a6))
    return coefs


def make_g16(seed: int = 16) -> Network:
    """BASELINE.json configs[0]: 16 species, 48 reactions.

    A_i = 4(i+1).  The 64 triples i <= j with (i+1)+(j+1) = (k+1) <= 16 are
    the candidate captures i+j->k; 32 are kept, and 16 of those also get their
    inverse decay k->i+j.  Rates span 1e-6..1e6 s^-1 at (T9, rho) = (3, 1e8).
    """
    rng = np.random.default_rng(seed)
    A = [4 * (i + 1) for i in range(16)]
    cand = [(i, j, i + j + 1) for i in range(16) for j in range(i, 16) if i + j + 1 < 16]
    assert len(cand) == 64
    cap = [cand[c] for c in sorted(rng.choice(64, size=32, replace=False))]
    inv = [cap[c] for c in sorted(rng.choice(32, size=16, replace=False))]
    reactions = [((i, j), (k,)) for i, j, k in cap] + [((k,), (i, j)) for i, j, k in inv]
    order = rng.permutation(len(reactions))
    reactions = [reactions[o] for o in order]
    coefs = _draw_coefs(rng, reactions, -6.0, 6.0, 3.0, 1e8, charged=(), a2_all=10.0)
    return _pack(A, reactions, coefs, "g16", {"seed": seed, "T9ref": 3.0, "rhoref": 1e8})


def make_hub_network(
    N: int,
    M: int,
    seed: int,
    lo: float = -5.0,
    hi: float = 10.0,
    T9ref: float = 5.0,
    rhoref: float = 1e9,
    heavy_pairs: int = 0,
) -> Network:
    """Hub network G(N, M, seed, lo, hi, T9ref, rhoref) of SURVEY §8(d).

    Species 0, 1 have A = 1 ("n"-, "p"-like), species 2 has A = 4
    ("alpha"-like); heavy species h = 0..N-4 sit at index 3+h with
    A = 12 + h // w, w = 3 isobars per A for N <= 200, else 5.
    Reaction families (quotas 30 % / 65 % / 5 % one-/two-/three-body):
      beta-like X -> X' (same A);
      capture X + l -> X'' paired with photodisintegration X'' -> X + l;
      exchange X + l -> X'' + l' paired with its inverse;
      three-body X + l + l' -> X'';
      fixed pair 3 alpha -> (first A=12) and back.
    heavy_pairs = k appends k heavy + heavy fusions X + X' -> X'' (+ l) among the light end of
    the heavy species (A <= 24: the 12C+12C, 12C+16O, 16O+16O class of the paper's Type Ia
    network), each paired with its inverse, from a separate seeded stream, at
    seeded positions of the reaction list: M + 2k reactions in all, the first M tables
    identical to heavy_pairs = 0.
    """
    assert N >= 32
    rng = np.random.default_rng(seed)
    w = 3 if N <= 200 else 5
    n_heavy = N - 3
    A = [1, 1, 4] + [12 + h // w for h in range(n_heavy)]
    a_light = (1, 1, 4)
    A_max = A[-1]
    iso: dict[int, list[int]] = {}
    for h in range(n_heavy):
        iso.setdefault(A[3 + h], []).append(3 + h)

    M1 = int(round(0.30 * M))
    M3 = int(round(0.05 * M))
    M2 = M - M1 - M3
    n_cap = int(round(0.75 * (M1 - 1)))
    if (M2 - n_cap) % 2:
        n_cap += 1
    n_beta = M1 - 1 - n_cap
    n_exch = (M2 - n_cap) // 2
    n_three = M3 - 1
    assert n_beta >= 0 and n_exch >= 0 and n_three >= 0

    seen = set()
    reactions = []

    def key(re, pr):
        return (tuple(sorted(re)), tuple(sorted(pr)))

    def try_add(*pairs):
        ks = [key(re, pr) for re, pr in pairs]
        if any(k in seen or k[0] == k[1] for k in ks) or len(set(ks)) != len(ks):
            return False
        for k, (re, pr) in zip(ks, pairs):
            seen.add(k)
            reactions.append((tuple(re), tuple(pr)))
        return True

    c12 = iso[12][0]
    assert try_add(((2, 2, 2), (c12,)), ((c12,), (2, 2, 2)))

    def heavy():
        return 3 + int(rng.integers(0, n_heavy))

    def pick(Aq, exclude=None):
        if Aq not in iso:
            return None
        pool = [s for s in iso[Aq] if s != exclude]
        if not pool:
            return None
        return pool[int(rng.integers(0, len(pool)))]

    def fill(count, draw):
        added, tries = 0, 0
        while added < count:
            tries += 1
            assert tries < 200 * (count + 10), "generator could not meet quota"
            pairs = draw()
            if pairs is not None and try_add(*pairs):
                added += 1

    def draw_beta():
        X = heavy()
        X2 = pick(A[X], exclude=X)
        return None if X2 is None else (((X,), (X2,)),)

    def draw_capture():
        X, l = heavy(), int(rng.integers(0, 3))
        X2 = pick(A[X] + a_light[l])
        return None if X2 is None else (((X, l), (X2,)), ((X2,), (X, l)))

    def draw_exchange():
        X, l = heavy(), int(rng.integers(0, 3))
        l2 = (l + 1 + int(rng.integers(0, 2))) % 3
        X2 = pick(A[X] + a_light[l] - a_light[l2], exclude=X)
        return None if X2 is None else (((X, l), (X2, l2)), ((X2, l2), (X, l)))

    def draw_three():
        X = heavy()
        l, l2 = sorted(int(v) for v in rng.integers(0, 3, size=2))
        X2 = pick(A[X] + a_light[l] + a_light[l2])
        return None if X2 is None else (((X, l, l2), (X2,)),)

    fill(n_beta, draw_beta)
    fill(n_cap, draw_capture)
    fill(n_exch, draw_exchange)
    fill(n_three, draw_three)
    assert len(reactions) == M and A_max == A[-1]

    order = rng.permutation(M)
    reactions = [reactions[o] for o in order]
    coefs = _draw_coefs(rng, reactions, lo, hi, T9ref, rhoref, charged=(1, 2))
    counts = [sum(1 for re, _ in reactions if len(re) == n) for n in (1, 2, 3)]
    meta = {
        "seed": seed,
        "T9ref": T9ref,
        "rhoref": rhoref,
        "body_counts": counts,
        "first_A12": c12,
        "first_A16": iso[16][0],
    }
    if heavy_pairs:
        rng2 = np.random.default_rng([seed, 0x4848])
        light_end = [s for s in range(3, N) if A[s] <= 24]
        extra = []
        tries = 0
        while len(extra) < 2 * heavy_pairs:
            tries += 1
            assert tries < 1000 * (heavy_pairs + 10), "generator could not place the heavy pairs"
            X, X1 = (light_end[int(v)] for v in rng2.integers(0, len(light_end), size=2))
            if not extra:
                X1 = X  # the first pair is an identical one (the 12C+12C shape: flux R Y^2/2, F- = 2f)
            l = int(rng2.integers(-1, 3))  # -1: pure fusion, else the emitted light particle
            X2 = pick_from(rng2, iso, A[X] + A[X1] - (a_light[l] if l >= 0 else 0))
            if X2 is None:
                continue
            pr = (X2,) if l < 0 else (X2, l)
            if try_add(((X, X1), pr), (pr, (X, X1))):
                extra += reactions[-2:]
                del reactions[-2:]
        coefs = list(coefs) + _draw_coefs(rng2, extra, lo, hi, T9ref, rhoref, charged=(1, 2))
        reactions = list(reactions) + extra
        order2 = rng2.permutation(len(reactions))
        reactions = [reactions[o] for o in order2]
        coefs = [coefs[o] for o in order2]
        meta["heavy_pairs"] = heavy_pairs
        return _pack(A, reactions, coefs, f"hub{N}_{M}hh{heavy_pairs}", meta)
    return _pack(A, reactions, coefs, f"hub{N}_{M}", meta)


def pick_from(rng, iso, Aq):
    """A seeded species of mass number Aq, or None."""
    pool = iso.get(Aq)
    return None if not pool else pool[int(rng.integers(0, len(pool)))]


def make_toy(A, reactions, rates, name="toy") -> Network:
    """Hand-built network with temperature-independent rates (a1..a6 = 0).

    ``rates[r]`` is the desired rate *including* the statistical prefactor at
    rho = 1, so a0 = ln(rate) - ln(prefactor).  Used by the pins and by tiny
    parity cases.
    """
    coefs = []
    for (re, _), k in zip(reactions, rates):
        coefs.append((log(k) - _stat_log_prefactor(re), 0, 0, 0, 0, 0, 0))
    return _pack(A, [(tuple(r), tuple(p)) for r, p in reactions], coefs, name, {})
