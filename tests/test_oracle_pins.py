"""Pins P1-P10 of SURVEY.md §8(c): the oracle against what the paper and the
mathematics fix (closed forms, fixed points, invariants, brute force).

None of these re-types the oracle's formula as the expectation: every expected
value comes from an independent route (long-double libm, an analytic closed
form, a dense matrix power, an RK4 integration of the ODE of PAPER.md Eq. (1)).
"""
from math import factorial

import numpy as np
import pytest

from gen import Network, make_toy
from gen.network import _pack
from oracle import Oracle, OracleParams


def toy_with_coefs(A, reactions, coefs):
    return _pack(A, reactions, coefs, "toy", {})


# ---------------------------------------------------------------- P1: rates
def test_p1_rate_constant_coefficients():
    """a1..a6 = 0  =>  R = p * rho^(n-1) * exp(a0), p = 1/prod(m!)  (S:Q1, Q2)."""
    A = [1, 1, 2, 3, 4]
    reactions = [
        ((0,), (1,)),          # 1-body, p = 1
        ((0, 1), (2,)),        # 2-body distinct, p = 1
        ((0, 0), (2,)),        # 2-body identical, p = 1/2
        ((0, 0, 0), (3,)),     # 3-body identical, p = 1/6
        ((0, 0, 2), (4,)),     # 3-body, one pair, p = 1/2
        ((0, 1, 2), (4,)),     # 3-body distinct, p = 1
    ]
    a0 = [0.3, -1.2, 2.0, 0.7, -0.4, 1.1]
    coefs = [(a, 0, 0, 0, 0, 0, 0) for a in a0]
    o = Oracle(toy_with_coefs(A, reactions, coefs))
    rho = 3.0e7
    R = o.rates(T9=2.7, rho=rho)
    pref = [1, 1, 1 / 2, 1 / 6, 1 / 2, 1]
    nre = [1, 2, 2, 3, 3, 3]
    expect = np.array([p * rho ** (n - 1) * np.exp(a) for p, n, a in zip(pref, nre, a0)])
    np.testing.assert_allclose(R, expect, rtol=1e-14)


def test_p1_rate_T9_one_and_eight():
    """T9 = 1: ln R = a0+..+a5.  T9 = 8: T9^(1/3) = 2 and T9^(5/3) = 32 exactly."""
    a = (0.5, -0.25, 0.125, 1.0, -0.5, 0.0625, 1.5)
    o = Oracle(toy_with_coefs([1, 1], [((0,), (1,))], [a]))
    R1 = o.rates(T9=1.0, rho=123.0)[0]
    assert R1 == pytest.approx(np.exp(sum(a[:6])), rel=1e-15)
    R8 = o.rates(T9=8.0, rho=123.0)[0]
    ln8 = a[0] + a[1] / 8 + a[2] / 2 + a[3] * 2 + a[4] * 8 + a[5] * 32 + a[6] * np.log(8.0)
    assert R8 == pytest.approx(np.exp(ln8), rel=4e-15)


def test_p1_rate_vs_long_double(hub150):
    """Cross-check O2 against 80-bit powl/expl/logl on the real tables."""
    o = Oracle(hub150)
    L = np.longdouble
    third = L(1) / L(3)
    for T9, rho in ((1.0, 1e7), (3.3, 2.2e8), (7.0, 1e8), (10.0, 3.1e9)):
        R = o.rates(T9, rho)
        T = L(T9)
        a = hub150.coef.astype(L)
        terms = np.stack([
            a[:, 0], a[:, 1] / T, a[:, 2] * T ** (-third), a[:, 3] * T ** third, a[:, 4] * T,
            a[:, 5] * T ** (L(5) * third), a[:, 6] * np.log(T),
        ], axis=1)
        lnp = np.array([
            -sum(np.log(L(factorial(list(re[:n]).count(s)))) for s in set(re[:n]))
            for re, n in zip(hub150.react, hub150.n_react)
        ], dtype=L)
        dens = (hub150.n_react.astype(L) - 1) * np.log(L(rho))
        expect = np.exp(terms.sum(axis=1) + lnp + dens)
        # one rounding (2^-53) per term of the exponent, amplified by its size
        scale = np.abs(terms).sum(axis=1) + np.abs(lnp) + np.abs(dens) + 1
        rel = np.abs((R.astype(L) - expect) / expect).astype(np.float64)
        assert (rel <= 8 * 2.0**-53 * scale.astype(np.float64)).all(), rel.max()


# ------------------------------------------------------ P2/P3: single decay
def decay_net(k):
    return make_toy([1, 1], [((0,), (1,))], [k])


@pytest.mark.parametrize("k,dt,branch", [(1.0, 0.25, "euler"), (1.0, 1.0, "asym"),
                                          (1.0, 4.0, "asym"), (2.0, 0.25, "euler")])
def test_p2_single_decay_discrete_closed_forms(k, dt, branch):
    """A -> B, F+_A = 0: Euler gives Y0 (1 - k dt)^n, Eq. (3) gives Y0/(1 + k dt)^n.
    k dt = 1 exactly must take the asymptotic branch ('>=')."""
    o = Oracle(decay_net(k))
    n, Y0 = 40, 0.75
    out = o.integrate_fixed(1.0, 1.0, [Y0, 0.0], dt, n)
    YA, YB = out["Y"][0]
    a = k * dt
    if branch == "euler":
        assert a < 1
        assert YA == pytest.approx(Y0 * (1 - a) ** n, rel=1e-13)
        assert YA + YB == pytest.approx(Y0, rel=1e-14)  # Euler conserves exactly
        assert out["n_asym"][0] == 0
    else:
        assert a >= 1
        assert YA == pytest.approx(Y0 / (1 + a) ** n, rel=1e-13)
        # B is fed from the OLD Y_A each step (explicit):
        # Y_B(n) = a Y0 sum_{j<n} (1+a)^-j
        q = 1 / (1 + a)
        assert YB == pytest.approx(a * Y0 * (1 - q**n) / (1 - q), rel=1e-13)
        assert out["n_asym"][0] == n  # species A every step, species B never (k_B = 0)


def test_p3_single_decay_continuum():
    """Y0 exp(-k t) at k dt = 1e-4, t = 1/k: first-order error ~ k dt / 2."""
    k = 1.0
    o = Oracle(decay_net(k))
    out = o.integrate_fixed(1.0, 1.0, [1.0, 0.0], 1e-4, 10_000)
    rel = abs(out["Y"][0, 0] / np.exp(-1.0) - 1)
    assert 4e-5 < rel < 6e-5


# ------------------------------------------------ pins found missing by mutation
@pytest.mark.parametrize("y_floor,Y0", [(1e-10, 2.5e-11), (1e-3, 2.5e-4)])
def test_y_floor_value_sets_the_step_sequence(y_floor, Y0):
    """O6 (S:Q7): the candidate of a species BELOW the floor is eps*Y_floor/|dY/dt|, not
    eps*Y/|dY/dt|.  Worked by hand for A -> B, k = 1, eps = 0.05, Y_A(0) = Y_floor/4, Y_B = 1
    (B's candidate eps*1/(k Y_A) is astronomically large; the growth cap 2*t_hydro never binds):
      step 1: dt = eps*Y_floor/(k Y_A) = 4 eps = 0.2     k dt = 0.2  -> Euler, Y_A *= 0.8
      step 2: dt = 0.2/0.8 = 0.25                         k dt = 0.25 -> Euler, Y_A *= 0.75
      step 3: dt_ctrl = 0.25/0.75 = 1/3, but t_hydro = 0.2 + 0.25 + 1/6 leaves 1/6:
              clamped, k dt = 1/6 -> Euler, Y_A *= 5/6
    so 3 steps, Y_A = Y0 * 0.8 * 0.75 * 5/6 = Y0/2, returned dt = 1/3 (unclamped).
    A floor 100x larger gives dt_1 = 20 > t_hydro (1 step); a floor 100x smaller, or none,
    puts Y_A above it and gives dt = eps/k = 0.05 (13 steps)."""
    o = Oracle(decay_net(1.0), OracleParams(eps_y=0.05, y_floor=y_floor))
    t_hydro = 0.2 + 0.25 + 1.0 / 6.0
    out = o.integrate(1.0, 1.0, [[Y0, 1.0]], t_hydro)
    assert out["n_steps"][0] == 3 and out["status"][0] == 0 and out["n_asym"][0] == 0
    assert out["Y"][0, 0] == pytest.approx(Y0 / 2, rel=1e-13)
    assert out["dt"][0] == pytest.approx(1.0 / 3.0, rel=1e-13)
    assert out["Y"][0, 1] == pytest.approx(1.0 + Y0 / 2, rel=1e-15)


def test_end_clamp_guard_decides_one_step_or_two():
    """O6 (S:Q9): the step is the last one when dt_ctrl >= rem*(1 - 1e-12).  A -> B, k = 1,
    Y_A = 1, Y_B = 100, eps = 0.05: dt_ctrl = eps*Y_A/(k Y_A) = 0.05 to an ulp.
      t_hydro = 0.05*(1 + 5e-13): dt_ctrl is below rem by 5e-13 relative -- inside the guard:
          ONE step of exactly t_hydro (without the guard: a second, 2.5e-14 s sliver step);
      t_hydro = 0.05*(1 + 5e-12): outside the guard: TWO steps.
    Either way the returned dt is the unclamped 0.05 and Y_A = 1 - t_hydro to rounding."""
    o = Oracle(decay_net(1.0), OracleParams(eps_y=0.05))
    for excess, want_steps in ((5e-13, 1), (5e-12, 2)):
        t_hydro = 0.05 * (1.0 + excess)
        out = o.integrate(1.0, 1.0, [[1.0, 100.0]], t_hydro)
        assert out["n_steps"][0] == want_steps, (excess, out["n_steps"][0])
        assert out["dt"][0] == pytest.approx(0.05, rel=1e-14)
        assert out["Y"][0, 0] == pytest.approx(1.0 - t_hydro, rel=1e-13)


@pytest.mark.parametrize("a,branch", [(0.5, "euler"), (1.0, "euler"), (1.5, "euler"),
                                       (2.0, "asym"), (3.0, "asym")])
def test_p2_closed_forms_at_kappa_two(a, branch):
    """The branch threshold is the parameter kappa, not the constant 1: at
    kappa = 2 a single decay with k dt = 1 or 1.5 still takes forward Euler --
    Y0 (1 - k dt)^n, i.e. exactly 0 after one step at k dt = 1 and a sign-alternating
    Y0 (-1/2)^n at 1.5 (the closed form holds for either sign: F- = k Y) -- and
    k dt = 2 exactly is the first asymptotic value, Y0/(1 + k dt)^n."""
    o = Oracle(decay_net(1.0), OracleParams(kappa=2.0))
    n, Y0 = 12, 0.75
    out = o.integrate_fixed(1.0, 1.0, [Y0, 0.0], a, n)
    YA = out["Y"][0, 0]
    if branch == "euler":
        want = Y0 * (1 - a) ** n
        assert YA == pytest.approx(want, rel=1e-13, abs=0.0)
        assert out["n_asym"][0] == 0
    else:
        assert YA == pytest.approx(Y0 / (1 + a) ** n, rel=1e-13)
        assert out["n_asym"][0] == n


def test_growth_cap_is_the_parameter():
    """O6 (S:Q7): dt <= g*dt_prev with g the parameter.  A -> B, k = 1, Y_A = 1, Y_B = 100,
    eps = 0.05 (candidate 0.05), g = 1.5, trial dt 0.01:
      dt = 0.015, 0.0225, 0.03375 (cap binds), then 1.5*0.03375 = 0.050625 > 0.05: the candidate;
      t_hydro = 0.07125 + 2*0.05 = 0.17125 is reached in exactly 5 steps,
      Y_A = 0.985 * 0.9775 * 0.96625 * 0.95^2.   (g = 2 would take 0.02, 0.04, 0.05, ...)"""
    o = Oracle(decay_net(1.0), OracleParams(eps_y=0.05, growth=1.5))
    out = o.integrate(1.0, 1.0, [[1.0, 100.0]], 0.17125, dt=[0.01])
    assert out["n_steps"][0] == 5
    assert out["Y"][0, 0] == pytest.approx(0.985 * 0.9775 * 0.96625 * 0.95**2, rel=1e-13)
    assert out["dt"][0] == pytest.approx(0.05, rel=1e-13)


# ------------------------------------------------- P4: two-species fixed point
@pytest.mark.parametrize("dt", [1e-3, 0.5, 10.0, 1e3])
def test_p4_two_species_equilibrium_ratio(dt):
    """A <-> B: Y_A/Y_B = k_r/k_f is a fixed point of both branches at any dt."""
    kf, kr = 3.0, 1.0
    o = Oracle(make_toy([1, 1], [((0,), (1,)), ((1,), (0,))], [kf, kr]))
    Y = np.array([[0.9, 0.1]])
    for _ in range(60):
        Y = o.integrate_fixed(1.0, 1.0, Y, dt, 1000)["Y"]
    assert Y[0, 0] / Y[0, 1] == pytest.approx(kr / kf, rel=1e-12)


def test_p4_total_drift_shrinks_with_eps():
    """With the controller on and t long enough to enter the asymptotic branch,
    |Y_A + Y_B - 1| is a bounded diagnostic, not an identity (Eq. (3) does not
    conserve): small, and smaller at the tighter eps_Y."""
    kf, kr = 3.0, 1.0
    net = make_toy([1, 1], [((0,), (1,)), ((1,), (0,))], [kf, kr])
    drift = []
    for eps in (0.05, 0.0125):
        o = Oracle(net, OracleParams(eps_y=eps))
        out = o.integrate(1.0, 1.0, [[0.9, 0.1]], 10.0)
        assert out["n_asym"][0] > 0
        drift.append(abs(out["Y"].sum() - 1.0))
    assert 1e-6 < drift[0] < 1e-2 and drift[1] < drift[0]


# ------------------------------------------------------- P5: A-conservation
def test_p5_nucleon_number_euler_regime(g16):
    """Config 1 is all-Euler: sum(A_i Y_i) stays 1 to rounding over 1e4 steps."""
    o = Oracle(g16)
    Y0 = np.zeros(16)
    Y0[0], Y0[1] = 0.5 / 4, 0.5 / 8
    out = o.integrate_fixed(3.0, 1e8, Y0, 1e-10, 10_000)
    assert out["n_asym"][0] == 0
    assert abs((out["Y"][0] * g16.A).sum() - 1.0) < 1e-12


def test_p5_every_family_conserves(hub150):
    """Tiny Euler steps from a state with every species populated: any wrong
    edge, sign or multiplicity in any reaction family breaks sum(A Y)."""
    o = Oracle(hub150)
    rng = np.random.default_rng(5)
    Y0 = rng.uniform(0.5, 1.5, 150)
    Y0 /= (Y0 * hub150.A).sum()
    out = o.integrate_fixed(4.0, 1e8, Y0, 1e-16, 50)
    assert out["n_asym"][0] == 0
    assert not np.allclose(out["Y"][0], Y0, rtol=1e-9)  # something did happen
    assert abs((out["Y"][0] * hub150.A).sum() - 1.0) < 1e-13


# ----------------------------------------------------------- P6: positivity
def test_p6_positivity(hub150):
    o = Oracle(hub150)
    rng = np.random.default_rng(6)
    z = 6
    T9 = rng.uniform(1, 10, z)
    rho = 10 ** rng.uniform(7, 9.5, z)
    Y0 = np.zeros((z, 150))
    Y0[:, 3], Y0[:, 15] = 0.5 / 12, 0.5 / 16
    Y = Y0
    for dt in (1e-12, 1e-9, 1e-7, 1e-6):  # from all-Euler to mixed (1e-3 overflows: Eq. (3) does not conserve)
        Y = o.integrate_fixed(T9, rho, Y, dt, 200)["Y"]
        assert (Y >= 0).all() and np.isfinite(Y).all()
    out = o.integrate(T9, rho, Y0, 1e-7)
    assert (out["Y"] >= 0).all() and (out["status"] == 0).all()


# ---------------------------------------------------------- P7: brute force
def ode_rhs(net: Network, R, Y):
    """dY/dt of Eq. (1) straight from the reaction list (independent of the
    oracle's edge list): each reaction moves rate = R prod(Y) from its
    reactants to its products, one unit per occurrence."""
    d = np.zeros_like(Y)
    for r in range(net.n_reactions):
        re = net.react[r, : net.n_react[r]]
        pr = net.prod[r, : net.n_prod[r]]
        rate = R[r] * np.prod(Y[re])
        for s in re:
            d[s] -= rate
        for s in pr:
            d[s] += rate
    return d


def rk4(net, R, Y, t_end, n):
    h = t_end / n
    for _ in range(n):
        k1 = ode_rhs(net, R, Y)
        k2 = ode_rhs(net, R, Y + 0.5 * h * k1)
        k3 = ode_rhs(net, R, Y + 0.5 * h * k2)
        k4 = ode_rhs(net, R, Y + h * k3)
        Y = Y + h / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
    return Y


def tiny_net():
    # species: a(A=1) b(A=1) c(A=2) d(A=3) e(A=4) g(A=4)
    A = [1, 1, 2, 3, 4, 4]
    reactions = [
        ((0,), (1,)),            # a -> b
        ((1,), (0,)),            # b -> a
        ((0, 1), (2,)),          # a + b -> c
        ((2,), (0, 1)),          # c -> a + b
        ((0, 0), (2,)),          # a + a -> c      (identical pair)
        ((0, 1, 2), (4,)),       # a + b + c -> e  (3-body)
        ((0, 0, 0), (3,)),       # 3a -> d         (3-body identical)
        ((3, 0), (5,)),          # d + a -> g
        ((5,), (4,)),            # g -> e
        ((4,), (2, 2)),          # e -> c + c      (identical products)
    ]
    rates = [2.0, 1.0, 30.0, 0.5, 8.0, 200.0, 90.0, 40.0, 3.0, 0.7]
    return make_toy(A, reactions, rates)


def test_p7_brute_force_tiny_network():
    net = tiny_net()
    Y0 = np.array([0.5, 0.3, 0.1, 0.0, 0.0, 0.0])
    Y0 /= (Y0 * net.A).sum()
    t_end = 0.8
    o = Oracle(net)
    R = o.rates(1.0, 1.0)
    ref = rk4(net, R, Y0.copy(), t_end, 8_000)
    assert abs((ref * net.A).sum() - 1.0) < 1e-12
    errs = []
    for eps in (0.04, 0.01, 0.0025):
        out = Oracle(net, OracleParams(eps_y=eps)).integrate(1.0, 1.0, Y0, t_end)
        X, Xr = out["Y"][0] * net.A, ref * net.A
        m = Xr > 1e-6
        errs.append(np.abs(X[m] / Xr[m] - 1).max())
    assert errs[0] < 4e-2                       # O(eps_Y)
    assert errs[1] < 0.45 * errs[0] and errs[2] < 0.45 * errs[1]  # ~linear in eps_Y


def test_p7_fixed_small_dt_matches_forward_euler_exactly():
    """In the all-Euler regime the oracle IS forward Euler on Eq. (1)."""
    net = tiny_net()
    Y0 = np.array([0.5, 0.3, 0.1, 0.01, 0.02, 0.03])
    o = Oracle(net)
    R = o.rates(1.0, 1.0)
    dt, n = 1e-4, 300
    Y = Y0.copy()
    for _ in range(n):
        Y = Y + dt * ode_rhs(net, R, Y)
    out = o.integrate_fixed(1.0, 1.0, Y0, dt, n)
    assert out["n_asym"][0] == 0
    np.testing.assert_allclose(out["Y"][0], Y, rtol=1e-12)


# ------------------------------------------------------ P8: linear networks
def test_p8_linear_network_dense_matrix_power():
    """All 1-body reactions, Euler regime: Y_n = (I + dt K)^n Y0."""
    rng = np.random.default_rng(8)
    n_light, n_heavy = 6, 3  # A = 1 species and A = 2 species
    N = n_light + n_heavy
    A = [1] * n_light + [2] * n_heavy
    reactions, rates = [], []
    for _ in range(24):
        i, j = rng.choice(n_light, 2, replace=False)
        reactions.append(((int(i),), (int(j),)))
        rates.append(float(rng.uniform(0.1, 5.0)))
    for h in range(n_heavy):  # heavy -> j + j (nu = 2 on the product side) and -> j + j'
        j = int(rng.integers(0, n_light))
        reactions.append(((n_light + h,), (j, j)))
        rates.append(float(rng.uniform(0.1, 5.0)))
        j2 = (j + 1 + int(rng.integers(0, n_light - 1))) % n_light
        reactions.append(((n_light + h,), (j, j2)))
        rates.append(float(rng.uniform(0.1, 5.0)))
    net = make_toy(A, reactions, rates)
    K = np.zeros((N, N))
    for (re, pr), k in zip(reactions, rates):
        K[re[0], re[0]] -= k
        for s in pr:
            K[s, re[0]] += k
    dt, n = 5e-3, 400
    Y0 = rng.uniform(0.1, 1.0, N)
    expect = np.linalg.matrix_power(np.eye(N) + dt * K, n) @ Y0
    out = Oracle(net).integrate_fixed(1.0, 1.0, Y0, dt, n)
    assert out["n_asym"][0] == 0
    np.testing.assert_allclose(out["Y"][0], expect, rtol=1e-12)


# ------------------------------------------------- P9: permutation invariance
def test_p9_permutation_invariance(hub150):
    net2, sigma = hub150.permuted(seed=99)
    o1, o2 = Oracle(hub150), Oracle(net2)
    Y0 = np.zeros(150)
    Y0[3], Y0[15] = 0.5 / 12, 0.5 / 16
    Y0p = np.zeros(150)
    Y0p[sigma] = Y0
    a = o1.integrate_fixed(6.0, 5e8, Y0, 1e-9, 500)["Y"][0]
    b = o2.integrate_fixed(6.0, 5e8, Y0p, 1e-9, 500)["Y"][0][sigma]
    X = a * hub150.A
    m = X > 1e-12
    assert m.sum() > 10
    assert np.abs(b[m] / a[m] - 1).max() < 1e-10
    ra = o1.integrate(6.0, 5e8, Y0, 1e-7)
    rb = o2.integrate(6.0, 5e8, Y0p, 1e-7)
    a, b = ra["Y"][0], rb["Y"][0][sigma]
    m = a * hub150.A > 1e-12
    assert np.abs(b[m] / a[m] - 1).max() < 1e-7
    assert abs(int(ra["n_steps"][0]) - int(rb["n_steps"][0])) <= max(1, ra["n_steps"][0] // 100)


# ------------------------------------------------ P10: 3-body multiplicity
def test_p10_three_alpha_multiplicity():
    """3a -> C with raw rate Rraw: f = Rraw Ya^3 / 6, F-_a = 3 f, F+_C = f."""
    Rraw, Ya = 7.0, 0.2
    net = toy_with_coefs([4, 12], [((0, 0, 0), (1,)), ((1,), (0, 0, 0))],
                         [(np.log(Rraw), 0, 0, 0, 0, 0, 0), (np.log(0.5), 0, 0, 0, 0, 0, 0)])
    o = Oracle(net)
    R = o.rates(1.0, 1.0)
    assert R[0] == pytest.approx(Rraw / 6, rel=1e-15)
    f, Fp, Fm = o.rhs(R, [Ya, 0.0])
    assert f[0] == pytest.approx(Rraw * Ya**3 / 6, rel=1e-15)
    assert Fm[0] == pytest.approx(3 * Rraw * Ya**3 / 6, rel=1e-15) and Fp[1] == f[0]
    # reverse: C -> 3a feeds alpha three times
    f, Fp, Fm = o.rhs(R, [0.0, 0.1])
    assert Fp[0] == pytest.approx(3 * 0.5 * 0.1, rel=1e-15) and Fm[1] == pytest.approx(0.05, rel=1e-15)
    # first Euler step
    dt = 1e-3
    Y = o.integrate_fixed(1.0, 1.0, [Ya, 0.0], dt, 1)["Y"][0]
    assert Y[0] == pytest.approx(Ya - dt * 3 * Rraw * Ya**3 / 6, rel=1e-15)
    assert Y[1] == pytest.approx(dt * Rraw * Ya**3 / 6, rel=1e-15)


# ------------------------------------------- controller and call contract
def test_dt_controller_contract():
    """O3/O6/O8-O9 (S:Q7, Q9-Q11) on a single decay where every step is known.

    A -> B with k = 1, Y_A = 1, Y_B = 100, eps = 0.05: c_A = eps Y_A/(k Y_A) =
    0.05 and c_B = eps Y_B/(k Y_A) >= 5, so dt_ctrl = 0.05 every step once the
    growth cap allows; t_hydro = 1 takes exactly 20 steps (the last one clamped
    through the 1e-12 guard) and the returned dt is the unclamped 0.05."""
    o = Oracle(decay_net(1.0), OracleParams(eps_y=0.05, growth=2.0))
    Y0 = [1.0, 100.0]
    out = o.integrate(1.0, 1.0, Y0, 1.0)
    assert out["n_steps"][0] == 20 and out["status"][0] == 0
    assert out["dt"][0] == pytest.approx(0.05, rel=1e-12)
    assert out["Y"][0, 0] == pytest.approx(0.95**20, rel=1e-12)
    # trial dt honoured with the growth cap: dt_in = 0.01 -> 0.02, 0.04, then 0.05 ...
    out = o.integrate(1.0, 1.0, Y0, 1.0, dt=[0.01])
    # t after 2 steps = 0.06; remaining 0.94 / 0.05 = 18.8 -> 19 more steps
    assert out["n_steps"][0] == 21
    assert out["Y"][0, 0] == pytest.approx(0.98 * 0.96 * 0.95**18 * (1 - 0.04), rel=1e-12)
    # a short clamped final step does not poison the returned dt (S:Q10)
    assert out["dt"][0] == pytest.approx(0.05, rel=1e-12)
    # max_steps -> status bit 1
    o2 = Oracle(decay_net(1.0), OracleParams(eps_y=0.05, max_steps=5))
    out = o2.integrate(1.0, 1.0, Y0, 1.0)
    assert out["n_steps"][0] == 5 and out["status"][0] == 1
    # t_hydro <= 0: nothing happens
    out = o.integrate(1.0, 1.0, Y0, 0.0, dt=[0.3])
    assert out["n_steps"][0] == 0 and out["dt"][0] == 0.3 and out["Y"][0, 0] == 1.0


def test_nonfinite_status_bit_worked_by_hand():
    """P:L110 / SURVEY 8(b): status bit 2 = a non-finite abundance was produced (O9's check).

    Overflow, every step known.  A -> B with k = 1, Y_A = Y_B = 1.5e308, eps_Y = 0.25,
    t_hydro = 10, no trial dt.  Step 1: F_A = -1.5e308, F_B = +1.5e308, so c_A = c_B =
    0.25 * 1.5e308 / 1.5e308 = 0.25 < growth * t_hydro: dt = 0.25, k_A dt = 0.25 < kappa,
    Euler on both: Y_A = 1.5e308 * 0.75 and Y_B = 1.5e308 * 1.25 = 1.875e308 > DBL_MAX = +inf.
    From then on Y_B = inf has F- = 0 (k = 0, Euler, stays inf) and an infinite candidate;
    Y_A keeps c_A = 0.25 and loses a quarter per step.  0.25 is a binary fraction, so t hits
    10 exactly on step 40 (the last one through the 1e-12 guard): n_steps = 40, dt = 0.25,
    Y_A = 1.5e308 * 0.75^40, status = 2 and NOT 1 | 2."""
    o = Oracle(decay_net(1.0), OracleParams(eps_y=0.25))
    out = o.integrate(1.0, 1.0, [1.5e308, 1.5e308], 10.0)
    assert out["status"][0] == 2 and out["n_steps"][0] == 40 and out["dt"][0] == 0.25
    assert np.isposinf(out["Y"][0, 1])
    assert out["Y"][0, 0] == pytest.approx(1.5e308 * 0.75**40, rel=1e-13)
    # a start whose total Y_A + Y_B = 1.6e308 stays below DBL_MAX never overflows: bit 2 stays clear
    out = o.integrate(1.0, 1.0, [0.8e308, 0.8e308], 10.0)
    assert out["status"][0] == 0 and np.isfinite(out["Y"]).all() and out["n_steps"][0] == 40
    # fixed-dt mode overflows the same way: one Euler step of dt = 0.5 from 1.5e308 overflows B
    out = o.integrate_fixed(1.0, 1.0, [1.5e308, 1.5e308], 0.5, 1)
    assert np.isposinf(out["Y"][0, 1]) and out["Y"][0, 0] == 0.75e308
    # NaN from the inputs: T9 < 0 makes ln T9 (a6 term) NaN whenever a6 != 0, every rate of such a
    # reaction NaN, every flux NaN; a NaN candidate never wins the dt minimum ('<' is false), so the
    # zone takes ONE step of the whole t_hydro, returns dt = growth * t_hydro, and flags bit 2;
    # zones beside it in the batch are untouched
    c = build_config(3, zones=3)
    good = Oracle(c["network"]).integrate(c["T9"], c["rho"], c["Y0"], c["t_hydro"])
    T9 = c["T9"].copy()
    T9[1] = -1.0
    bad = Oracle(c["network"]).integrate(T9, c["rho"], c["Y0"], c["t_hydro"])
    assert bad["status"].tolist() == [0, 2, 0] and bad["n_steps"][1] == 1
    assert bad["dt"][1] == 2.0 * c["t_hydro"] and np.isnan(bad["Y"][1]).any()
    for z in (0, 2):
        assert np.array_equal(bad["Y"][z], good["Y"][z]) and bad["n_steps"][z] == good["n_steps"][z]


def test_zero_abundance_species_use_euler():
    """S:Q8: Y_i = 0 => k_i = 0 => Euler: Y_i' = dt F+_i, however large dt is."""
    o = Oracle(make_toy([1, 1, 1], [((0,), (1,)), ((1,), (2,))], [2.0, 1e6]))
    Y = o.integrate_fixed(1.0, 1.0, [1.0, 0.0, 0.0], 10.0, 1)["Y"][0]
    assert Y[1] == pytest.approx(10.0 * 2.0 * 1.0, rel=1e-15)  # fed from old Y_0
    assert Y[0] == pytest.approx(1.0 / 21.0, rel=1e-15)        # k dt = 20 -> Eq. (3)
    assert Y[2] == 0.0                                           # old Y_1 was 0


def test_fp32_variant_tracks_fp64(hub150):
    """P12 (PARITY UNPINNED: the paper gives no bound) - sanity only."""
    o = Oracle(hub150)
    Y0 = np.zeros((1, 150))
    Y0[0, 3], Y0[0, 15] = 0.5 / 12, 0.5 / 16
    a = o.integrate(7.0, 1e8, Y0, 1e-7, precision=64)
    b = o.integrate(7.0, 1e8, Y0, 1e-7, precision=32)
    X = a["Y"][0] * hub150.A
    m = X > 1e-12
    assert np.abs(b["Y"][0][m] / a["Y"][0][m] - 1).max() < 1e-2
    assert abs(int(a["n_steps"][0]) - int(b["n_steps"][0])) <= max(2, a["n_steps"][0] // 50)


from gen import build_config  # noqa: E402


# ---------------------------------------------------------------- energy release (Q19)
def test_energy_single_decay_closed_form():
    """A -> B with rate k, fixed dt in the Euler regime: Y_A(n) = Y0 (1 - k dt)^n exactly, so
    E = (B_B - B_A) * Y0 * (1 - (1 - k dt)^n)."""
    k, dt, n, y0 = 3.0, 0.01, 40, 0.25
    net = make_toy([1, 1], [((0,), (1,))], [k])
    o = Oracle(net)
    Y0 = np.array([[y0, 0.0]])
    out = o.integrate_fixed(1.0, 1.0, Y0, dt, n)
    B = np.array([1.5, 9.25])
    want = (B[1] - B[0]) * y0 * (1.0 - (1.0 - k * dt) ** n)
    assert Oracle.energy(B, Y0, out["Y"])[0] == pytest.approx(want, rel=1e-13)


def test_energy_is_sum_of_q_values_times_integrated_fluxes(g16):
    """In the all-Euler regime dY_i = dt * sum_r nu_ir f_r, so the energy release equals
    sum_r Q_r * (integrated flux of r) with Q_r = B(products) - B(reactants): an identity
    through the reaction list, independent of the species sums the definition uses."""
    c = build_config(1)
    o = Oracle(g16)
    rng = np.random.default_rng(5)
    B = g16.A * 8.0 + rng.normal(0, 1.0, g16.n_species)
    Q = np.array([sum(B[s] for s in g16.prod[r, :g16.n_prod[r]]) - sum(B[s] for s in g16.react[r, :g16.n_react[r]])
                  for r in range(g16.n_reactions)])
    R = o.rates(c["T9"][0], c["rho"][0])
    Y = c["Y0"].copy()
    dt, n, acc = 1e-10, 400, 0.0
    for _ in range(n):
        f, _, _ = o.rhs(R, Y[0])
        acc += dt * float(Q @ f)
        step = o.integrate_fixed(c["T9"], c["rho"], Y, dt, 1)
        assert step["n_asym"][0] == 0
        Y = step["Y"]
    E = Oracle.energy(B, c["Y0"], Y)[0]
    assert E != 0.0 and E == pytest.approx(acc, rel=1e-9)


def test_energy_vanishes_when_binding_is_proportional_to_mass_number(g16):
    """B_i = c A_i makes E = c * delta(sum A_i Y_i), which the Euler regime conserves (P5)."""
    c = build_config(1)
    out = Oracle(g16).integrate_fixed(c["T9"], c["rho"], c["Y0"], 1e-10, 2000)
    assert out["n_asym"][0] == 0
    E = Oracle.energy(7.5 * g16.A, c["Y0"], out["Y"])[0]
    assert abs(E) < 1e-11


# ------------------------------------------------ the long-double arbiter (precision = 80)
def test_arbiter_rates_vs_numpy_longdouble(hub150):
    """O2 of the arbiter against numpy's own long-double libm route, term by term."""
    o = Oracle(hub150)
    L = np.longdouble
    third = L(1) / L(3)
    for T9, rho in ((1.0, 1e7), (3.3, 2.2e8), (10.0, 3.1e9)):
        R = o.rates_ld(T9, rho)
        T = L(T9)
        a = hub150.coef.astype(L)
        lnp = np.array([
            -sum(np.log(L(factorial(list(re[:n]).count(s)))) for s in set(re[:n]))
            for re, n in zip(hub150.react, hub150.n_react)
        ], dtype=L)
        ln = (a[:, 0] + a[:, 1] / T + a[:, 2] * T ** (-third) + a[:, 3] * T ** third + a[:, 4] * T
              + a[:, 5] * T ** (L(5) * third) + a[:, 6] * np.log(T)
              + lnp + (hub150.n_react.astype(L) - 1) * np.log(L(rho)))
        rel = np.abs(R / np.exp(ln) - 1).astype(np.float64)
        assert rel.max() < 2e-16  # exponent arguments ~1e2 amplify an extended-precision ulp (5e-20)
        # and the fp64 rates are the arbiter's rates to fp64 rounding
        assert np.abs(o.rates(T9, rho) / R.astype(np.float64) - 1).max() < 2e-13


@pytest.mark.parametrize("k,dt,branch", [(1.0, 0.25, "euler"), (1.0, 1.0, "asym"), (1.0, 4.0, "asym")])
def test_arbiter_single_decay_closed_forms(k, dt, branch):
    """P2 on the arbiter: same closed forms, now met to the last bit or two of a double."""
    o = Oracle(decay_net(k))
    n, Y0 = 40, 0.75
    out = o.integrate_fixed(1.0, 1.0, [Y0, 0.0], dt, n, precision=80)
    a = np.longdouble(k) * np.longdouble(dt)
    want = np.longdouble(Y0) * ((1 - a) ** n if branch == "euler" else (1 + a) ** (-n))
    assert out["Y"][0, 0] == pytest.approx(float(want), rel=4e-16)
    assert out["n_asym"][0] == (0 if branch == "euler" else n)


def test_arbiter_controller_contract_and_agreement_with_fp64(g16, hub150):
    """The arbiter runs the same controller (20 steps / dt 0.05 on the worked single decay),
    and on well-conditioned runs it agrees with the fp64 oracle to fp64 rounding: fixed dt on
    config 1 (<= 1e-12), adaptive on a short hub150 step (same step count, <= 1e-9)."""
    o = Oracle(decay_net(1.0), OracleParams(eps_y=0.05, growth=2.0))
    out = o.integrate(1.0, 1.0, [[1.0, 100.0]], 1.0, precision=80)
    assert out["n_steps"][0] == 20 and out["dt"][0] == pytest.approx(0.05, rel=1e-15)
    assert out["Y"][0, 0] == pytest.approx(0.95**20, rel=1e-15)
    c = build_config(1)
    og = Oracle(g16)
    a = og.integrate_fixed(c["T9"], c["rho"], c["Y0"], 1e-5, 1000)
    b = og.integrate_fixed(c["T9"], c["rho"], c["Y0"], 1e-5, 1000, precision=80)
    m = a["Y"] * g16.A > 1e-12
    assert (a["n_asym"] == b["n_asym"]).all() and np.abs(a["Y"][m] / b["Y"][m] - 1).max() < 1e-12
    oh = Oracle(hub150)
    Y0 = np.zeros((1, 150))
    Y0[0, 3], Y0[0, 15] = 0.5 / 12, 0.5 / 16
    a = oh.integrate(4.0, 1e8, Y0, 1e-8)
    b = oh.integrate(4.0, 1e8, Y0, 1e-8, precision=80)
    m = a["Y"] * hub150.A > 1e-12
    assert a["n_steps"][0] == b["n_steps"][0] and np.abs(a["Y"][m] / b["Y"][m] - 1).max() < 1e-9


# ------------------------------------------------ QSS variant (reading Q20)
QSS = dict(method=1)


@pytest.mark.parametrize("a,num,den", [(1.0, 252, 685), (2.0, 21, 155)])
def test_qss_single_decay_hand_worked_factor(a, num, den):
    """A -> B, F+_A = 0: per step Y_A *= (1 + (alpha - 1) a)/(1 + alpha a), a = k dt.
    By hand: alpha(1) = (1+11+60+180)/(1+12+60+360) = 252/433 -> factor (252/433)/(685/433)
    = 252/685; alpha(2) = (8+44+120+180)/(8+48+120+360) = 352/536 = 44/67 -> factor
    (1 - 46/67)/(1 + 88/67) = 21/155.  B receives what A loses (F+_B = F-_A, k_B = 0)."""
    for precision in (64, 80):
        o = Oracle(decay_net(1.0), OracleParams(**QSS))
        n, Y0 = 10, 0.75
        out = o.integrate_fixed(1.0, 1.0, [Y0, 0.0], a, n, precision=precision)
        assert out["Y"][0, 0] == pytest.approx(Y0 * (num / den) ** n, rel=1e-13)
        # B: k_B = 0 -> plain Euler on F+_B = k Y_A(old): Y_B = a Y0 sum_j f^j
        f = num / den
        assert out["Y"][0, 1] == pytest.approx(a * Y0 * (1 - f**n) / (1 - f), rel=1e-13)


@pytest.mark.parametrize("a,tol", [(1e-3, 1e-12), (0.1, 2e-12), (0.5, 1e-7), (1.0, 1.1e-5), (2.0, 1.2e-3)])
def test_qss_tracks_the_exact_exponential(a, tol):
    """With the exact weight the quasi-steady-state step reproduces Y0 e^{-k dt} for constant k
    and F+ = 0; the Pade alpha is within 4e-6 of it at k dt = 1 and 1.5e-4 at k dt = 2
    (absolute, per step).  Forward Euler at k dt = 0.5 is off by 0.1."""
    o = Oracle(decay_net(1.0), OracleParams(**QSS))
    Y = o.integrate_fixed(1.0, 1.0, [1.0, 0.0], a, 1)["Y"][0, 0]
    assert abs(Y - np.exp(-a)) < tol * max(1.0, 1.0) and Y != 1 - a


def test_qss_euler_limit_and_stiff_limit():
    """alpha -> 1/2 as k dt -> 0: the step is y (1 - a/2)/(1 + a/2) = y (1 - a + a^2/2 - ...),
    forward Euler to first order: after n = 100 steps at a = 1e-4 the ratio to the Euler closed
    form (1 - a)^n is 1 + n a^2/2 = 1 + 5e-7.  alpha -> 1 as k dt -> infinity: with a source,
    y' -> y + (F+ - k y)/k = F+/k, the steady state, as Eq. (3) does."""
    o = Oracle(decay_net(1.0), OracleParams(**QSS))
    a, n = 1e-4, 100
    Y = o.integrate_fixed(1.0, 1.0, [1.0, 0.0], a, n)["Y"][0, 0]
    assert Y / (1 - a) ** n - 1 == pytest.approx(n * a * a / 2, rel=2e-2)
    kf, kr = 3.0e9, 1.0e9
    o2 = Oracle(make_toy([1, 1], [((0,), (1,)), ((1,), (0,))], [kf, kr]), OracleParams(**QSS))
    Y = o2.integrate_fixed(1.0, 1.0, [0.9, 0.1], 1.0, 1)["Y"][0]
    assert Y[0] == pytest.approx(kr * 0.1 / kf, rel=1e-7)  # F+_A / k_A from the old Y_B


@pytest.mark.parametrize("dt", [1e-3, 0.5, 10.0, 1e3])
def test_qss_two_species_equilibrium_ratio(dt):
    """F+ = k y at Y_A/Y_B = k_r/k_f whatever alpha is: an exact fixed point at any dt (started
    there, the state does not move).  The error mode contracts for moderate dt; at k dt ~ 1e3
    the Jacobi predictor hands each species the other's steady state and the mode decays only
    like 1 - O(1/(k dt)^2) per step, so there only boundedness and positivity are asserted."""
    kf, kr = 3.0, 1.0
    o = Oracle(make_toy([1, 1], [((0,), (1,)), ((1,), (0,))], [kf, kr]), OracleParams(**QSS))
    Y = o.integrate_fixed(1.0, 1.0, [[0.25, 0.75]], dt, 1000)["Y"]
    assert Y[0, 0] == pytest.approx(0.25, rel=1e-13) and Y[0, 1] == pytest.approx(0.75, rel=1e-13)
    Y = np.array([[0.9, 0.1]])
    for _ in range(60):
        Y = o.integrate_fixed(1.0, 1.0, Y, dt, 1000)["Y"]
    if dt <= 10.0:
        assert Y[0, 0] / Y[0, 1] == pytest.approx(kr / kf, rel=1e-12)
    else:
        assert (Y > 0).all() and Y.sum() < 10.0


def test_qss_brute_force_tiny_network_and_positivity(hub150):
    """The variant as an approximation of Eq. (1): RK4 on the tiny network, error O(eps_Y) and
    shrinking with it; on hub150 it stays non-negative and finite, and it is a different
    integrator from the asymptotic one (results differ) behind the same controller."""
    net = tiny_net()
    Y0 = np.array([0.5, 0.3, 0.1, 0.0, 0.0, 0.0])
    Y0 /= (Y0 * net.A).sum()
    t_end = 0.8
    R = Oracle(net).rates(1.0, 1.0)
    ref = rk4(net, R, Y0.copy(), t_end, 8_000)
    errs = []
    for eps in (0.04, 0.01, 0.0025):
        out = Oracle(net, OracleParams(eps_y=eps, **QSS)).integrate(1.0, 1.0, Y0, t_end)
        X, Xr = out["Y"][0] * net.A, ref * net.A
        m = Xr > 1e-6
        errs.append(np.abs(X[m] / Xr[m] - 1).max())
    assert errs[0] < 4e-2 and errs[1] < 0.45 * errs[0] and errs[2] < 0.45 * errs[1]
    rng = np.random.default_rng(6)
    z = 6
    T9, rho = rng.uniform(1, 10, z), 10 ** rng.uniform(7, 9.5, z)
    Y0 = np.zeros((z, 150))
    Y0[:, 3], Y0[:, 15] = 0.5 / 12, 0.5 / 16
    q = Oracle(hub150, OracleParams(**QSS)).integrate(T9, rho, Y0, 1e-7)
    a = Oracle(hub150).integrate(T9, rho, Y0, 1e-7)
    assert (q["Y"] >= 0).all() and np.isfinite(q["Y"]).all() and (q["status"] == 0).all()
    assert q["n_asym"].sum() > 0 and not np.allclose(q["Y"], a["Y"], rtol=1e-6, atol=1e-30)
