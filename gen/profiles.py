"""Seeded zone profiles (T9, rho) and initial compositions."""
from __future__ import annotations

import numpy as np

from .network import Network


def zone_profile(zones: int, seed: int, log_rho=(7.0, 9.5), T9=(1.0, 10.0)):
    """Synthetic detonation profile: T9 ~ U[T9], log10(rho) ~ U[log_rho].

    Stands in for the hydro zones of a Type Ia simulation (PAPER.md L102 gives
    T = 7e9 K, rho = 1e8 g/cm^3 as the representative strongly-burning zone).
    """
    rng = np.random.default_rng(seed)
    t9 = rng.uniform(T9[0], T9[1], size=zones)
    rho = 10.0 ** rng.uniform(log_rho[0], log_rho[1], size=zones)
    return t9.astype(np.float64), rho.astype(np.float64)


def config1_state(net: Network) -> np.ndarray:
    """Config 1: mass fractions 0.5 / 0.5 in species 0 and 1; returns Y [1, N]."""
    Y = np.zeros((1, net.n_species))
    Y[0, 0] = 0.5 / net.A[0]
    Y[0, 1] = 0.5 / net.A[1]
    return Y


def co_start(net: Network, zones: int) -> np.ndarray:
    """C/O-like start: X = 0.5 in the first A=12 and the first A=16 species."""
    Y = np.zeros((zones, net.n_species))
    c, o = net.meta["first_A12"], net.meta["first_A16"]
    Y[:, c] = 0.5 / net.A[c]
    Y[:, o] = 0.5 / net.A[o]
    return Y


def binding_energies(net: Network, seed: int = 7) -> np.ndarray:
    """Synthetic per-species binding energies B_i (MeV per nucleus) for the energy-release
    output: a smooth liquid-drop-like curve in A with made-up coefficients plus seeded
    isobar-to-isobar noise.  Not nuclear data: it only gives the energy test inputs with
    the right size and sign structure (B/A rising to a plateau near A ~ 56)."""
    rng = np.random.default_rng(seed)
    A = net.A.astype(np.float64)
    per_nucleon = 8.9 - 9.5 / np.cbrt(np.maximum(A, 1.0)) - 0.004 * np.abs(A - 56.0)
    B = A * np.maximum(per_nucleon, 0.0) + rng.normal(0.0, 0.3, A.shape)
    B[A <= 1] = 0.0  # free nucleons
    return B


def perturbed_co_start(net: Network, zones: int, seed: int, sigma: float = 0.1) -> np.ndarray:
    """Config 4: each non-zero Y_i times exp(sigma*N(0,1)), then / sum(A_i Y_i)."""
    rng = np.random.default_rng(seed)
    Y = co_start(net, zones)
    noise = np.exp(sigma * rng.standard_normal(Y.shape))
    Y = np.where(Y > 0, Y * noise, 0.0)
    Y /= (Y * net.A[None, :]).sum(axis=1, keepdims=True)
    return Y
