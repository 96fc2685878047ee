"""Seeded synthetic inputs (networks, zone profiles, compositions).

Test infrastructure shared by the CPU oracle and the CUDA path: it emits plain
numpy arrays and holds none of the integrator's arithmetic.
"""
from .network import Network, make_g16, make_hub_network, make_toy
from .profiles import (
    binding_energies,
    co_start,
    config1_state,
    perturbed_co_start,
    zone_profile,
)
from .configs import CONFIGS, build_config

__all__ = [
    "Network",
    "make_g16",
    "make_hub_network",
    "make_toy",
    "binding_energies",
    "co_start",
    "config1_state",
    "perturbed_co_start",
    "zone_profile",
    "CONFIGS",
    "build_config",
]
