"""BASELINE.json configs 1-5 as concrete seeded inputs."""
from __future__ import annotations

from functools import lru_cache

from .network import Network, make_g16, make_hub_network
from .profiles import co_start, config1_state, perturbed_co_start, zone_profile

import numpy as np

CONFIGS = {
    1: dict(net="g16", zones=1, mode="fixed", dt_fixed=1e-10, n_steps=10_000),
    2: dict(net="hub150", zones=1, mode="adaptive", t_hydro=1e-2, calls=1),
    3: dict(net="hub150", zones=128, mode="adaptive", t_hydro=1e-6, calls=10, profile_seed=3),
    4: dict(net="hub150", zones=16384, mode="adaptive", t_hydro=1e-6, calls=1, profile_seed=4),
    5: dict(net="hub365", zones=4096, mode="adaptive", t_hydro=1e-6, calls=1, profile_seed=5),
}


@lru_cache(maxsize=None)
def network(name: str) -> Network:
    if name == "g16":
        return make_g16(16)
    if name == "hub150":
        return make_hub_network(150, 1604, seed=1409)
    if name == "hub150hh":  # hub150 plus 16 heavy + heavy fusions and their inverses
        return make_hub_network(150, 1604, seed=1409, heavy_pairs=16)
    if name == "hub365":
        return make_hub_network(365, 4400, seed=365)
    raise KeyError(name)


def build_config(idx: int, zones: int | None = None) -> dict:
    """Inputs of config ``idx``; ``zones`` overrides the zone count (prefix of
    the same seeded stream is NOT guaranteed — the profile is redrawn)."""
    c = dict(CONFIGS[idx])
    net = network(c["net"])
    z = c["zones"] if zones is None else zones
    c["zones"] = z
    c["network"] = net
    if idx == 1:
        c["T9"] = np.full(z, 3.0)
        c["rho"] = np.full(z, 1e8)
        c["Y0"] = np.repeat(config1_state(net), z, axis=0)
    elif idx == 2:
        c["T9"] = np.full(z, 5.0)
        c["rho"] = np.full(z, 1e9)
        c["Y0"] = co_start(net, z)
    elif idx == 3:
        c["T9"], c["rho"] = zone_profile(z, c["profile_seed"])
        c["Y0"] = co_start(net, z)
    elif idx == 4:
        c["T9"], c["rho"] = zone_profile(z, c["profile_seed"])
        c["Y0"] = perturbed_co_start(net, z, seed=1000 + c["profile_seed"])
    elif idx == 5:
        c["T9"], c["rho"] = zone_profile(z, c["profile_seed"], log_rho=(7.0, 9.0))
        c["Y0"] = co_start(net, z)
    else:
        raise KeyError(idx)
    return c
