"""N > 1 host logic on CPU: two gloo ranks shard one seeded batch (SURVEY 8(e):
contiguous zone ranges, replicated tables, no data-path collective), each runs
its shard, and the pieces reassemble to exactly the single-process result.  The
per-zone work here is done by the oracle (no GPU in this test); what is under
test is the sharding and the max/sum job reduction bench.py uses."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from paper_1409_5826_b200.shard import reduce_job, zone_shard, zone_shard_balanced  # noqa: E402


def test_zone_shard_partitions_exactly():
    for total in (0, 1, 7, 128, 16384, 16385):
        for world in (1, 2, 3, 8):
            cuts = [zone_shard(total, r, world) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == total
            assert all(a[1] == b[0] for a, b in zip(cuts, cuts[1:]))
            sizes = [hi - lo for lo, hi in cuts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        zone_shard(10, 2, 2)


def test_zone_shard_balanced_partitions_and_deals_by_temperature():
    rng = np.random.default_rng(8)
    for total in (0, 1, 7, 128, 1001):
        T9 = rng.uniform(1, 10, total)
        if total > 3:
            T9[3] = np.nan  # a NaN zone is ranked last, never lost
        for world in (1, 2, 3, 8):
            parts = [zone_shard_balanced(T9, r, world) for r in range(world)]
            assert np.array_equal(np.sort(np.concatenate(parts)), np.arange(total))
            sizes = [len(p) for p in parts]
            assert max(sizes) - min(sizes) <= 1
            assert all((np.diff(p) > 0).all() for p in parts)
    # the deal itself, worked by hand: ranking hottest first = zones 4 1 3 0 2 5, snake over 2
    # ranks = 0 1 1 0 0 1  ->  rank 0: {4, 0, 2}, rank 1: {1, 3, 5}
    T9 = np.array([4.0, 9.0, 3.0, 5.0, 9.5, 1.0])
    assert zone_shard_balanced(T9, 0, 2).tolist() == [0, 2, 4]
    assert zone_shard_balanced(T9, 1, 2).tolist() == [1, 3, 5]
    # three ranks: 0 1 2 2 1 0  ->  rank 0: {4, 5}, rank 1: {1, 2}, rank 2: {3, 0}
    assert [zone_shard_balanced(T9, r, 3).tolist() for r in range(3)] == [[4, 5], [1, 2], [0, 3]]
    with pytest.raises(ValueError):
        zone_shard_balanced(T9, 2, 2)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank: int, world: int, port: int, total: int, out_dir: str):
    import torch.distributed as dist

    from gen import build_config
    from oracle import Oracle

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        c = build_config(3, zones=total)
        lo, hi = zone_shard(total, rank, world)
        out = Oracle(c["network"]).integrate(c["T9"][lo:hi], c["rho"][lo:hi], c["Y0"][lo:hi], c["t_hydro"])
        # per-rank "time" = its sub-step count (deterministic stand-in for a clock)
        my_time, my_steps = float(out["n_steps"].sum()), int(out["n_steps"].sum())
        (t_max,), (zones_all, steps_all) = reduce_job([my_time], [hi - lo, my_steps])
        np.savez(os.path.join(out_dir, f"rank{rank}.npz"), Y=out["Y"], n_steps=out["n_steps"], lo=lo,
                 hi=hi, t_max=t_max, zones_all=zones_all, steps_all=steps_all, my_time=my_time)
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_reassemble_the_single_process_result(tmp_path):
    import torch.multiprocessing as mp

    from gen import build_config
    from oracle import Oracle

    total, world = 13, 2  # ragged: 7 + 6 zones
    mp.spawn(_rank_main, args=(world, _free_port(), total, str(tmp_path)), nprocs=world, join=True)
    c = build_config(3, zones=total)
    ref = Oracle(c["network"]).integrate(c["T9"], c["rho"], c["Y0"], c["t_hydro"])
    parts = [np.load(tmp_path / f"rank{r}.npz") for r in range(world)]
    assert [int(p["lo"]) for p in parts] == [0, 7] and [int(p["hi"]) for p in parts] == [7, 13]
    Y = np.concatenate([p["Y"] for p in parts])
    steps = np.concatenate([p["n_steps"] for p in parts])
    assert np.array_equal(Y, ref["Y"])  # zones are independent: sharding changes nothing
    assert np.array_equal(steps, ref["n_steps"])
    for p in parts:  # every rank holds the same job-level figures
        assert float(p["zones_all"]) == total
        assert float(p["steps_all"]) == float(ref["n_steps"].sum())
        assert float(p["t_max"]) == max(float(q["my_time"]) for q in parts)


def _ramp_profile(total: int):
    """A grid whose hot zones are neighbours: T9 falls along the zone index (the i.i.d. profile
    of configs[2] hides the imbalance a contiguous split has on such a grid)."""
    from gen import build_config

    c = build_config(3, zones=total)
    return c, np.linspace(9.5, 1.5, total)


def _rank_balanced(rank: int, world: int, port: int, total: int, out_dir: str):
    import torch.distributed as dist

    from oracle import Oracle

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        c, T9 = _ramp_profile(total)
        idx = zone_shard_balanced(T9, rank, world)
        out = Oracle(c["network"]).integrate(T9[idx], c["rho"][idx], c["Y0"][idx], c["t_hydro"])
        my_steps = int(out["n_steps"].sum())
        (t_max,), (zones_all, steps_all) = reduce_job([float(my_steps)], [len(idx), my_steps])
        np.savez(os.path.join(out_dir, f"rank{rank}.npz"), Y=out["Y"], n_steps=out["n_steps"], idx=idx,
                 t_max=t_max, zones_all=zones_all, steps_all=steps_all)
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_balanced_shards_even_out_a_grid_with_contiguous_hot_zones(tmp_path):
    """PAPER.md L200 (fn. 1): zones need varying numbers of steps.  On a temperature ramp the
    contiguous split leaves one of two ranks with most of the sub-steps; the temperature deal
    brings both within 10 % of each other, and scattering the pieces back by their indices gives
    the single-process result bit for bit (no data-path collective either way)."""
    import torch.multiprocessing as mp

    from oracle import Oracle

    total, world = 48, 2
    mp.spawn(_rank_balanced, args=(world, _free_port(), total, str(tmp_path)), nprocs=world, join=True)
    c, T9 = _ramp_profile(total)
    ref = Oracle(c["network"]).integrate(T9, c["rho"], c["Y0"], c["t_hydro"])
    parts = [np.load(tmp_path / f"rank{r}.npz") for r in range(world)]
    Y, steps = np.full_like(ref["Y"], np.nan), np.full_like(ref["n_steps"], -1)
    for p in parts:
        Y[p["idx"]], steps[p["idx"]] = p["Y"], p["n_steps"]
    assert np.array_equal(Y, ref["Y"]) and np.array_equal(steps, ref["n_steps"])
    work = [float(p["n_steps"].sum()) for p in parts]
    assert max(work) <= 1.10 * min(work), work
    contiguous = [float(ref["n_steps"][slice(*zone_shard(total, r, world))].sum()) for r in range(world)]
    assert max(contiguous) > 3 * min(contiguous), contiguous  # what the deal is there to remove
    for p in parts:
        assert float(p["zones_all"]) == total and float(p["steps_all"]) == float(ref["n_steps"].sum())
        assert float(p["t_max"]) == max(work)
