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

from paper_1409_5826_b200.shard import reduce_job, zone_shard  # noqa: E402


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
