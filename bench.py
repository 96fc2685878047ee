"""bench.py -- zone-networks integrated per second over one hydro step
(150 species / 1604 reactions, fp64): BASELINE.json's metric on configs[3]
(16384 zones, one hydro step of 1e-6 s, seeded synthetic network and profile).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A "step" is one net_integrate call over the whole batch (rates, then every
sub-step of every zone: the whole hot path).  Prints ONE JSON line.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "zone-networks integrated per second over one hydro step (150sp/1604rx, fp64)"
UNIT = "zone-networks/s"
ZONES_PER_GPU = 16384
T_HYDRO = 1e-6
PROFILE_SEED = 4
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the zone kernel on the default
# workload, from the `ncu --set full` capture summarised in the file named beside it (the
# writes of the last zones are still in L2 when the capture ends).  Reported only for that
# exact configuration; any other run reports null.
DRAM_BYTES_PER_LAUNCH = 20466944
DRAM_BYTES_SOURCE = "profiles/r03a_pull2_kernel.md"
SURVEY_FP64_PER_ZONE_SUBSTEP = 13000  # SURVEY.md 8(d), 150 species / 1604 reactions

# Algorithmic work per zone per sub-step: one multiply per
# reactant of every reaction, one add per F+/F- entry, ~10 flops per species for
# k, the branch, the update and the dt candidate; 8-byte shared-memory traffic:
# Y gathers, flux writes, flux gathers, ~5 words per species.
def algorithmic_work(net, n_entries):
    n_react_total = int(net.n_react.sum())
    flops = n_react_total + n_entries + 10 * net.n_species
    smem_bytes = 8 * (n_react_total + net.n_reactions + n_entries + 5 * net.n_species)
    return flops, smem_bytes


def pull_design_smem_bytes(kn, info, ybytes):
    """Shared-memory bytes per zone-substep that the PULL design itself must move (DESIGN.md
    section 6), counted from the compiled schedule, not from the kernel: every species publishes
    4 words; every P-slot reads one word, plus one per second factor; every N-slot reads one;
    the six hub rows go through shared memory once per warp (one store and one load each)."""
    if not info["pull_ok"] or info["kernel"] == 0:
        return None
    T = info["pull_threads"]
    pslots = int((kn.schedule_table("pull_slot_rxn") >= 0).sum())
    second = int((kn.schedule_table("pull_slot_f2") != 4 * T + 3).sum()) if info["pull_slots2"] else 0
    nslots = int(kn.schedule_table("pull_n_nslots").sum())
    warps = info["threads"] // 32
    return ybytes * (4 * info["n_species"] + pslots + second + nslots + 2 * 6 * warps)


# FP64 / shared-memory peaks: measured on this pool's B200 with
# `python bench_peaks.py` (profiles/peaks.json); fallback =
# unit counts x clocks.max.sm from the guides (64 FP64 lanes and 128 B of shared
# memory per clock per SM, 148 SMs, 1965 MHz).
NOMINAL_FP64_TINSTR = 148 * 64 * 1.965e9 / 1e12
NOMINAL_SMEM_TBS = 148 * 128 * 1.965e9 / 1e12


def load_peaks():
    path = os.path.join(ROOT, "profiles", "peaks.json")
    if os.path.exists(path):
        with open(path) as fh:
            p = json.load(fh)
        return p["fp64_add_tinstr_s"], p["smem_lds64_tb_s"], "measured (profiles/peaks.json)"
    return NOMINAL_FP64_TINSTR, NOMINAL_SMEM_TBS, "nominal (148 SM x 64 lanes | 128 B x 1965 MHz)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(max(mx)) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def workload(rank: int, world: int, zones_per_gpu: int = ZONES_PER_GPU, name: str = "hub150",
             shard: str = "contiguous"):
    """Weak scaling: the global batch is world x 16384 zones of one seeded profile;
    rank r integrates the contiguous shard r, or with shard = "t9" the zones dealt to it by
    falling temperature (shard.zone_shard_balanced); no data-path collective either way."""
    from gen import perturbed_co_start, zone_profile
    from gen.configs import network

    net = network(name)
    total = zones_per_gpu * world
    if world == 1:  # (the reference arm comes through here: it must not load the product library)
        lo, hi = 0, total
    else:
        from paper_1409_5826_b200.shard import zone_shard, zone_shard_balanced

        lo, hi = zone_shard(total, rank, world)
    T9, rho = zone_profile(total, PROFILE_SEED)
    Y0 = perturbed_co_start(net, total, seed=1000 + PROFILE_SEED)
    if world > 1 and shard == "t9":
        idx = zone_shard_balanced(T9, rank, world)
        return net, T9[idx].copy(), rho[idx].copy(), Y0[idx].copy()
    return net, T9[lo:hi].copy(), rho[lo:hi].copy(), Y0[lo:hi].copy()


def cpu_sample_size(o, T9, rho, Y0, cores, target_s):
    """Prefix of the workload that costs the oracle about target_s seconds on
    these cores, sized from a short probe (8 zones per core)."""
    probe = int(min(len(T9), 8 * cores))
    t0 = time.perf_counter()
    o.integrate(T9[:probe], rho[:probe], Y0[:probe], T_HYDRO, n_threads=cores)
    rate = probe / max(time.perf_counter() - t0, 1e-6)
    return int(max(probe, min(len(T9), rate * target_s)))


def cpu_baseline(net, T9, rho, Y0, target_s=15.0, method=0):
    """The oracle as it stands on the host cores, on a bounded prefix sample
    (about target_s seconds of CPU work)."""
    from oracle import Oracle, OracleParams, max_threads

    cores = max_threads()
    o = Oracle(net, OracleParams(method=method))
    n = cpu_sample_size(o, T9, rho, Y0, cores, target_s)
    t0 = time.perf_counter()
    out = o.integrate(T9[:n], rho[:n], Y0[:n], T_HYDRO, n_threads=cores)
    best = time.perf_counter() - t0
    steps = int(out["n_steps"].sum())
    return {"value": n / best, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {n} of {len(T9)} zones of the same workload, {steps} sub-steps, "
                      f"{best:.2f} s, gcc -O2 -ffp-contract=off, OpenMP dynamic over zones",
            "zone_substeps_per_s": steps / best}


def cpu_baseline_1core(net, T9, rho, Y0, zones=64, method=0):
    """BASELINE.md CPU-baseline plan (i): the oracle on ONE host core, first `zones` zones."""
    from oracle import Oracle, OracleParams

    o = Oracle(net, OracleParams(method=method))
    t0 = time.perf_counter()
    out = o.integrate(T9[:zones], rho[:zones], Y0[:zones], T_HYDRO, n_threads=1)
    el = time.perf_counter() - t0
    steps = int(out["n_steps"].sum())
    return {"value": zones / el, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"first {zones} zones of the same workload, {steps} sub-steps, {el:.2f} s, one thread",
            "zone_substeps_per_s": steps / el}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    net, T9, rho, Y0 = workload(0, 1)
    from oracle import Oracle, max_threads

    cores = max_threads()
    o = Oracle(net)
    # each step a bounded sample: the whole --steps/--warmup run ends within ~2 minutes
    n = cpu_sample_size(o, T9, rho, Y0, cores, 100.0 / max(1, args.steps + args.warmup))
    for _ in range(args.warmup):
        o.integrate(T9[:n], rho[:n], Y0[:n], T_HYDRO, n_threads=cores)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        out = o.integrate(T9[:n], rho[:n], Y0[:n], T_HYDRO, n_threads=cores)
    el = time.perf_counter() - t0
    value = n * args.steps / el
    sample = (f"each step = first {n} of {ZONES_PER_GPU} zones, {int(out['n_steps'].sum())} sub-steps; "
              "gcc -O2 -ffp-contract=off, OpenMP dynamic over zones")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": el / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": "configs[3]: hub150 (150sp/1604rx), one hydro step 1e-6 s; CPU oracle on a bounded sample",
                   "zones_per_step": n},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def run_ours(args):
    import torch

    import paper_1409_5826_b200 as K

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist

        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    assert world == args.gpus, f"--gpus {args.gpus} but WORLD_SIZE={world}"
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)

    net, T9h, rhoh, Y0h = workload(rank, world, args.zones, args.network, args.shard)
    z, N = Y0h.shape
    method = {"asymptotic": 0, "qss": 1}[args.method]
    kn = K.Net(net, K.NetParams(precision=args.precision, kernel=args.kernel, method=method))
    info = kn.schedule_info()
    ynp = np.float64 if args.precision == 64 else np.float32
    ybytes = 8 if args.precision == 64 else 4
    Y0h = np.ascontiguousarray(Y0h.astype(ynp))
    T9, rho = torch.from_numpy(T9h).to(dev), torch.from_numpy(rhoh).to(dev)
    Y0 = torch.from_numpy(Y0h).to(dev)
    Y = torch.empty_like(Y0)
    dt = torch.zeros(z, dtype=torch.float64, device=dev)
    n_steps = torch.zeros(z, dtype=torch.int32, device=dev)
    status = torch.zeros(z, dtype=torch.int32, device=dev)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)  # > 126 MB L2
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def one_step(timed_events=None):
        Y.copy_(Y0)       # restore the start state outside the timed launch
        dt.zero_()
        flush.zero_()     # L2 flush between timed iterations
        if timed_events is not None:
            timed_events[0].record(stream)
        kn.net_integrate(z, T9, rho, Y, T_HYDRO, dt, n_steps, status, stream)
        if timed_events is not None:
            timed_events[1].record(stream)

    for _ in range(args.warmup):
        one_step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    events = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
              for _ in range(args.steps)]
    barrier()
    t0 = time.perf_counter()
    for ev in events:
        one_step(ev)
    barrier()
    wall = time.perf_counter() - t0
    clocks = sampler.stop() if rank == 0 else None
    kernel_ms = [a.elapsed_time(b) for a, b in events]
    total_ms = float(sum(kernel_ms))
    substeps = int(n_steps.sum().item())
    assert int(status.max().item()) == 0, "a zone reported a status bit"

    # ---- e2e: the same step through the host-buffer entry point ------------------
    # pinned HOST buffers in, results back in pinned HOST buffers, everything inside the timed
    # region.  Default: zero-copy (the zone kernel reads and writes the mapped host buffers
    # itself).  Also timed: the staged path (cudaMemcpyAsync through device scratch).
    Ysrc = torch.from_numpy(Y0h.copy())
    Yp = torch.from_numpy(Y0h.copy()).pin_memory()
    T9p, rhop = torch.from_numpy(T9h.copy()).pin_memory(), torch.from_numpy(rhoh.copy()).pin_memory()
    dtp = torch.zeros(z, dtype=torch.float64).pin_memory()
    stp = torch.zeros(z, dtype=torch.int32).pin_memory()
    sts = torch.zeros(z, dtype=torch.int32).pin_memory()
    e2e_steps = max(1, min(args.steps, 5))

    def time_host_path(net_obj):
        total = 0.0
        for it in range(1 + e2e_steps):
            Yp.copy_(Ysrc)
            dtp.zero_()
            flush.zero_()
            barrier()
            t1 = time.perf_counter()
            net_obj.net_integrate_host(z, T9p.numpy(), rhop.numpy(), Yp.numpy(), T_HYDRO, dtp.numpy(),
                                       stp.numpy(), sts.numpy())
            if it > 0:
                total += time.perf_counter() - t1
        assert int(sts.max()) == 0 and int(stp.sum()) == substeps
        return total

    e2e_s = time_host_path(kn)
    kn_staged = K.Net(net, K.NetParams(precision=args.precision, kernel=args.kernel, host_chunk=-z, method=method))
    staged_s = time_host_path(kn_staged)
    h2d = z * (N * ybytes + 8 + 8 + 8)
    d2h = z * (N * ybytes + 8 + 4 + 4)
    steps_host = n_steps.cpu().numpy()

    # ---- secondary points: config 3 and config 5 ---------------
    extra = {}
    if world == 1 and not args.no_extra and args.network == "hub150" and args.precision == 64 and method == 0:
        from gen import build_config

        def dev_t(a, dtype=torch.float64):
            return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype).to(dev)

        c3 = build_config(3)
        z3 = c3["zones"]
        T3, r3, Y3 = dev_t(c3["T9"]), dev_t(c3["rho"]), dev_t(c3["Y0"])
        Yw, dtw = torch.empty_like(Y3), torch.zeros(z3, dtype=torch.float64, device=dev)
        st3 = torch.zeros(z3, dtype=torch.int32, device=dev)
        best3, sub3 = None, 0
        for it in range(3):
            Yw.copy_(Y3)
            dtw.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            sub3 = 0
            e0.record(stream)
            for _ in range(c3["calls"]):
                kn.net_integrate(z3, T3, r3, Yw, c3["t_hydro"], dtw, st3, None, stream)
            e1.record(stream)
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            best3 = ms if best3 is None else min(best3, ms)
        extra["config3"] = {"what": "configs[2]: 128 zones x 10 consecutive hydro steps, dt carried (best of 3)",
                            "ms_per_10_calls": best3, "zone_networks_per_s": z3 * c3["calls"] / (best3 * 1e-3)}
        c5 = build_config(5)
        k5 = K.Net(c5["network"])
        z5 = c5["zones"]
        T5, r5, Y5 = dev_t(c5["T9"]), dev_t(c5["rho"]), dev_t(c5["Y0"])
        Yw, dtw = torch.empty_like(Y5), torch.zeros(z5, dtype=torch.float64, device=dev)
        st5 = torch.zeros(z5, dtype=torch.int32, device=dev)
        best5 = None
        for it in range(3):
            Yw.copy_(Y5)
            dtw.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            k5.net_integrate(z5, T5, r5, Yw, c5["t_hydro"], dtw, st5, None, stream)
            e1.record(stream)
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            best5 = ms if best5 is None else min(best5, ms)
        sub5 = int(st5.sum().item())
        extra["config5"] = {"what": "configs[4]: hub365 (365sp/4400rx), 4096 zones, one hydro step (best of 3)",
                            "ms": best5, "zone_networks_per_s": z5 / (best5 * 1e-3), "sub_steps": sub5,
                            "ns_per_zone_substep": best5 * 1e6 / sub5,
                            "kernel": k5.schedule_info()["kernel"], "threads_per_zone": k5.schedule_info()["threads"]}

        # the secondary claims on the configs[3] batch itself, one launch each, best of 3 (VERDICT r02
        # item 5: a regression on any of them must show in the driver's line)
        def variant(label, what, network_name="hub150", **params):
            vnet, Yvh = (net, Y0h) if network_name == "hub150" else workload(0, 1, z, network_name)[::3]
            prec = params.get("precision", 64)
            kv = K.Net(vnet, K.NetParams(**params))
            Yv0 = torch.from_numpy(np.ascontiguousarray(Yvh.astype(np.float64 if prec == 64 else np.float32))).to(dev)
            Yv, dtv = torch.empty_like(Yv0), torch.zeros(z, dtype=torch.float64, device=dev)
            stv = torch.zeros(z, dtype=torch.int32, device=dev)
            sv = torch.zeros(z, dtype=torch.int32, device=dev)
            best = None
            for it in range(3):
                Yv.copy_(Yv0)
                dtv.zero_()
                flush.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                kv.net_integrate(z, T9, rho, Yv, T_HYDRO, dtv, stv, sv, stream)
                e1.record(stream)
                torch.cuda.synchronize()
                ms = e0.elapsed_time(e1)
                best = ms if best is None else min(best, ms)
            sub = int(stv.sum().item())
            vi = kv.schedule_info()
            extra[label] = {"what": what + f", {z} zones, one hydro step (best of 3)", "ms": best,
                            "zone_networks_per_s": z / (best * 1e-3), "sub_steps": sub,
                            "ns_per_zone_substep": best * 1e6 / sub, "kernel": vi["kernel"],
                            "threads_per_zone": vi["threads"], "status_max": int(sv.max().item())}
            kv.close()

        variant("hub150hh", "hub150 + 16 heavy + heavy fusion pairs and inverses (N-slots)", "hub150hh")
        variant("qss", "QSS variant of the update (net_params_t.method = 1)", method=1)
        variant("fp32", "single-precision study (PAPER.md L132)", precision=32)
        variant("kernel2", "forced one-species-per-thread pull kernel (params.kernel = 2)", kernel=2)
        variant("kernel1", "forced generic flux-array kernel (params.kernel = 1)", kernel=1)

        # SURVEY 8(d)'s optional "pre-burned" variant: the second consecutive hydro step of the same
        # batch (start = state after one call, dt carried; tens of species populated instead of two)
        best_pb, sub_pb = None, 0
        stpb = torch.zeros(z, dtype=torch.int32, device=dev)
        for it in range(3):
            Y.copy_(Y0)
            dt.zero_()
            kn.net_integrate(z, T9, rho, Y, T_HYDRO, dt, None, None, stream)
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            kn.net_integrate(z, T9, rho, Y, T_HYDRO, dt, stpb, status, stream)
            e1.record(stream)
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            best_pb = ms if best_pb is None else min(best_pb, ms)
        sub_pb = int(stpb.sum().item())
        extra["preburned"] = {"what": f"second consecutive hydro step of the configs[3] batch ({z} zones, start = state "
                                      "after one call, dt carried; best of 3)",
                              "ms": best_pb, "zone_networks_per_s": z / (best_pb * 1e-3), "sub_steps": sub_pb,
                              "ns_per_zone_substep": best_pb * 1e6 / sub_pb, "status_max": int(status.max().item())}

        # pageable host buffers through the staged pipeline in 4 chunks (kinnet.h: upload and kernels
        # of chunk c are enqueued before the blocking download of chunk c-1)
        kn_page = K.Net(net, K.NetParams(host_chunk=-(z // 4)))
        best_p = None
        for it in range(3):
            Ypg, dtpg = Y0h.copy(), np.zeros(z)
            stpg, sspg = np.zeros(z, np.int32), np.zeros(z, np.int32)
            flush.zero_()
            torch.cuda.synchronize()
            t1 = time.perf_counter()
            kn_page.net_integrate_host(z, T9h, rhoh, Ypg, T_HYDRO, dtpg, stpg, sspg)
            el = time.perf_counter() - t1
            if it > 0:
                best_p = el if best_p is None else min(best_p, el)
        assert int(sspg.max()) == 0 and int(stpg.sum()) == substeps
        extra["host_pageable_4chunks"] = {
            "what": "net_integrate_host on PAGEABLE numpy buffers, staged path in 4 chunks of "
                    f"{z // 4} zones over three streams (host wall clock, best of 2 after one warm-up)",
            "ms": best_p * 1e3, "zone_networks_per_s": z / best_p}
        kn_page.close()

    # ---- max over ranks ---------------------------------------------------
    from paper_1409_5826_b200.shard import reduce_job

    best_ms, median_ms = float(np.min(kernel_ms)), float(np.median(kernel_ms))
    (total_ms, e2e_s, staged_s, best_ms, median_ms), (substeps_all,) = reduce_job(
        [total_ms, e2e_s, staged_s, best_ms, median_ms], [substeps], device=dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    ms_per_step = total_ms / args.steps
    value = z * world / (ms_per_step * 1e-3)
    e2e_value = z * world / (e2e_s / e2e_steps)
    staged_value = z * world / (staged_s / e2e_steps)
    flops, smem_b = algorithmic_work(net, info["n_entries"])
    pull_b = pull_design_smem_bytes(kn, info, ybytes)
    fp64_peak, smem_peak, peak_src = load_peaks()
    per_launch_substeps = substeps  # rank 0's launch
    k_ms = float(np.mean(kernel_ms))
    fp64_ach = flops * per_launch_substeps / (k_ms * 1e-3) / 1e12
    default_run = (z == ZONES_PER_GPU and args.precision == 64 and args.kernel == 0 and args.network == "hub150"
                   and method == 0)
    traffic = DRAM_BYTES_PER_LAUNCH if default_run else None
    dtype = "f64" if args.precision == 64 else "f32"
    kname = ({0: "zone_kernel", 1: "zone_kernel_pull", 2: "zone_kernel_pull2"}[info["kernel"]]
             + f"<{'double' if args.precision == 64 else 'float'}, adaptive>")
    out = {
        "metric": METRIC if args.precision == 64 else METRIC.replace("fp64", "fp32 study"),
        "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": dtype,
        "data": "synthetic",
        "config": {
            "workload": f"configs[3]: synthetic 150sp/{net.n_reactions}rx hub network ({args.network}, seed 1409), "
                        "16384 zones per GPU, T9~U[1,10], log10 rho~U[7,9.5] (seed 4), lognormal-perturbed "
                        "C/O start, one hydro step of 1e-6 s, adaptive dt"
                        + ("" if method == 0 else "; QSS variant of the update (net_params_t.method = 1)"),
            "zones_per_gpu": z, "sub_steps_per_step": substeps_all,
            "mean_sub_steps_per_zone": substeps_all / (z * world),
            "sub_steps_per_zone": {"min": int(steps_host.min()), "median": float(np.median(steps_host)),
                                   "p99": float(np.percentile(steps_host, 99)), "max": int(steps_host.max())},
            "l2": "256 MB buffer written between timed iterations (L2 flush)",
            "parallelism": (f"zones sharded contiguously over {world} GPU(s), no collective" if args.shard == "contiguous"
                            else f"zones dealt by falling T9 over {world} GPU(s) (zone_shard_balanced), no collective"),
            "threads_per_zone": info["threads"], "zones_per_sm": info["zones_per_sm"],
        },
        "ms_per_step_best": best_ms, "ms_per_step_median": median_ms,
        "value_best": z * world / (best_ms * 1e-3), "value_median": z * world / (median_ms * 1e-3),
        "zone_substeps_per_s": substeps_all / (ms_per_step * 1e-3),
        "wall_s_timed_region": wall,
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": e2e_steps,
                "api": "net_integrate_host on pinned host buffers: zero-copy -- the zone kernel reads each "
                       "zone's inputs from, and writes its results to, the mapped host buffers over the link, "
                       "inside the timed region; no staging copy",
                "staged": {"value": staged_value,
                           "api": "the same call with params.host_chunk < 0: cudaMemcpyAsync H2D, launch, "
                                  "cudaMemcpyAsync D2H through device scratch"}},
        # per step: memset + histogram + scatter of the launch order (2 kernels) and the zone kernel
        "gpu_launches": 3 * args.steps,
        "roofline": {
            "bound": "alu", "kernel": kname, "achieved": fp64_ach,
            "peak": fp64_peak, "unit": "Tinstr/s", "frac": fp64_ach / fp64_peak, "traffic": traffic,
            "traffic_source": (f"constant from the ncu capture in {DRAM_BYTES_SOURCE}, not measured by this run"
                               if default_run else None),
            # SURVEY 8(d) quotes ~13 k FP64 instructions per zone-substep for the 150/1604 network; the
            # count above is the stricter one this file derives from the tables
            "frac_survey_count": (SURVEY_FP64_PER_ZONE_SUBSTEP * per_launch_substeps / (k_ms * 1e-3) / 1e12 / fp64_peak
                                  if args.network == "hub150" else None),
            "what": f"{flops} algorithmic FP64 instructions (FMA = 1) per zone-substep x {per_launch_substeps} "
                    f"zone-substeps per launch / {k_ms:.2f} ms; peak = FP64 issue rate, {peak_src}; "
                    f"traffic = dram bytes of one launch from the ncu capture in {DRAM_BYTES_SOURCE}"
                    + ("" if default_run else " (not this configuration: null)"),
        },
        "roofline_smem_direct": {
            "bound": "smem", "achieved": smem_b * per_launch_substeps / (k_ms * 1e-3) / 1e12, "peak": smem_peak,
            "unit": "TB/s", "frac": smem_b * per_launch_substeps / (k_ms * 1e-3) / 1e12 / smem_peak,
            "what": f"context only: {smem_b} shared-memory bytes per zone-substep of the DIRECT (flux-array) "
                    f"design of SURVEY 8(d), which this kernel does not execute; peak {peak_src}",
        },
    }
    if pull_b is not None:
        ach = pull_b * per_launch_substeps / (k_ms * 1e-3) / 1e12
        out["roofline_smem"] = {
            "bound": "smem", "achieved": ach, "peak": smem_peak, "unit": "TB/s", "frac": ach / smem_peak,
            "what": f"{pull_b} shared-memory bytes per zone-substep that the pull design must move (4 publishes per "
                    f"species, one word per P-slot, second factor and N-slot, the hub-row hand-over), counted "
                    f"from the compiled schedule; peak {peak_src}",
        }
    if extra:
        out["extra"] = extra
    if world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(net, T9h, rhoh, Y0h, method=method)
        out["cpu_baseline_1core"] = cpu_baseline_1core(net, T9h, rhoh, Y0h, method=method)
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def run_sweep(args):
    """Fig. 8 analogue (time against the number of concurrent networks)
    and Fig. 6a analogue (L154-160: time per step against the network size), on one GPU.
    Each point: 2 warm-up launches, best of 3 timed; one JSON line per point."""
    import torch

    import paper_1409_5826_b200 as K
    from gen import co_start, make_hub_network, zone_profile

    dev = torch.device("cuda", 0)
    stream = torch.cuda.current_stream()

    def time_point(net, T9h, rhoh, Y0h):
        kn = K.Net(net)
        z = len(T9h)
        T9, rho = torch.from_numpy(T9h).to(dev), torch.from_numpy(rhoh).to(dev)
        Y0 = torch.from_numpy(Y0h).to(dev)
        Y, dt = torch.empty_like(Y0), torch.zeros(z, dtype=torch.float64, device=dev)
        steps = torch.zeros(z, dtype=torch.int32, device=dev)
        best = None
        for it in range(5):
            Y.copy_(Y0)
            dt.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            kn.net_integrate(z, T9, rho, Y, T_HYDRO, dt, steps, None, stream)
            e1.record(stream)
            torch.cuda.synchronize()
            if it >= 2:
                ms = e0.elapsed_time(e1)
                best = ms if best is None else min(best, ms)
        return best, int(steps.sum().item()), kn.schedule_info()

    if args.sweep == "zones":
        net, T9h, rhoh, Y0h = workload(0, 1)
        for z in (1, 16, 74, 148, 296, 444, 445, 592, 888, 1776, 4096, 16384):
            ms, sub, info = time_point(net, T9h[:z].copy(), rhoh[:z].copy(), Y0h[:z].copy())
            print(json.dumps({"sweep": "zones", "zones": z, "ms": ms, "sub_steps": sub,
                              "zone_networks_per_s": z / (ms * 1e-3),
                              "zone_substeps_per_s": sub / (ms * 1e-3), "zones_per_sm": info["zones_per_sm"]}))
    else:
        for N, M in ((32, 330), (48, 500), (96, 1020), (150, 1604), (250, 2900), (365, 4400)):
            net = make_hub_network(N, M, seed=N)
            z = 4096
            T9h, rhoh = zone_profile(z, 6)
            ms, sub, info = time_point(net, T9h, rhoh, co_start(net, z))
            print(json.dumps({"sweep": "size", "n_species": N, "n_reactions": M, "zones": z, "ms": ms,
                              "sub_steps": sub, "ns_per_zone_substep": ms * 1e6 / sub,
                              "kernel": {0: "generic", 1: "pull (1 species/thread)", 2: "pull (2 species/thread)"}[info["kernel"]],
                              "threads_per_zone": info["threads"], "zones_per_sm": info["zones_per_sm"]}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the secondary config 3 / config 5 points")
    ap.add_argument("--zones", type=int, default=ZONES_PER_GPU,
                    help="zones per GPU (profiling only; the metric is quoted at the default)")
    ap.add_argument("--precision", type=int, default=64, choices=[64, 32],
                    help="32 = the paper's single-precision study (PAPER.md L132); the metric is fp64")
    ap.add_argument("--kernel", type=int, default=0, choices=[0, 1, 2],
                    help="net_params_t.kernel: 0 = automatic, 1 = generic flux-array kernel, "
                         "2 = one-species-per-thread pull kernel (A/B runs)")
    ap.add_argument("--network", default="hub150", choices=["hub150", "hub150hh"],
                    help="hub150 = the metric's network; hub150hh = the same plus 16 heavy + heavy reactions "
                         "and their inverses (the fast path must survive them, DESIGN.md 4.8)")
    ap.add_argument("--method", default="asymptotic", choices=["asymptotic", "qss"],
                    help="qss = the explicit quasi-steady-state variant of the update (PAPER.md L217-219, "
                         "DESIGN.md reading Q20); the metric is quoted on the paper's asymptotic method")
    ap.add_argument("--shard", default="contiguous", choices=["contiguous", "t9"],
                    help="N > 1: contiguous zone ranges, or zones dealt to ranks by falling T9 (balanced step counts)")
    ap.add_argument("--sweep", choices=["zones", "size"],
                    help="SURVEY 8(f) NEXT 1: saturation curve over the zone count (Fig. 8 analogue) or "
                         "time per sub-step over the network size (Fig. 6a analogue); one JSON line per point")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.sweep:
        run_sweep(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
