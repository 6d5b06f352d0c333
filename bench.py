#!/usr/bin/env python
"""bench.py -- BASELINE.json's metric on its config: CG iterations/s (and FFT / matvec
HBM GB/s) for the 32^4 complex64 lattice, batch of 12 Gaussian sources solved to 1e-6.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl wz|reference]

One "step" = one pass of the whole hot path over one batch: wz_cg_solve of all sources
of config 4 (every solve runs to the stop rule; nothing is skipped or cached).
Prints ONE JSON line (rank 0).  Multi-GPU: sources are independent, so
every rank solves its own batch with phi replicated and no data-path collective
("weak" scaling); time = max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "CG iterations/s at 32^4 (complex64, 12 sources to 1e-6)"
NOMINAL_HBM_GBS = 8000.0  # the "~8 TB/s" BASELINE.json's north star quotes; the roofline uses the MEASURED peak
UNIT = "CG iterations/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="wz", choices=["wz", "reference"])
    ap.add_argument("--config", default="4", help="inputs.CONFIGS key (4 = the metric's workload)")
    ap.add_argument("--sources", type=int, default=0, help="override the number of sources (0 = config's)")
    ap.add_argument("--max-iter", type=int, default=200000,
                    help="CG iteration cap; lower it ONLY for profiler runs (the line then says so)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the separate FFT / matvec timings")
    ap.add_argument("--full-table", action="store_true",
                    help="also solve config 5b (64^4; about two minutes) in the table of the other configs")
    return ap.parse_args()


def workload_string(key, cfg, nsrc):
    """One description of the workload for both arms (the driver compares the strings)."""
    return ("config %s: %s lattice, %s, %d Gaussian sources per GPU to tol %g, m=%g g=%g rho=%g, seed %d"
            % (key, "x".join(map(str, cfg["dims"])), cfg["dtype"], nsrc, cfg["tol"], cfg["m"], cfg["g"], cfg["rho"],
               cfg["seed"]))


def get_cfg(key):
    from paper_1005_3276_b200 import inputs

    k = int(key) if key.isdigit() else key
    return dict(inputs.CONFIGS[k]), k


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(cfg, n_iter, threads=0):
    """The oracle as it stands (O4', complex64-rounded CG with reliable updates) on
    source 0 of the workload for n_iter iterations; returns (iterations/s, threads, text, seconds)."""
    import numpy as np

    from oracle import wz_oracle as orc
    from paper_1005_3276_b200 import inputs

    orc.build()
    dims = cfg["dims"]
    npdt = np.complex64 if cfg["dtype"] == "c64" else np.complex128
    phi = inputs.make_phi(cfg["seed"], dims, cfg["sigma"], npdt).astype(np.complex128)
    b = inputs.make_source(cfg["seed"], 0, dims, npdt).astype(np.complex128)
    all_threads = orc.set_threads(0)
    threads = orc.set_threads(threads) if threads > 0 else all_threads
    fn = orc.cg_c64ru if cfg["dtype"] == "c64" else orc.cg
    t0 = time.perf_counter()
    _, info = fn(phi, b, cfg["m"], cfg["g"], cfg["rho"], cfg["tol"], n_iter)
    dt = time.perf_counter() - t0
    orc.set_threads(all_threads)
    its = max(info.iterations, 1)
    text = "source 0 of the workload, first %d CG iterations of the oracle (%s), %.1f s on %d threads" % (
        its, "O4' complex64+reliable updates" if cfg["dtype"] == "c64" else "O4 complex128", dt, threads)
    return its / dt, threads, text, dt


def oracle_pieces(cfg, threads):
    """Oracle timings beside the GPU's (SURVEY 8(d) "Oracle timed beside it"): one 4-spinor 4D FFT, one
    M^dag M, and CG seconds per iteration, on `threads` OpenMP threads (0 = all)."""
    import numpy as np

    from oracle import wz_oracle as orc
    from paper_1005_3276_b200 import inputs

    orc.build()
    dims = cfg["dims"]
    npdt = np.complex64 if cfg["dtype"] == "c64" else np.complex128
    phi = inputs.make_phi(cfg["seed"], dims, cfg["sigma"], npdt).astype(np.complex128)
    b = inputs.make_source(cfg["seed"], 0, dims, npdt).astype(np.complex128)
    all_threads = orc.set_threads(0)
    used = orc.set_threads(threads) if threads > 0 else all_threads
    t0 = time.perf_counter()
    orc.dft4d(b, +1, True)
    t_fft = time.perf_counter() - t0
    t0 = time.perf_counter()
    orc.apply_MdagM(phi, b, cfg["m"], cfg["g"], cfg["rho"])
    t_mv = time.perf_counter() - t0
    n_it = 2 if used == 1 else 6
    fn = orc.cg_c64ru if cfg["dtype"] == "c64" else orc.cg
    t0 = time.perf_counter()
    _, info = fn(phi, b, cfg["m"], cfg["g"], cfg["rho"], cfg["tol"], n_it)
    t_cg = (time.perf_counter() - t0) / max(info.iterations, 1)
    orc.set_threads(all_threads)
    return {"threads": used, "fft4d_4spinor_s": t_fft, "MdagM_s": t_mv, "cg_s_per_iteration": t_cg,
            "cg_iterations_per_s": 1.0 / t_cg, "cg_sample_iterations": n_it}


def small_config_table(dev, full=False):
    """Time to solution and CG iterations/s at the configs other than the metric's (BASELINE.json configs 1, 2,
    3, 5a, [5b], and config 4 with a single source), each with the iteration chunks replayed as a CUDA graph
    and enqueued kernel by kernel, next to the oracle's time on the host cores: full solve for configs 1, 2,
    per-iteration sample x the GPU's iteration count (labelled extrapolated) for config 3
    ("Small configs (1-3) ... report absolute times")."""
    import numpy as np
    import torch

    from oracle import wz_oracle as orc
    from paper_1005_3276_b200 import inputs, wz

    table = {}
    keys = [(1, None), (2, None), (3, None), (4, 1), ("5a", None)] + ([("5b", None)] if full else [])
    for key, nsrc_override in keys:
        cfg = inputs.CONFIGS[key]
        dims, nsrc = cfg["dims"], nsrc_override or cfg["nsrc"]
        npdt = np.complex64 if cfg["dtype"] == "c64" else np.complex128
        phi = inputs.make_phi(cfg["seed"], dims, cfg["sigma"], npdt)
        b = inputs.make_sources(cfg["seed"], nsrc, dims, npdt)
        d_phi, d_b = torch.from_numpy(phi).to(dev), torch.from_numpy(b).to(dev)
        plan = wz.Plan(dims, cfg["dtype"], nsrc, dev)
        x = torch.empty(b.shape, dtype=torch.complex128, device=dev)
        row = {"lattice": "x".join(map(str, dims)), "dtype": cfg["dtype"], "sources": nsrc, "tol": cfg["tol"]}
        for graph in (True, False):
            plan.set_graph(graph)
            best = None
            for rep in range(3 if key in (1, 2, 3) else 1):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                _, infos = plan.cg_solve(d_phi, d_b, cfg["m"], cfg["g"], cfg["rho"], cfg["tol"], 500000, out=x,
                                         raise_on_fail=False)
                e1.record()
                e1.synchronize()
                t = e0.elapsed_time(e1) * 1e-3
                best = t if best is None else min(best, t)
            its = sum(i.iterations for i in infos)
            row["graph" if graph else "stream_launches"] = {
                "time_to_solution_s": best, "iterations": [i.iterations for i in infos], "iterations_per_s": its / best,
                "us_per_iteration_per_source": 1e6 * best / max(its, 1),
                "worst_true_residual": max(i.rel_residual_true for i in infos),
                "all_converged": all(i.converged for i in infos)}
        row["graph_speedup"] = row["stream_launches"]["time_to_solution_s"] / row["graph"]["time_to_solution_s"]
        plan.close()
        if key in (1, 2, 3):
            phi128, b0 = phi.astype(np.complex128), b[0].astype(np.complex128)
            fn = orc.cg_c64ru if cfg["dtype"] == "c64" else orc.cg
            threads = orc.set_threads(0)
            if key == 3:
                t0 = time.perf_counter()
                _, io = fn(phi128, b0, cfg["m"], cfg["g"], cfg["rho"], cfg["tol"], 40)
                per_it = (time.perf_counter() - t0) / max(io.iterations, 1)
                row["oracle"] = {"kind": "extrapolated: 40-iteration sample x the GPU's iteration count of source 0",
                                 "threads": threads, "s_per_iteration": per_it,
                                 "time_to_solution_s_source0": per_it * row["graph"]["iterations"][0]}
            else:
                t0 = time.perf_counter()
                _, io = fn(phi128, b0, cfg["m"], cfg["g"], cfg["rho"], cfg["tol"], 100000)
                dt = time.perf_counter() - t0
                row["oracle"] = {"kind": "full solve", "threads": threads, "iterations": io.iterations,
                                 "time_to_solution_s_source0": dt}
        table["config_%s%s" % (key, "_single_source" if nsrc_override else "")] = row
    return table


def paper_lattice_table(dev):
    """The paper's own lattices (Tables V, VI): 4D FFT of a spinor field (Gflop/s by the
    paper's 5 N log2 N with N = 4V, reading G13) and the CG solve at Table VI's parameters m = 1, g = 1/5 with and
    without preconditioning, single and double precision.  Synthetic Gaussian phi (sigma = 0.5) stands in for the
    paper's RHMC configurations; the paper's numbers (GTX 285) ride along as context."""
    import math

    import numpy as np
    import torch

    from paper_1005_3276_b200 import inputs, wz

    paper = {  # (seconds, iterations) NPC / PC and FFT Gflop/s "cuFFT" / "ours", Tables VI and V
        ("8^3x32", "c64"): {"npc": (1.3, 830), "pc": (0.038, 8), "fft_gflops": (6.9, 24)},
        ("8^3x32", "c128"): {"npc": (4.9, 1600), "pc": (0.13, 15), "fft_gflops": (4.4, 11)},
        ("16^3x32", "c64"): {"npc": (7.1, 870), "pc": (0.20, 8), "fft_gflops": (14, 71)},
        ("16^3x32", "c128"): {"npc": (31, 1800), "pc": (0.74, 15), "fft_gflops": (10, 35)},
        ("32^3x64", "c64"): {"npc": (420, 1600), "pc": (6.8, 8), "fft_gflops": (20, None)},
        ("32^3x64", "c128"): {"npc": (2200, 3900), "pc": (25, 15), "fft_gflops": (10, None)},
    }
    out = {}
    for name, dims in (("8^3x32", (32, 8, 8, 8)), ("16^3x32", (32, 16, 16, 16)), ("32^3x64", (64, 32, 32, 32))):
        for dtype, tol in (("c64", 1e-6), ("c128", 1e-12)):
            npdt = np.complex64 if dtype == "c64" else np.complex128
            phi = torch.from_numpy(inputs.make_phi(5, dims, 0.5, npdt)).to(dev)
            b = torch.from_numpy(inputs.make_sources(5, 1, dims, npdt)).to(dev)
            plan = wz.Plan(dims, dtype, 1, dev)
            row = {"paper_GTX285": paper[(name, dtype)]}
            f = torch.empty_like(b)
            ts = []
            for i in range(8):
                a, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                plan.fft4d(b, +1, True, out=f)
                e.record()
                e.synchronize()
                if i >= 3:
                    ts.append(a.elapsed_time(e) * 1e-3)
            n4 = b.numel()
            row["fft4d_us"] = 1e6 * statistics.median(ts)
            row["fft4d_gflops_5NlogN"] = 5.0 * n4 * math.log2(n4 / 4) / statistics.median(ts) / 1e9
            for pc in (False, True):
                best, infos = None, None
                for rep in range(2):
                    a, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record()
                    _, infos = plan.cg_solve(phi, b, 1.0, 0.2, 1.0, tol, 100000, raise_on_fail=False, precondition=pc)
                    e.record()
                    e.synchronize()
                    t = a.elapsed_time(e) * 1e-3
                    best = t if best is None else min(best, t)
                row["pc" if pc else "npc"] = {"secs": best, "iterations": infos[0].iterations,
                                              "true_residual": infos[0].rel_residual_true,
                                              "converged": infos[0].converged}
            row["pc_speedup"] = row["npc"]["secs"] / row["pc"]["secs"]
            plan.close()
            out["%s_%s" % (name, dtype)] = row
    return out


def oracle_iters_for(cfg):
    V = 1
    for d in cfg["dims"]:
        V *= d
    return max(6, min(4000, int(24 * (1 << 20) / V)))


def run_reference(args):
    """--impl reference: the oracle (test infrastructure, never tuned) on the host cores,
    each step a bounded sample of the same workload.  Rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cfg, key = get_cfg(args.config)
    n_iter = oracle_iters_for(cfg)
    for _ in range(args.warmup):
        oracle_sample(cfg, max(2, n_iter // 4))
    tot_it, tot_t, threads, text = 0.0, 0.0, 0, ""
    for _ in range(args.steps):
        ips, threads, text, dt = oracle_sample(cfg, n_iter)
        tot_it += ips * dt
        tot_t += dt
    value = tot_it / tot_t
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / max(args.steps, 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_string(key, cfg, args.sources or cfg["nsrc"]),
                   "sample": "the oracle runs a bounded sample of this workload: " + text},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": text},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# algorithmic HBM bytes per launch in units of u (one spinor), nbatch = 1
ALGO_U = {"p01_fwd": 2.0, "p23_mult": 2.0, "p01_mid": 4.25, "p01_end": 3.25, "p23_fft": 2.0, "p01_inv": 2.0,
          "p01_fwdcg": 6.0, "p01_endcg": 4.25}


def rank_sources(rank: int, nsrc: int):
    """Source ids (generator streams 1 + id) of rank `rank`: every rank solves its own nsrc
    sources, disjoint across ranks, phi replicated (replicas only, no data-path collective)."""
    return list(range(rank * nsrc, (rank + 1) * nsrc))


def reduce_over_ranks(secs: float, counts, device=None):
    """Job time = MAX over ranks of the device-timed seconds; counts (iterations, launches, ...)
    = SUM over ranks.  Works with any initialised torch.distributed backend (NCCL on the GPUs,
    gloo in the CPU tests); single process: identity."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return secs, list(counts)
    t = torch.tensor([secs], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor(list(counts), dtype=torch.float64, device=device)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), [int(round(v)) for v in c.tolist()]


def load_traffic():
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f)
    return {}


def run_wz(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_1005_3276_b200 import inputs, wz

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    torch.cuda.set_device(dev)
    wz.lib()  # fail loudly if the extension is missing

    cfg, key = get_cfg(args.config)
    dims = cfg["dims"]
    nsrc = args.sources or cfg["nsrc"]
    npdt = np.complex64 if cfg["dtype"] == "c64" else np.complex128
    m, g, rho, tol = cfg["m"], cfg["g"], cfg["rho"], cfg["tol"]
    # host inputs (pinned); rank r takes sources r*nsrc .. (r+1)*nsrc-1, phi replicated
    h_phi = torch.from_numpy(inputs.make_phi(cfg["seed"], dims, cfg["sigma"], npdt)).pin_memory()
    h_b = torch.from_numpy(np.stack([inputs.make_source(cfg["seed"], j, dims, npdt)
                                     for j in rank_sources(rank, nsrc)])).pin_memory()
    d_phi, d_b = h_phi.to(dev), h_b.to(dev)
    d_x = torch.empty(h_b.shape, dtype=torch.complex128, device=dev)
    h_x = torch.empty(h_b.shape, dtype=torch.complex128).pin_memory()
    plan = wz.Plan(dims, cfg["dtype"], nsrc, dev)
    u = 4 * int(np.prod(dims)) * (8 if cfg["dtype"] == "c64" else 16)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        _, infos = plan.cg_solve(d_phi, d_b, m, g, rho, tol, args.max_iter, out=d_x, raise_on_fail=False)
        return infos

    for _ in range(args.warmup):
        infos = step()
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    plan.reset_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    iters = 0
    for _ in range(args.steps):
        infos = step()
        iters += sum(i.iterations for i in infos)
    e1.record()
    barrier()
    clocks = sampler.stop()
    launches = plan.launch_count
    secs = e0.elapsed_time(e1) * 1e-3
    conv = all(i.converged for i in infos)
    worst_true = max(i.rel_residual_true for i in infos)
    secs, (iters, launches) = reduce_over_ranks(secs, [iters, launches], dev)
    value = iters / secs

    # ---- end to end through the public API with HOST buffers (pinned), every step ----
    barrier()
    t0 = torch.cuda.Event(enable_timing=True)
    t1 = torch.cuda.Event(enable_timing=True)
    t0.record()
    d_phi.copy_(h_phi, non_blocking=True)
    d_b.copy_(h_b, non_blocking=True)
    infos_e = step()
    h_x.copy_(d_x, non_blocking=True)
    t1.record()
    barrier()
    e_secs = t0.elapsed_time(t1) * 1e-3
    e_iters = sum(i.iterations for i in infos_e)
    e_secs, (e_iters,) = reduce_over_ranks(e_secs, [e_iters], dev)
    e2e = {"value": e_iters / e_secs, "unit": UNIT,
           "h2d_bytes_per_step": int(h_phi.numel() * h_phi.element_size() + h_b.numel() * h_b.element_size()),
           "d2h_bytes_per_step": int(h_x.numel() * h_x.element_size())}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- per-kernel durations, live, CUDA events on the plan's stream (one source) ----
    peak, peak_src = measured_peaks()
    plan.profile(True)
    # the same batched solve as the timed steps, first iterations only (all sources active)
    _, pinfo = plan.cg_solve(d_phi, d_b, m, g, rho, tol, min(400, args.max_iter), out=d_x, raise_on_fail=False)
    prof = plan.profile_read()
    plan.profile(False)
    # mean duration of an ACTIVE launch: the solve also enqueues a few idle launches (chunks already
    # in flight when the last source stops; ~3 us each, they return at once), so divide the summed
    # time by the launches that did work = iterations x launches per iteration of that kind
    piters = max(i.iterations for i in pinfo)
    per_iter = {"p23_mult": 2}
    kinds = {k: {"us": 1e3 * ms / (piters * per_iter.get(k, 1)), "launches": piters * per_iter.get(k, 1), "share": 0.0}
             for k, (ms, n) in prof.items() if k in ("p01_fwdcg", "p23_mult", "p01_mid", "p01_endcg")}
    tot = sum(v["us"] * v["launches"] for v in kinds.values()) or 1.0
    for k, v in kinds.items():
        v["share"] = v["us"] * v["launches"] / tot
        v["algo_bytes"] = ALGO_U[k] * u * nsrc
        v["gbs"] = v["algo_bytes"] / (v["us"] * 1e-6) / 1e9
        v["frac"] = v["gbs"] / peak
    dom = max(kinds, key=lambda k: kinds[k]["share"])
    tr = load_traffic()
    traffic = tr.get(dom)
    roofline = {"bound": "hbm", "kernel": dom, "achieved": kinds[dom]["gbs"], "peak": peak, "unit": "GB/s",
                "frac": kinds[dom]["frac"], "traffic": traffic,
                "traffic_source": tr.get("_source", "none") + " (static file, refreshed with every kernel change; "
                                  "not measured in this run)",
                "peak_source": peak_src, "nominal_peak": NOMINAL_HBM_GBS,
                "frac_of_nominal": kinds[dom]["gbs"] / NOMINAL_HBM_GBS,
                "algo_bytes_per_launch": kinds[dom]["algo_bytes"], "us_per_launch": kinds[dom]["us"],
                "share_of_step": kinds[dom]["share"],
                "all_kernels": {k: {"us": round(v["us"], 2), "GB/s": round(v["gbs"], 1), "frac": round(v["frac"], 3),
                                    "share": round(v["share"], 3)} for k, v in kinds.items()}}

    extras = {}
    if not args.no_extras:
        extras = time_pieces(plan, d_phi, d_b[:1], m, g, rho, u, peak)
        extras.update(time_pieces_batched(plan, d_phi, d_b, m, g, rho, u, peak))
    per_iter_us = 1e6 * secs * world / max(iters, 1)
    extras.update({"cg_us_per_iteration": per_iter_us, "iterations_per_source": [i.iterations for i in infos],
                   "reliable_updates_per_source": [i.reliable_updates for i in infos],
                   "time_to_solution_s_per_source": secs / args.steps / nsrc,
                   "all_converged": conv, "worst_true_residual": worst_true,
                   "cg_algorithmic_GBs": 18.5 * u / (per_iter_us * 1e-6) / 1e9,
                   "cg_frac_of_measured_peak": 18.5 * u / (per_iter_us * 1e-6) / 1e9 / peak,
                   "cg_frac_of_nominal_8TBs": 18.5 * u / (per_iter_us * 1e-6) / 1e9 / NOMINAL_HBM_GBS})

    if not args.no_extras:
        extras["preconditioned"] = time_preconditioned(plan, d_phi, d_b, d_x, cfg, secs / args.steps)
        extras["heatbath_rational_sum"] = time_rational(plan, d_phi, d_b, d_x, cfg)
        extras["mixed_precision_to_1e-10"] = time_mixed(plan, d_phi, d_b, cfg, dev)

    if not args.no_extras and key == 4:
        extras["binary16_storage_to_1e-6"] = time_half_storage(plan, d_phi, d_b, d_x, cfg, secs / args.steps,
                                                               [i.iterations for i in infos])

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        ips, threads, text, _ = oracle_sample(cfg, oracle_iters_for(cfg))
        cpu = {"value": ips, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": text,
               # two columns (1 thread, all cores); FFT, M^dag M and CG per iteration of the oracle
               "all_cores": oracle_pieces(cfg, 0), "one_thread": oracle_pieces(cfg, 1)}
        if not args.no_extras:
            extras["other_configs"] = small_config_table(dev, args.full_table)
            extras["paper_lattices_tables_V_VI"] = paper_lattice_table(dev)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32 (complex64 vectors, f64 reductions, complex128 reliable updates)"
        if cfg["dtype"] == "c64" else "f64",
        "data": "synthetic",
        "config": {"workload": workload_string(key, cfg, nsrc),
                   "l2": "no flush: working set of one solve (8 vectors, %.0f MB) exceeds the 126 MB L2" % (8.25 * u / 1e6),
                   "sources": "independent, advanced in lock step through shared launches; sharded across ranks, phi replicated"},
        "max_iter": args.max_iter, "valid": bool(conv),
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
        "cpu_baseline": cpu, "extras": extras,
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def time_pieces(plan, d_phi, d_b1, m, g, rho, u, peak):
    """FFT and matvec timed separately (config 4), warm and with an L2 flush between
    repetitions (cold), CUDA events on the plan's stream."""
    import torch

    out = torch.empty_like(d_b1)
    scratch = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=d_b1.device)

    def timed(fn, reps=20, cold=False):
        ts = []
        for i in range(reps + 3):
            if cold:
                scratch.fill_(i & 0xFF)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn()
            b.record()
            b.synchronize()
            if i >= 3:
                ts.append(a.elapsed_time(b) * 1e-3)
        return statistics.median(ts), min(ts)

    V4 = d_b1.numel()
    import math
    flops_fft = 5.0 * V4 * math.log2(V4 / 4)
    res = {}
    for name, fn, nu in [
        ("fft4d_forward", lambda: plan.fft4d(d_b1, +1, True, out=out), 4.0),
        ("fft4d_inverse", lambda: plan.fft4d(d_b1, -1, True, out=out), 4.0),
        ("apply_M", lambda: plan.apply_M(d_phi, d_b1, m, g, rho, False, out=out), 7.25),
        ("apply_MdagM", lambda: plan.apply_MdagM(d_phi, d_b1, m, g, rho, out=out), 13.5),
    ]:
        for cold in (False, True):
            med, mn = timed(fn, cold=cold)
            key = name + ("_cold" if cold else "_warm")
            res[key] = {"us_median": 1e6 * med, "us_min": 1e6 * mn, "algo_GBs": nu * u / med / 1e9,
                        "frac_of_peak": nu * u / med / 1e9 / peak}
            if name.startswith("fft4d"):
                res[key]["gflops_5NlogN"] = flops_fft / med / 1e9
    res["matvecs_per_s_warm"] = 1.0 / (res["apply_MdagM_warm"]["us_median"] * 1e-6)
    return res


def time_pieces_batched(plan, d_phi, d_b, m, g, rho, u, peak):
    """The same calls on the whole batch of sources (steady state: ~20 waves per launch, working
    set far beyond L2); times are per source."""
    import torch

    nb = d_b.shape[0]
    out = torch.empty_like(d_b)
    res = {}
    for name, fn, nu in [
        ("fft4d_forward", lambda: plan.fft4d(d_b, +1, True, out=out), 4.0),
        ("fft4d_inverse", lambda: plan.fft4d(d_b, -1, True, out=out), 4.0),
        ("apply_M", lambda: plan.apply_M(d_phi, d_b, m, g, rho, False, out=out), 7.25),
        ("apply_MdagM", lambda: plan.apply_MdagM(d_phi, d_b, m, g, rho, out=out), 13.5),
    ]:
        ts = []
        for i in range(13):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn()
            b.record()
            b.synchronize()
            if i >= 3:
                ts.append(a.elapsed_time(b) * 1e-3 / nb)
        med = statistics.median(ts)
        res[name + "_batched"] = {"us_median_per_source": 1e6 * med, "algo_GBs": nu * u / med / 1e9,
                                  "frac_of_peak": nu * u / med / 1e9 / peak, "sources": nb}
    res["matvecs_per_s_batched"] = 1.0 / (res["apply_MdagM_batched"]["us_median_per_source"] * 1e-6)
    return res


def time_preconditioned(plan, d_phi, d_b, d_x, cfg, plain_secs):
    """NEXT-1 (Table VI): the same batch through wz_cg_solve_pc, at the
    workload's own (strong) coupling and at the paper's Table VI parameters m = 1, g = 1/5."""
    import torch

    def solve(m, g, pc):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        _, infos = plan.cg_solve(d_phi, d_b, m, g, cfg["rho"], cfg["tol"], 200000, out=d_x,
                                 raise_on_fail=False, precondition=pc)
        b.record()
        b.synchronize()
        return a.elapsed_time(b) * 1e-3, infos

    t_pc, i_pc = solve(cfg["m"], cfg["g"], True)
    t_w0, i_w0 = solve(1.0, 0.2, False)
    t_w1, i_w1 = solve(1.0, 0.2, True)
    return {
        "workload_coupling": {"plain_s": plain_secs, "pc_s": t_pc, "speedup": plain_secs / t_pc,
                              "pc_iterations": [i.iterations for i in i_pc],
                              "pc_worst_true_residual": max(i.rel_residual_true for i in i_pc),
                              "pc_all_converged": all(i.converged for i in i_pc)},
        "table_VI_parameters_m1_g0.2": {"plain_s": t_w0, "pc_s": t_w1, "speedup": t_w0 / t_w1,
                                        "plain_iterations": [i.iterations for i in i_w0],
                                        "pc_iterations": [i.iterations for i in i_w1],
                                        "paper": "Table VI, GTX 285: 8 iterations (single), speed-up 34-62"},
    }


def time_rational(plan, d_phi, d_b, d_x, cfg):
    """NEXT-2 (Eq. 7.6-7.7, 927-950, Table VII): the degree-20 rational sum, three ways --
    one plain solve per shift (Eq. 7.13), the paper's rule (preconditioned, Eq. 7.14, up to beta = 100, plain
    above), and multi-shift CG (all shifts above the cutoff, or all shifts, from one Krylov space) -- at the
    paper's heatbath parameters m = 1, g = 0.1 for the whole batch and at the workload's own coupling for two
    sources.  The shifts are a synthetic geometric ladder (inputs.rational_ladder): the paper's coefficients
    are not printed."""
    import torch

    from paper_1005_3276_b200 import inputs

    a0, al, be = inputs.rational_ladder(20, 1e-2, 1e3)

    def run(phi, b, out, m, g, cutoff, ms, max_iter):
        a, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        _, infos = plan.rational_apply(phi, b, m, g, a0, al, be, cfg["rho"], cfg["tol"], max_iter, out=out,
                                       raise_on_fail=False, pc_cutoff=cutoff, multishift=ms)
        e.record()
        e.synchronize()
        its = [[i.iterations for i in row] for row in infos]
        return {"secs": a.elapsed_time(e) * 1e-3, "sources": len(its[0]),
                "iterations_per_shift_max": [max(row) for row in its],
                "iterations_sum_over_shifts": sum(max(row) for row in its),
                "all_converged": all(i.converged for row in infos for i in row),
                "worst_true_residual": max(i.rel_residual_true for row in infos for i in row)}

    res = {"shifts": 20, "paper": "Table VII, GTX 285, single: 360-540 iterations in total over 20 shifts, 0.93-220 s"}
    res["table_VII_parameters_m1_g0.1"] = {
        "paper_rule_pc_up_to_100": run(d_phi, d_b, d_x, 1.0, 0.1, 100.0, False, 5000),
        "multishift_above_100": run(d_phi, d_b, d_x, 1.0, 0.1, 100.0, True, 5000),
        "multishift_all_shifts": run(d_phi, d_b, d_x, 1.0, 0.1, -1.0, True, 5000),
        "plain_solve_per_shift": run(d_phi, d_b, d_x, 1.0, 0.1, -1.0, False, 5000)}
    b2, x2 = d_b[:2].contiguous(), d_x[:2].contiguous()
    res["workload_coupling_m%g_g%g_2_sources" % (cfg["m"], cfg["g"])] = {
        "paper_rule_pc_up_to_100": run(d_phi, b2, x2, cfg["m"], cfg["g"], 100.0, False, 100000),
        "multishift_all_shifts": run(d_phi, b2, x2, cfg["m"], cfg["g"], -1.0, True, 100000),
        "plain_solve_per_shift": run(d_phi, b2, x2, cfg["m"], cfg["g"], -1.0, False, 100000)}
    return res


def time_half_storage(plan, d_phi, d_b, d_x, cfg, c64_secs, c64_iterations):
    """NEXT-3, third form (oracle O10): the same batch to the same tolerance by wz_cg_solve_dc_half --
    defect correction with the inner solver's t, chi, r, p stored in binary16 (10.5u of traffic per iteration instead
    of 18.5u) -- next to the complex64 solver of the timed steps.  The true residual is recomputed in complex128."""
    import torch

    a, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    _, infos = plan.cg_solve_dc(d_phi, d_b, cfg["m"], cfg["g"], cfg["rho"], cfg["tol"], 1e-1, 400000, out=d_x,
                                raise_on_fail=False, half_storage=True)
    e.record()
    e.synchronize()
    t = a.elapsed_time(e) * 1e-3
    its = [i.iterations for i in infos]
    # the same storage with reliable updates instead of restarts (wz_cg_solve_half, oracle O11)
    a, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    _, iru = plan.cg_solve(d_phi, d_b, cfg["m"], cfg["g"], cfg["rho"], cfg["tol"], 400000, out=d_x, raise_on_fail=False,
                           half_storage=True)
    e.record()
    e.synchronize()
    tru = a.elapsed_time(e) * 1e-3
    itru = [i.iterations for i in iru]
    ru = {"secs": tru, "iterations": itru, "reliable_updates": [i.reliable_updates for i in iru],
          "us_per_source_iteration": 1e6 * tru / max(sum(itru), 1),
          "worst_true_residual": max(i.rel_residual_true for i in iru), "all_converged": all(i.converged for i in iru),
          "speedup_time_to_solution": c64_secs / tru}
    return {"with_reliable_updates": ru,
            "secs": t, "inner_tol": 1e-1, "inner_iterations": its, "outer_corrections": [i.reliable_updates for i in infos],
            "us_per_source_iteration": 1e6 * t / max(sum(its), 1), "worst_true_residual": max(i.rel_residual_true for i in infos),
            "all_converged": all(i.converged for i in infos),
            "complex64_solver": {"secs": c64_secs, "iterations": c64_iterations,
                                 "us_per_source_iteration": 1e6 * c64_secs / max(sum(c64_iterations), 1)},
            "speedup_per_iteration": (c64_secs / max(sum(c64_iterations), 1)) / (t / max(sum(its), 1)),
            "speedup_time_to_solution": c64_secs / t}


def time_mixed(plan, d_phi, d_b, cfg, dev, nsrc=2):
    """NEXT-3 (mixed-precision CG): the first `nsrc` sources of the workload solved to the
    double-precision tolerance 1e-10, once by the complex64 plan (complex128 reliable updates, reading G9)
    and once by a complex128 plan on the same values."""
    import torch

    from paper_1005_3276_b200 import wz

    def solve(pl, phi, b):
        a, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        _, infos = pl.cg_solve(phi, b, cfg["m"], cfg["g"], cfg["rho"], 1e-10, 200000, raise_on_fail=False)
        e.record()
        e.synchronize()
        return a.elapsed_time(e) * 1e-3, infos

    b = d_b[:nsrc].contiguous()
    t32, i32 = solve(plan, d_phi, b)
    # the other route: defect correction, complex64 inner solves restarted inside a complex128 outer loop
    a, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    _, idc = plan.cg_solve_dc(d_phi, b, cfg["m"], cfg["g"], cfg["rho"], 1e-10, 1e-3, 400000, raise_on_fail=False)
    e.record()
    e.synchronize()
    tdc = a.elapsed_time(e) * 1e-3
    plan128 = wz.Plan(cfg["dims"], "c128", nsrc, dev)
    t64, i64 = solve(plan128, d_phi.to(torch.complex128), b.to(torch.complex128))
    plan128.close()
    return {"sources": nsrc, "tol": 1e-10,
            "c64_plan": {"secs": t32, "iterations": [i.iterations for i in i32],
                         "reliable_updates": [i.reliable_updates for i in i32],
                         "worst_true_residual": max(i.rel_residual_true for i in i32),
                         "all_converged": all(i.converged for i in i32)},
            "c64_plan_defect_correction": {"secs": tdc, "inner_tol": 1e-3, "inner_iterations": [i.iterations for i in idc],
                                           "outer_corrections": [i.reliable_updates for i in idc],
                                           "worst_true_residual": max(i.rel_residual_true for i in idc),
                                           "all_converged": all(i.converged for i in idc)},
            "c128_plan": {"secs": t64, "iterations": [i.iterations for i in i64],
                          "worst_true_residual": max(i.rel_residual_true for i in i64),
                          "all_converged": all(i.converged for i in i64)},
            "speedup": t64 / t32}


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_wz(args)


if __name__ == "__main__":
    main()
