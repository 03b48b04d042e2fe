#!/usr/bin/env python
"""bench.py -- Fourier-accelerated Landau gauge-fixing throughput on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2b] [--inner 100] [--impl ours|reference]

A "step" is one lgf_iterate(inner, alpha = 0.08) call on one resident lattice: `inner` full iterations
(S1 Delta/theta/F, S2 FFT + p2max/p2 filter + inverse FFT, S3 g build, S4 link update, S5 bookkeeping) plus the
closing measurement (reading A5).  metric = iterations/s at 32^4 SU(3) fp64, 12-real storage (config C2b of
BASELINE.json configs[2]); value = N * K * inner / (max over ranks of the CUDA-event time of the K steps).
N > 1: one independent configuration per GPU (replicas, weak scaling), no collective on the
data path.  The JSON line also carries: e2e (host buffers through the C ABI), roofline (dominant kernel, live
CUDA-event timing), kernels (every kernel), iteration (whole iteration: effective = algorithmic bytes over time, and dram =
the DRAM bytes of the committed ncu capture over the same time), time_to_theta (lgf_fix),
cpu_baseline (the oracle timed on the host cores), clocks, gpu_launches, and other_configs (C3: iterate(500), C4: iterate(200) and
lgf_fix, each on its own BASELINE.json ensemble with its own kernel table, HBM fraction and clocks).

--impl reference times the CPU oracle (oracle/, radix-2 FFT mode) on the host cores on the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

ALPHA = 0.08
THETA_TOL = 1e-15
METRIC = "FA gauge-fix iterations/s at 32^4 SU(3) fp64"
UNIT = "iterations/s"

# Algorithmic HBM bytes per site per launch of each hot-path kernel:
# links cost 16*NC bytes per direction (NC = 6 two-row, 9 full), the packed field 64 B/site.
def kernel_bytes_per_site(nc: int, cb: int = 16) -> dict:
    """cb: bytes of one stored complex number (16 fp64, 8 fp32)."""
    lk = 4 * nc * cb
    fld, g = 4 * cb, 6 * cb
    return {
        "k_fft01_delta_fwd": lk + fld,       # read own links once (backward neighbours: cache), write Delta~ field
        "k_delta": lk + fld,
        "k_fft01_fwd": 2 * fld,
        "k_fft23_mid": 2 * fld,              # read + write the field (forward, filter, inverse on chip)
        "k_fft01_inv": 2 * fld,
        "k_fft01_inv_g": fld + g,
        "k_update_x": fld + 2 * lk,          # read X once (neighbours: cache), read + write links
        "k_update_g": g + 2 * lk,
        "k_update_quad": fld + 2 * lk,       # same traffic as k_update_x, one thread per link
        "k_fa_fwd1": 2 * fld,                # 64-extent planes: forward axes 0,1 from/to the field, one component per CTA
        "k_fa_inv1": 2 * fld,
        "k_finalize": 0,
        # compile-time-sized passes (fft_fast.cuh): same traffic as the generic passes they replace
        "k_fa_delta_fwd": lk + fld,
        "k_cl_delta_fwd": lk + fld,          # 64 x 64 planes: S1 + pass A on CTA pairs
        "k_ta_delta_fwd": lk + fld,          # S1 + pass A with the links staged by the TMA unit
        "k_fa_mid": 2 * fld,
        "k_fr_mid": 2 * fld,                 # pass B with whole lines in registers: same traffic
        "k_fa_inv": 2 * fld,
        "k_fa_inv_g": fld + g,               # read X~ field, write rows 0,1 of g
        "k_tb_mid": 2 * fld,                 # pass B on TMA-staged tiles: same traffic
        "k_tm_mid": 2 * fld,                 # ... 64 extents
        "k_tr_mid": 2 * fld,                 # ... 64 extents, ring of half-chunk tiles
    }


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


TRAFFIC_CSV = "profiles/r03_ncu_traffic.csv"


def ncu_traffic(kernel: str, workload: str):
    """(DRAM bytes read + written per launch of `kernel` on `workload`, the commit the capture was taken at) from the
    committed ncu --set full capture (TRAFFIC_CSV; the command that made it is in the .md beside it), or (None, None).
    The number is NOT measured in this run (a bench value is never taken under a profiler): it is stamped with the
    commit of its capture so that a reader can tell whether the kernel has changed since."""
    import csv
    kernel = {"k_fa_inv1": "k_fa_inv"}.get(kernel, kernel)      # profiling slot name -> function name ncu prints (k_fa_inv<6,6,1>)
    try:
        with open(os.path.join(ROOT, TRAFFIC_CSV)) as f:
            for r in csv.DictReader(f):
                if r["kernel"] == kernel and r.get("workload", "C2b") == workload:
                    return int(r["dram_read_bytes"]) + int(r["dram_write_bytes"]), r.get("commit")
    except Exception:
        pass
    return None, None


def ncu_iteration_traffic(kernel_names, workload: str):
    """DRAM bytes of one whole iteration on `workload` from the same committed captures: the sum over the kernels this run
    launched (`kernel_names`), or (None, ...) when one of them has no capture for this workload.  Returns (bytes, the
    per-kernel bytes, the capture commits).  Like roofline.traffic: cold-cache single launches, not measured in this run."""
    per, commits = {}, set()
    for k in kernel_names:
        b, c = ncu_traffic(k, workload)
        if b is None:
            return None, {}, []
        per[k] = b
        commits.add(c)
    return sum(per.values()), per, sorted(c for c in commits if c)


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                       "-lms", "50"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self) -> dict:
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        time.sleep(0.25)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(", ") for r in open(self.f.name).read().strip().splitlines() if r.strip()]
        os.unlink(self.f.name)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for k, nm in enumerate(names):
                if len(r) > 3 + k and r[3 + k].strip().lower() == "active":
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ---------------------------------------------------------------------------------------------- replicas (N > 1)
# The path does not shard without two all-to-all exchanges per iteration, so N GPUs fix N
# independent configurations: no collective on the data path.  torch.distributed serves the barrier and the
# max-over-ranks time only.  These three helpers are the whole multi-rank host logic; tests/test_replicas.py runs
# them at world size 2 over gloo on the CPU.
def rank_stream(cfg: dict, rank: int) -> int:
    """Philox stream of rank `rank`: its own configuration of the same ensemble."""
    return int(cfg.get("stream", 0)) + 16 * int(rank)


def max_over_ranks(x: float, dist=None, device="cpu") -> float:
    """The slowest rank's time: every multi-GPU number is the max over ranks of device times."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, steps: int, inner: int, ms: float) -> float:
    """Iterations/s of the whole job: every rank did steps*inner iterations in the (max over ranks) time ms."""
    return world * steps * inner / (ms * 1e-3)


def make_links(workload: str, rank: int):
    import ensembles as E
    cfg = dict(E.CONFIGS[workload])
    if cfg["kind"] == "pure_gauge":
        U = E.pure_gauge(cfg["dims"], cfg["seed"], rank_stream(cfg, rank))
    else:
        U = E.noisy(cfg["dims"], cfg["seed"], cfg["eps"], rank_stream(cfg, rank))   # rank r: its own configuration
    return U, cfg


def dims_name(dims):
    return "x".join(str(d) for d in dims)


# ---------------------------------------------------------------------------------------------- shared by both arms
def workload_config(name: str, cfg: dict, links: str, inner: int, world: int, beta=None, sweeps=None, overrelax=0) -> dict:
    """The `config` object of the JSON line; both arms print the same one for the same workload."""
    dims, storage = cfg["dims"], cfg["storage"]
    V = int(np.prod(dims))
    nc = 6 if storage == 12 else 9
    if links == "wilson":
        src = f"Wilson-action heat bath beta={beta}, {sweeps} sweeps (ensembles.wilson)" if not overrelax else \
              f"Wilson-action heat bath + {overrelax} over-relaxation sweeps each, beta={beta}, {sweeps} compound sweeps (ensembles.wilson)"
    elif links == "device":
        src = "device-generated links (ensembles.device_su3)"
    elif links == "noisy_device":
        src = f"eps={cfg.get('eps')} (ensembles.noisy_device: the configs[1] recipe on torch's generator, reading A12b)"
    else:
        src = f"eps={cfg.get('eps')}"
    return {"workload": f"{name}: SU(3) {dims_name(dims)} {storage}-real, {src}, seed={cfg['seed']}, alpha=0.08",
            "iterations_per_step": inner,
            "l2": ("no flush between iterations: the links (%.0f MB per GPU, read and written every iteration) are %s the 126 MB L2; "
                   "the field (%.0f MB) %s -- iteration.dram_frac_of_measured is the HBM figure, iteration.effective_* counts algorithmic bytes"
                   % (V * nc * 64 / 1e6, "larger than" if V * nc * 64 > 126e6 else "NOT larger than", V * 64 / 1e6,
                      "is larger too" if V * 64 > 126e6 else "fits in L2, so passes B and C are partly L2-fed")),
            "parallelism": "replicas" if world > 1 else "single"}


# ---------------------------------------------------------------------------------------------- reference arm
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    U, cfg = make_links(args.workload, 0)
    dims, storage = cfg["dims"], cfg["storage"]
    o = oracle.Oracle(dims, storage, fft_mode=1)
    o.load(U)
    V = int(np.prod(dims))
    per_step = max(1, min(args.inner, int(round(2.0e6 / V)) or 1))     # bounded sample: ~2 iterations at 32^4
    for _ in range(args.warmup):
        o.iterate(1, ALPHA)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.iterate(per_step, ALPHA)
    dt = time.perf_counter() - t0
    val = args.steps * per_step / dt
    cores = oracle.num_threads()
    sample = (f"{per_step} iteration(s) per timed step (a bounded sample of the workload's {args.inner}) of {args.workload} "
              f"({dims_name(dims)}, {storage}-real), oracle radix-2 FFT mode")
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(args.workload, cfg, "host", args.inner, 1),
        "sample_iterations_per_step": per_step,
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------------------------- our arm
# kernels of the closing (inner+1)-th body of lgf_iterate(inner): launched inner+1 times, the last one returns at once
# on the stop flag, so their per-iteration time is the accumulated time over `inner`
TAIL_KERNELS = {"k_fa_inv", "k_fa_inv1", "k_fft01_inv", "k_fa_inv_g", "k_fft01_inv_g", "k_update_quad", "k_update_g"}


def profile_kernels(gf, reload, V: int, kb: dict, inner: int, peak: float):
    """Per-kernel device times: CUDA events around every launch on the library's stream (plain launches)."""
    reload()
    gf.iterate(10, ALPHA)
    gf.set_profiling(True)
    gf.iterate(inner, ALPHA)
    prof = gf.get_profile()
    gf.set_profiling(False)
    kernels = {}
    tot_ms = sum(v["ms"] for v in prof.values())
    for name, v in prof.items():
        n_eff = inner if (name in TAIL_KERNELS and v["launches"] == inner + 1) else v["launches"]
        us = v["ms"] / n_eff * 1e3
        b = kb.get(name, 0) * V
        kernels[name] = {"launches": v["launches"], "avg_us": us, "share": v["ms"] / tot_ms,
                         "bytes_per_launch": b, "gbs": b / us / 1e3 if us > 0 else None,
                         "frac": (b / us / 1e3) / peak if us > 0 else None}
    dom = max((k for k in kernels if kb.get(k, 0) > 0), key=lambda k: prof[k]["ms"])
    iter_bytes = sum(kb[k] * V for k in kernels if k in kb)      # each of them runs once per iteration
    return kernels, dom, iter_bytes


def iteration_block(iter_bytes: int, V: int, it_s: float, peak: float, kernel_names=(), workload: str = "") -> dict:
    """Whole-iteration figures.  `effective_*`: ALGORITHMIC bytes (every array each kernel must read or
    write, once) x iterations/s -- a model fraction, which counts bytes an L2-resident field never moves through HBM (at
    32^4 the 67 MB field stays in the 126 MB L2 between passes, so passes B and C write ~15 MB each instead of 67).
    `dram_*`: the DRAM bytes ncu counted for the same kernels (committed capture) x the iterations/s
    of THIS run -- the HBM throughput the iteration really sustains."""
    out = {"bytes_per_site": iter_bytes // V, "bytes": iter_bytes, "basis": "effective = algorithmic bytes / time; dram = ncu DRAM bytes / time",
           "effective_gbs": iter_bytes * it_s / 1e9, "effective_frac_of_measured": iter_bytes * it_s / 1e9 / peak,
           "effective_frac_of_spec_8000": iter_bytes * it_s / 1e9 / 8000.0}
    dram, per, commits = ncu_iteration_traffic([k for k in kernel_names], workload) if kernel_names else (None, {}, [])
    out["dram_bytes_ncu"] = dram
    out["dram_gbs_ncu"] = dram * it_s / 1e9 if dram else None
    out["dram_frac_of_measured"] = dram * it_s / 1e9 / peak if dram else None
    out["dram_bytes_ncu_per_kernel"] = per or None
    out["dram_source"] = (f"{TRAFFIC_CSV} (ncu --set full, one cold-cache launch per kernel; NOT measured in this run: captured at commit {','.join(commits)})"
                          if dram else f"no capture of every kernel of this workload in {TRAFFIC_CSV}")
    return out


def timed_fix(gf, reload, tol: float) -> dict:
    """lgf_fix from freshly loaded links, wall clock with all syncs (time to theta < tol)."""
    import torch
    reload()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    r = gf.fix(ALPHA, tol, 100000)
    torch.cuda.synchronize()
    return {"ms": (time.perf_counter() - t0) * 1e3, "n_iter": r["n_iter"], "status": r["status"], "F": r["F"],
            "theta": r["theta"], "theta_tol": tol}


def other_config(lgf, E, name: str, n_iter: int, peak: float, local: int, n_cpu: int = 0) -> dict:
    """One of the other BASELINE.json configs (C3: iterate(500); C4: iterate(200)), links resident, on the config's own
    ensemble generated on the device (ensembles.noisy_device, reading A12b): throughput of `n_iter` iterations in one
    lgf_iterate call, per-kernel table, whole-iteration HBM fraction, time to theta < 1e-15, clocks."""
    import torch
    cfg = dict(E.CONFIGS[name])
    dims, storage = cfg["dims"], cfg["storage"]
    V = int(np.prod(dims))
    nc = 6 if storage == 12 else 9
    d_in = E.noisy_device(dims, cfg["seed"], cfg["eps"], cfg.get("stream", 0))
    gf = lgf.GaugeFixer(dims, storage)

    def reload():
        gf.load_links_device(d_in.data_ptr())

    reload()
    _, _, plaq = gf.measure()
    gf.iterate(20, ALPHA)                                       # warm-up: graph capture, clocks
    reps = 3
    sampler = ClockSampler(local)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(gf.stream)
    for _ in range(reps):
        gf.iterate(n_iter, ALPHA)
    e1.record(gf.stream)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1) / reps
    it_s = n_iter / (ms * 1e-3)
    kernels, dom, iter_bytes = profile_kernels(gf, reload, V, kernel_bytes_per_site(nc, 16), min(n_iter, 50), peak)
    ttt = timed_fix(gf, reload, THETA_TOL)
    ttt["plaquette"] = plaq
    gf.destroy()
    cpu = None
    if n_cpu > 0:
        # the oracle as it stands on the host cores, on the same links (5 iterations at C3, 3 at C4)
        import oracle
        o = oracle.Oracle(dims, storage, fft_mode=1)
        o.load(d_in.cpu().numpy())
        o.iterate(1, ALPHA)
        t0 = time.perf_counter()
        o.iterate(n_cpu, ALPHA)
        dt = time.perf_counter() - t0
        cpu = {"value": n_cpu / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"{n_cpu} iterations of {name} ({dims_name(dims)}, {storage}-real), oracle radix-2 FFT mode, after 1 warm-up"}
        del o
    del d_in
    torch.cuda.empty_cache()
    return {"config": workload_config(name, cfg, "noisy_device", n_iter, 1), "value": it_s, "unit": UNIT, "cpu_baseline": cpu,
            "ms_per_step": ms, "steps": reps, "iteration": iteration_block(iter_bytes, V, it_s, peak, [k for k in kernels if kernels[k]["bytes_per_launch"] > 0], name),
            "dominant_kernel": dom, "kernels": kernels, "time_to_theta": ttt, "clocks": clocks}


def run_ours(args):
    import torch
    import paper_1301_3460_b200 as lgf

    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def max_ranks(x: float) -> float:
        return max_over_ranks(x, dist, "cuda")

    import ensembles as E
    device_links = args.links in ("device", "wilson", "noisy_device")
    if device_links:
        # seeded links generated on the device: for the large shapes (C3, C4), whose host recipe takes minutes;
        # throughput does not depend on the configuration.  No end-to-end leg, no CPU baseline.
        cfg = dict(E.CONFIGS[args.workload])
        U = None
    else:
        U, cfg = make_links(args.workload, rank)
    dims, storage = cfg["dims"], cfg["storage"]
    V = int(np.prod(dims))
    nc = 6 if storage == 12 else 9
    inner = args.inner
    fp32 = args.precision == "fp32"
    gf = lgf.GaugeFixer(dims, storage, precision=lgf.LGF_FP32 if fp32 else lgf.LGF_FP64)
    for kv in args.opt:                                   # kernel-selection switches (include/lgf.h lgf_option), e.g. --opt TMA=1
        k, v = kv.split("=")
        gf.set_option(getattr(lgf, "LGF_OPT_" + k.upper()), int(v))
    if device_links:
        if args.links == "wilson":
            wilson_hist = []
            d_in = E.wilson(dims, args.beta, args.sweeps, cfg["seed"] + 100 * rank, device="cuda", overrelax=args.overrelax, history=wilson_hist)
        elif args.links == "noisy_device":
            d_in = E.noisy_device(dims, cfg["seed"], cfg["eps"], rank_stream(cfg, rank))
        else:
            d_in = E.device_su3(dims, cfg["seed"] + 100 * rank, 0.15)
        h_in = h_out = None

        def reload():
            gf.load_links_device(d_in.data_ptr())
    else:
        # pinned host copies for the end-to-end leg
        h_in = torch.from_numpy(U.view(np.float64).reshape(-1)).pin_memory()
        h_out = torch.empty_like(h_in).pin_memory()
        del U

        def reload():
            gf.load_links(h_in.numpy())
    reload()
    _, _, plaq = gf.measure()
    stream = gf.stream            # the context's own torch stream: every kernel and copy is ordered on it

    def timed(fn, steps, warmup):
        for _ in range(warmup):
            fn()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(steps):
            fn()
        e1.record(stream)
        barrier()
        return max_ranks(e0.elapsed_time(e1))       # ms

    # ---- device-resident throughput (links already in HBM)
    sampler = ClockSampler(local) if rank == 0 else None
    res = {}

    def step():
        res["F"], res["theta"] = gf.iterate(inner, ALPHA)

    for _ in range(args.warmup):
        step()
    n_before = gf.launch_count()
    ms = timed(step, args.steps, 0)
    launches = gf.launch_count() - n_before
    clocks = sampler.stop() if sampler else None
    value = whole_job_value(world, args.steps, inner, ms)

    # ---- end to end through the C ABI with host buffers: H2D of the links, the iterations, D2H of the result.
    # Two-row storage goes with the two-row host format (lgf_load_links_12 / lgf_get_links_12: rows 0,1 of every link, 384
    # instead of 576 bytes per site over PCIe); the canonical 18-real format is timed beside it (e2e_canonical).
    def step_e2e_canonical():
        gf.load_links(h_in.numpy())
        gf.iterate(inner, ALPHA)
        gf.get_links(h_out.numpy().view(np.complex128).reshape(V, 4, 3, 3))

    e2e_steps = max(2, min(args.steps, 5))
    e2e = e2e_canon = None
    if not device_links:
        ms_c = timed(step_e2e_canonical, e2e_steps, 1)
        e2e_canon = {"value": whole_job_value(world, e2e_steps, inner, ms_c), "unit": UNIT, "h2d_bytes_per_step": V * 576,
                     "d2h_bytes_per_step": V * 576 + 16, "ms_per_step": ms_c / e2e_steps, "steps": e2e_steps,
                     "host_format": "canonical [V][4][3][3][2] (lgf_load_links / lgf_get_links)"}
        e2e = e2e_canon
        if storage == 12:
            rows_in = torch.from_numpy(np.ascontiguousarray(h_in.numpy().view(np.complex128).reshape(V, 4, 3, 3)[:, :, :2]).view(np.float64).reshape(-1)).pin_memory()
            rows_out = torch.empty_like(rows_in).pin_memory()

            def step_e2e_rows():
                gf.load_links_12(rows_in.numpy())
                gf.iterate(inner, ALPHA)
                gf.get_links_12(rows_out.numpy().view(np.complex128).reshape(V, 4, 2, 3))

            ms_r = timed(step_e2e_rows, e2e_steps, 1)
            e2e = {"value": whole_job_value(world, e2e_steps, inner, ms_r), "unit": UNIT, "h2d_bytes_per_step": V * 384,
                   "d2h_bytes_per_step": V * 384 + 16, "ms_per_step": ms_r / e2e_steps, "steps": e2e_steps,
                   "host_format": "two-row [V][4][2][3][2] (lgf_load_links_12 / lgf_get_links_12; PAPER.md:45 12-real representation)"}
            del rows_in, rows_out
        # e2e is quoted on the context's own host format (two-row for 12-real storage: the paper's representation);
        # the SURVEY.md 8(b) calls lgf_load_links / lgf_get_links (canonical 18-real) ride inside the same object
        if e2e is not e2e_canon:
            e2e["canonical"] = e2e_canon

    line = None
    if rank == 0:
        peak, peak_src = measured_peak()
        kb = kernel_bytes_per_site(nc, 8 if fp32 else 16)
        kernels, dom, iter_bytes = profile_kernels(gf, reload, V, kb, inner, peak)
        try:
            copy_gbs = lgf.copy_peak_gbs(1 << 30, 10)
            stream_gbs = {"read": lgf.stream_peak_gbs(V, False, 10), "read_write_in_place": lgf.stream_peak_gbs(V, True, 10)}
        except Exception:
            copy_gbs, stream_gbs = None, None
        try:
            fp64_tflops = lgf.fp64_peak_tflops(5)
        except Exception:
            fp64_tflops = None
        it_s_1 = value / world
        # ---- time to theta < 1e-15 (lgf_fix, links resident, all syncs included)
        tol = 1e-10 if fp32 else THETA_TOL                           # fp32 bottoms out near theta = 1e-14
        ttt = timed_fix(gf, reload, tol)
        ttt.update({"plaquette": plaq, "ensemble": args.workload})
        if args.links == "wilson":
            # thermalisation statement for the generated configuration: plaquette after every sweep, and the plateau test
            from ensembles.heatbath import plateau
            mean, spread, drift = plateau(wilson_hist, window=min(5, max(1, len(wilson_hist) // 2)))
            ttt["thermalisation"] = {"beta": args.beta, "sweeps": args.sweeps, "overrelax_per_sweep": args.overrelax,
                                     "plaquette_last_sweeps": wilson_hist[-10:], "plateau_mean": mean, "plateau_spread": spread,
                                     "drift_between_last_two_windows": drift, "thermalised": bool(abs(drift) <= max(spread, 1e-4))}
        # ---- step-size scan (lgf_scan_alpha): iteration counts from the same start, one lgf_fix per alpha
        if args.scan_alpha:
            alphas = [float(v) for v in args.scan_alpha.split(",")]
            reload()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            sc = gf.scan_alpha(alphas, tol, 20000)
            torch.cuda.synchronize()
            sc["ms"] = (time.perf_counter() - t0) * 1e3
            ttt["alpha_scan"] = sc
        # ---- the same with LGF_MIXED (fp32 phase + fp64 polish), fp64 workloads only
        if not fp32:
            try:
                gm = lgf.GaugeFixer(dims, storage, precision=lgf.LGF_MIXED)
                for _ in range(2):                       # first call: graph capture of both precisions
                    if device_links:
                        gm.load_links_device(d_in.data_ptr())
                    else:
                        gm.load_links(h_in.numpy())
                    torch.cuda.synchronize()
                    t0 = time.perf_counter()
                    rm = gm.fix(ALPHA, THETA_TOL, 100000)
                    torch.cuda.synchronize()
                    tm = (time.perf_counter() - t0) * 1e3
                ttt["mixed"] = {"ms": tm, "n_iter": rm["n_iter"], "fp32_iters": gm.get_option(lgf.LGF_OPT_MIXED_FP32_ITERS),
                                "status": rm["status"], "F": rm["F"], "theta": rm["theta"]}
                gm.destroy()
            except Exception as e:                       # reported, never fatal for the headline number
                ttt["mixed"] = {"error": str(e)}
        # ---- CPU baseline: the oracle as it stands on the host cores, bounded sample
        cpu = None
        if world == 1 and not args.no_cpu_baseline and not device_links:
            import oracle
            o = oracle.Oracle(dims, storage, fft_mode=1)
            o.load(h_in.numpy().view(np.complex128).reshape(V, 4, 3, 3))
            n_cpu = max(1, int(round(30.0 * (1 << 20) / V)))      # ~13 s of CPU work at 32^4 on 16 cores
            o.iterate(1, ALPHA)
            t0 = time.perf_counter()
            o.iterate(n_cpu, ALPHA)
            dt = time.perf_counter() - t0
            cpu = {"value": n_cpu / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                   "sample": f"{n_cpu} iterations of {args.workload} ({dims_name(dims)}, {storage}-real), oracle radix-2 FFT mode, after 1 warm-up"}
            del o
        # ---- the other BASELINE.json configs (C3: iterate(500), C4: iterate(200) + lgf_fix), each on its own ensemble
        others = None
        if world == 1 and not fp32 and args.workload == "C2b" and not args.no_other_configs:
            gf.destroy()
            del h_in, h_out
            others = {}
            for nm, n_it, n_cpu in (("C3", 500, 5), ("C4", 200, 3)):
                try:
                    others[nm] = other_config(lgf, E, nm, n_it, peak, local, 0 if args.no_cpu_baseline else n_cpu)
                except Exception as e:                   # reported, never fatal for the headline number
                    others[nm] = {"error": f"{type(e).__name__}: {e}"}
        traffic, traffic_commit = ncu_traffic(dom, args.workload) if not fp32 else (None, None)
        line = {
            "metric": METRIC.replace("fp64", "fp32") if fp32 else METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if fp32 else "f64", "data": "synthetic",
            "config": dict(workload_config(args.workload, cfg, args.links, inner, world, args.beta, args.sweeps, args.overrelax), **({"options": args.opt} if args.opt else {})),
            "e2e": e2e,
            "e2e_canonical": e2e_canon,
            "gpu_launches": int(launches),
            "clocks": clocks,
            "roofline": {"bound": "hbm", "kernel": dom, "achieved": kernels[dom]["gbs"], "peak": peak, "unit": "GB/s",
                         "frac": kernels[dom]["frac"], "traffic": traffic,
                         "traffic_source": f"{TRAFFIC_CSV} (ncu --set full, one launch, cold caches; NOT measured in this run: captured at commit {traffic_commit})",
                         "peak_source": peak_src,
                         "bytes_per_launch": kernels[dom]["bytes_per_launch"], "avg_us": kernels[dom]["avg_us"],
                         "copy_kernel_gbs": copy_gbs, "stream_yardstick_gbs": stream_gbs,
                         "fp64_fma_tflops": fp64_tflops},
            "iteration": iteration_block(iter_bytes, V, it_s_1, peak, [k for k in kernels if kernels[k]["bytes_per_launch"] > 0], args.workload) if not fp32 else iteration_block(iter_bytes, V, it_s_1, peak),
            "kernels": kernels,
            "time_to_theta": ttt,
            "cpu_baseline": cpu,
            "other_configs": others,
            "final": {"F": res["F"], "theta": res["theta"]},
        }
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--inner", type=int, default=100, help="iterations per step (one lgf_iterate call)")
    ap.add_argument("--workload", default="C2b", help="ensemble name from ensembles.CONFIGS (C2b = 32^4, eps 0.35)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the C3 / C4 blocks of the default C2b run")
    ap.add_argument("--scan-alpha", default="", metavar="A1,A2,...", help="also run lgf_scan_alpha over these step sizes (time_to_theta.alpha_scan)")
    ap.add_argument("--opt", action="append", default=[], metavar="NAME=VALUE",
                    help="set a library option on the timed context (lgf_option without the LGF_OPT_ prefix), e.g. --opt TMA=1; A/B runs and profiles")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32"],
                    help="fp64: the BASELINE.json metric (default); fp32: LGF_FP32 storage and arithmetic (SURVEY.md 8(f) NEXT-1), "
                         "reported with dtype f32 and its own byte model; time_to_theta then stops at theta < 1e-10")
    ap.add_argument("--beta", type=float, default=6.0, help="--links wilson: coupling of the Wilson action")
    ap.add_argument("--sweeps", type=int, default=20, help="--links wilson: heat-bath sweeps from a cold start")
    ap.add_argument("--overrelax", type=int, default=0, help="--links wilson: over-relaxation sweeps after every heat-bath sweep")
    ap.add_argument("--links", default="host", choices=["host", "device", "noisy_device", "wilson"],
                    help="host: the seeded BASELINE.json ensemble built with numpy (default); device: seeded links generated on the GPU "
                         "(large shapes C3, C4; no e2e leg, no CPU baseline); wilson: a thermalised Wilson-action configuration generated on the GPU "
                         "(ensembles.wilson: the kind of input the paper fixes), for time_to_theta on realistic links")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3                                   # timing rule: at least 3 warm-up steps
    sys.exit(run_reference(args) if args.impl == "reference" else run_ours(args))


if __name__ == "__main__":
    main()
