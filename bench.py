#!/usr/bin/env python
"""bench.py -- one JSON line for the collision-term hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--scaling strong|weak] [--impl reference]

A "step" is one full collision-term sweep (rbg_collision, or rbg_collision_update for the fused-Euler config: every
role, spatial cell, momentum cell and sample) of one workload.  The headline workload is BASELINE.json's largest
single-GPU fp64 config, config 4 (32^3 spatial x 20^3 momentum cells, 512 samples, 1.34e11 sample evaluations,
2.1 GB of f) -- "the most significant challenge ... high-dimensional integration at each phase space grid"
(PAPER.md:340).  At N = 1 the same line carries a `configs` object with the other BASELINE configs (1, 2, 3, 5), each
timed the same way, so that "every config at a stated fraction of the roofline" is one record.

N > 1: `--gpus N` launches N ranks by itself (torchrun, one rank per GPU) unless it already runs under torchrun.
`--scaling strong` (default): the workload's spatial cells are sharded over the ranks (paper_2308_04869_b200.sharding; the
paper's spatial sub-domains); `--scaling weak`: every rank sweeps its own copy at a distinct global
cell offset.  The path has no data-path collective; the only collective is the MAX all-reduce
of the timing.  value = sample evaluations of all ranks / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import socket
import statistics
import subprocess
import sys
import tempfile
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

import numpy as np  # noqa: E402

import workloads  # noqa: E402
from workloads import configs as wl  # noqa: E402

METRIC, UNIT = "collision_samples_per_s", "samples/s"
HEADLINE_CONFIG = 4
BLOCK_CONFIGS = (1, 2, 3, 5)

# Algorithmic FP64 work per sample of chain O1-O12 (FMA = 2 flops, every other
# add/mul/compare/sqrt/divide = 1), by |M|^2 kind, classical statistics (+10 with quantum factors).
FLOPS_PER_SAMPLE = {0: 141.0, 1: 155.0, 2: 157.0, 3: 142.0,
                    # Table III kinds: 138 (O2-O7, O10-O12) + t 11 + u 2 + T, U 2 + squares 3 + weight 3 + the row's
                    # rational function (5 / 14 / 14 / 5 / 12 / 12 / 16; a reciprocal = 1)
                    4: 164.0, 5: 173.0, 6: 173.0, 7: 164.0, 8: 171.0, 9: 171.0, 10: 175.0}
QUANTUM_EXTRA_FLOPS = 10.0
# Chain v3 (double chain only, O6): the azimuth is two tabulated angles and the addition theorem
# (2 multiplies + 2 FMAs = 6 flops) instead of two polynomial evaluations (29 flops): 23 flops fewer per sample.  The count
# is that of the tabulated form -- what an implementation has to compute -- not of the oracle's per-sample polynomials.
DOUBLE_CHAIN_V3_SAVING = 23.0
# the same count for the t-channel importance sampler (steps S1-S7), kinds 1 and 2
FLOPS_PER_SAMPLE_TCHANNEL = {1: 185.0, 2: 187.0}
FP64_LANES_PER_SM = 64          # FMA/clk/SM; confirmed by the live probe


def ncu_traffic(group, key):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu capture, profiles/traffic.json
    (written by hand from the capture named in profiles/traffic.md).  The file carries the digest of the library sources it
    was captured on; on any other build the number is not this build's, and (None, reason) is returned instead of a stale
    constant."""
    path = ROOT / "profiles" / "traffic.json"
    try:
        t = json.loads(path.read_text())
    except (OSError, ValueError):
        return None, "profiles/traffic.json missing or unreadable"
    from paper_2308_04869_b200.build import _digest
    if t.get("digest") != _digest():
        return None, (f"profiles/traffic.json was captured on build {str(t.get('digest'))[:12]}, this is build {_digest()[:12]}: "
                      "no ncu capture of this build")
    e = t.get(group, {}).get(str(key))
    if not e:
        return None, f"no capture for {group}/{key} in profiles/traffic.json"
    return float(e["dram_bytes_read"]) + float(e["dram_bytes_write"]), f"bytes per launch (dram read + write; {e['source']})"


def flops_per_sweep(problem, n_samples, fp32=False):
    tot = 0.0
    for r, p in zip(wl.roles(problem), wl.role_processes(problem)):
        q = any(problem["species"][s]["stat"] != 0 for s in r)
        table = FLOPS_PER_SAMPLE_TCHANNEL if p.get("sampler", 0) == 1 else FLOPS_PER_SAMPLE
        per = table[p["kind"]] + (QUANTUM_EXTRA_FLOPS if q else 0.0) - (0.0 if fp32 else DOUBLE_CHAIN_V3_SAVING)
        tot += per * problem["nx"] * int(np.prod(problem["grids"][r[0]]["n"])) * n_samples
    return tot


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu = gpu_index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def __enter__(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-i", str(self.gpu), "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None
        return self

    def __exit__(self, *a):
        if self.p:
            self.p.terminate()
            try:
                self.p.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.p.kill()

    def summary(self):
        self.f.flush()
        rows = [r.split(",") for r in Path(self.f.name).read_text().splitlines() if r.count(",") >= 8]
        os.unlink(self.f.name)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2]))
            except ValueError:
                continue
            for name, v in zip(names, r[5:9]):
                if v.strip().lower() == "active":
                    reasons.add(name)
        if not sm:
            # the timed region was shorter than one sampling period (configs 1 and 6): one sample right after it instead
            try:
                r = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i", str(self.gpu)],
                                   capture_output=True, text=True, timeout=20).stdout.strip().split(",")
                reasons = sorted(n for n, v in zip(names, r[5:9]) if v.strip().lower() == "active")
                return {"sm_mhz": float(r[1]), "sm_max_mhz": float(r[2]), "reasons": reasons, "samples": 0,
                        "note": "timed region shorter than the 100 ms sampling period: one sample taken right after it"}
            except (OSError, ValueError, IndexError, subprocess.TimeoutExpired):
                return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}


# ---- the oracle legs (cpu_baseline and --impl reference): the only places bench.py executes oracle/ ----------------
def oracle_leg(w, target_seconds, warmups=1):
    """Time the oracle, as it stands, on an evenly strided subset of the workload's spatial cells sized (from one
    calibration cell, which is also the warm-up) for about target_seconds of wall time on this box's host cores."""
    import oracle
    oracle.build()
    orc = oracle.Oracle(w["problem"], use_float=w["fp32"])
    nx = w["problem"]["nx"]
    per_cell = wl.sample_evals(dict(w["problem"], nx=1), w["n_samples"])
    for _ in range(max(1, warmups)):
        t0 = time.perf_counter()
        orc.collision(w["f"], w["n_samples"], w["seed"], ix_begin=0, ix_end=1)
        t_cell = time.perf_counter() - t0
    stride = max(1, int(np.ceil(nx * t_cell / max(target_seconds, 1e-3))))
    ncell = (nx + stride - 1) // stride
    t0 = time.perf_counter()
    orc.collision(w["f"], w["n_samples"], w["seed"], ix_begin=0, ix_end=nx, ix_stride=stride)
    dt = time.perf_counter() - t0
    return {"value": per_cell * ncell / dt, "unit": UNIT, "cores": oracle.threads(), "kind": "oracle",
            "sample": f"{ncell} of {nx} spatial cells (every {stride}-th linear cell index from 0); every role, momentum "
                      f"cell and sample of those cells ({per_cell * ncell:.3g} sample evaluations)", "seconds": dt}


def run_reference(args):
    """--impl reference: the oracle on this box's host cores, same config / metric (rank 0 only).  A step is a bounded
    sample of the workload (about --ref-seconds of CPU wall time)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    w = workloads.make(args.config, nx=args.nx, sampler=args.sampler)
    if args.nx is not None:
        w["name"] += f" [nx overridden to {args.nx}]"
    times, vals, r = [], [], None
    for i in range(args.steps):
        r = oracle_leg(w, args.ref_seconds, warmups=args.warmup if i == 0 else 1)
        times.append(r["seconds"]); vals.append(r["value"])
    value = float(np.mean(vals))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(times)), "higher_is_better": True,
            "scaling": args.scaling, "vs_baseline": None, "dtype": "f32" if w["fp32"] else "f64", "data": "synthetic",
            "config": config_block(w, args, 1),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"]},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def config_block(w, args, world):
    """The `config` object: identical for our arm and the reference arm of the same command."""
    return {"workload": w["name"], "cfg": w["cfg"], "nx": w.get("nx_global", w["problem"]["nx"]), "n_samples": w["n_samples"],
            "l2": "L2 flushed (256 MB write) between timed iterations", "parallelism": f"spatial-shard x{world}"}


# ---- the NEXT-4 kernels -----------------------------------------------------------------------------------------
def hbm_peak():
    try:
        peaks = json.loads((ROOT / "MEASURED_PEAKS.json").read_text())
        return float(peaks["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    except (OSError, ValueError, KeyError):
        return 6500.0, "B200_PROFILING.md fallback"


def run_be_steps(args):
    """--path be: the NEXT-4 kernels (rbg_moments, rbg_drift_step, rbg_vlasov_step) on the chosen config, one JSON line.
    A step = moments + one drift step + one Vlasov step over every phase-space cell.  HBM roofline: algorithmic bytes
    are 8 B per cell for the moments (f read once) and 16 B per cell for each stencil (f read once, f_out written once);
    peak = MEASURED_PEAKS.json hbm_gbs (sustained copy bandwidth), else the profiling guide's fallback 6500 GB/s."""
    import torch
    if int(os.environ.get("RANK", "0")) != 0:
        return
    torch.cuda.set_device(0)
    print(json.dumps(measure_be_steps(args, args.config, args.nx, args.steps, cpu_baseline=not args.no_cpu_baseline)))


def measure_be_steps(args, cfg, nx_override, steps, cpu_baseline, e2e=True):
    import torch
    import paper_2308_04869_b200 as rbg
    w = workloads.make(cfg, nx=nx_override)
    prob = w["problem"]
    nx = prob["nx"]
    side = round(nx ** (1.0 / 3.0))
    nxyz = (side, side, side) if side ** 3 == nx else (nx, 1, 1)
    charges = (-1.0, 1.0, 2.0, 0.5, -0.5, 0.0, 1.5)
    for sp, q in zip(prob["species"], charges):
        if sp.get("charge", 0.0) == 0.0:
            sp["charge"] = q                       # the Vlasov step needs charged species
    col = rbg.Collision(dict(prob, nx=nxyz))
    for kv in args.opt:
        k, v = kv.split("=")
        col.set_option(k, int(v))
    f = torch.from_numpy(w["f"]).cuda()
    out = torch.empty_like(f)
    rng = np.random.default_rng(5)
    E = torch.from_numpy(rng.normal(size=(nx, 3))).cuda()
    B = torch.from_numpy(rng.normal(size=(nx, 3))).cuda()
    cells = int(f.numel())
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()
    dx = (0.5, 0.5, 0.5)
    kernels = {"moments": (lambda: col.moments(f, stream=stream), 8.0),
               "drift": (lambda: col.drift_step(f, 0.01, dx, out=out, stream=stream), 16.0),
               "vlasov": (lambda: col.vlasov_step(f, 0.01, E, B, out=out, stream=stream), 16.0),
               # second-order flux-limited drift (Eq. 31-33): same 16 B per cell, but ~260 FP64 instructions per cell
               # (FP64-pipe-bound); reported against the same HBM peak, not part of the step
               "drift_pfl": (lambda: col.drift_step_pfl(f, 0.01, dx, out=out, stream=stream), 16.0)}
    peak, peak_src = hbm_peak()
    res, launches = {}, 0
    with ClockSampler(0) as cs:
        for name, (fn, bytes_per_cell) in kernels.items():
            for _ in range(max(args.warmup, 3)):
                fn()
            torch.cuda.synchronize()
            ts = []
            for _ in range(steps):
                flush.fill_(1)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream); fn(); e1.record(stream)
                torch.cuda.synchronize()
                ts.append(e0.elapsed_time(e1))
            launches += col.last_launch_count() * steps
            ms = sum(ts) / len(ts)
            gbs = bytes_per_cell * cells / (ms * 1e-3) / 1e9
            res[name] = {"ms": ms, "algorithmic_bytes_per_cell": bytes_per_cell, "achieved_gbs": gbs, "frac": gbs / peak,
                         "traffic": None, "traffic_unit": "not a full-size default run"}
            if nx_override is None and not args.opt:
                res[name]["traffic"], res[name]["traffic_unit"] = ncu_traffic(f"be_cfg{cfg}", name)
    clocks = cs.summary()
    t_step = sum(r["ms"] for k, r in res.items() if k != "drift_pfl") * 1e-3
    dom = max(("drift", "vlasov"), key=lambda k: res[k]["ms"])
    kern_name = {"drift": "rbg::drift_upfd_kernel", "vlasov": "rbg::vlasov_sym_kernel / rbg::vlasov_upfd_kernel"}[dom]
    line = {"metric": "be_step_phase_space_cells_per_s", "value": cells / t_step, "unit": "cells/s", "n_gpus": 1, "steps": steps,
            "warmup": max(args.warmup, 3), "ms_per_step": t_step * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w["name"] + " [moments + UPFD drift + UPFD Vlasov, NEXT-4]", "cfg": cfg, "nxyz": list(nxyz),
                       "cells": cells, "f_bytes": int(w["f"].nbytes), "l2": "L2 flushed (256 MB write) between timed iterations"},
            "clocks": clocks, "gpu_launches": launches,
            "roofline": {"bound": "hbm", "achieved": res[dom]["achieved_gbs"], "peak": peak, "unit": "GB/s", "frac": res[dom]["frac"],
                         "traffic": res[dom]["traffic"], "traffic_unit": res[dom]["traffic_unit"], "kernel": kern_name,
                         "peak_source": peak_src},
            "kernels": res}
    if e2e:
        # e2e: host buffers in, host buffers out, for the three calls of one step
        f_host = torch.from_numpy(w["f"]).pin_memory()
        o_host = torch.empty_like(f_host).pin_memory()
        t0 = time.perf_counter()
        fd = f_host.cuda(non_blocking=True)
        M, tot, em = col.moments(fd)
        o1 = col.drift_step(fd, 0.01, dx)
        o2 = col.vlasov_step(o1, 0.01, E, B)
        o_host.copy_(o2, non_blocking=True); em_h = em.cpu()
        torch.cuda.synchronize()
        t_e2e = time.perf_counter() - t0
        line["e2e"] = {"value": cells / t_e2e, "unit": "cells/s", "h2d_bytes_per_step": int(w["f"].nbytes),
                       "d2h_bytes_per_step": int(w["f"].nbytes) + int(em.numel() * 8), "ms_per_step": t_e2e * 1e3}
        del f_host, o_host, fd, o1, o2
    if cpu_baseline:
        from oracle import be_steps as bs
        ncell = max(1, min(nx, 8))
        sub = dict(prob, nx=ncell)
        fsub = np.concatenate([w["f"][o:o + ncell * int(np.prod(g["n"]))] for o, g in zip(wl.f_layout(prob)[0], prob["grids"])])
        t0 = time.perf_counter()
        bs.moments(sub, fsub)
        g1 = bs.drift_upfd(sub, fsub, (ncell, 1, 1), 0.01, dx)
        bs.vlasov_upfd(sub, g1, 0.01, E.cpu().numpy()[:ncell], B.cpu().numpy()[:ncell])
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": fsub.size / dt, "unit": "cells/s", "cores": 1, "kind": "oracle",
                                "sample": f"{ncell} of {nx} spatial cells as an {ncell}x1x1 periodic box, every species and momentum cell"}
    del f, out, flush, col, E, B
    torch.cuda.empty_cache()
    return line


# ---- launcher -------------------------------------------------------------------------------------------------------
def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def self_launch(args):
    """`python bench.py --gpus N` with N > 1 outside torchrun: start N ranks (one per GPU) and pass the arguments on."""
    if not args.launch_check:
        import torch
        have = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if have < args.gpus:
            raise SystemExit(f"bench.py: --gpus {args.gpus} requested but only {have} CUDA device(s) are visible; refusing to "
                             f"run fewer ranks than asked for")
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")                  # the communicator lines (nranks, NVLS) go to the log
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    env.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")       # NCCL logs to stdout by default: stdout carries the JSON line only
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()), str(Path(__file__).resolve()), *sys.argv[1:]]
    raise SystemExit(subprocess.run(cmd, env=env).returncode)


def rank_env(args):
    """(rank, world, local_rank) from the torchrun environment; refuses a world size that contradicts --gpus."""
    rank, world, local = (int(os.environ.get(k, d)) for k, d in (("RANK", "0"), ("WORLD_SIZE", "1"), ("LOCAL_RANK", "0")))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}; launch with --nproc-per-node {args.gpus}")
    return rank, world, local


def launch_check(args):
    """--launch-check: the launcher and rank plumbing alone (gloo, no GPU work): every rank reports its environment and
    the spatial cells it would own; rank 0 prints one JSON line.  Used by tests/test_sharding_gloo.py."""
    import torch
    import torch.distributed as dist
    from paper_2308_04869_b200.sharding import cell_range, max_over_ranks
    rank, world, local = rank_env(args)
    if world > 1:
        dist.init_process_group("gloo")
    nx = wl.NOMINAL_NX[args.config] if args.nx is None else args.nx
    lo, hi = cell_range(nx, rank, world) if args.scaling == "strong" else (rank * nx, (rank + 1) * nx)
    mine = torch.tensor([rank, local, lo, hi], dtype=torch.int64)
    rows = [torch.zeros_like(mine) for _ in range(world)]
    if world > 1:
        dist.all_gather(rows, mine)
    else:
        rows = [mine]
    tmax = max_over_ranks(float(rank + 1))                 # the timing reduction: MAX over ranks
    if rank == 0:
        print(json.dumps({"launch_check": True, "n_gpus": world, "scaling": args.scaling, "nx": nx,
                          "ranks": [[int(v) for v in r] for r in rows], "max_over_ranks": tmax,
                          "nccl_debug": os.environ.get("NCCL_DEBUG")}))
    if world > 1:
        dist.destroy_process_group()


# ---- the collision path ----------------------------------------------------------------------------------------------
def time_config(rbg, torch, cfg, args, steps, warmup, rank, world, local, e2e=True):
    """Times one workload on this rank (its shard under strong scaling) and returns the measurements; the caller reduces
    over ranks.  Timed region: `steps` sweeps, each preceded by an L2 flush, CUDA events on the launching stream."""
    from paper_2308_04869_b200.sharding import cell_range, max_over_ranks
    nx_all = wl.NOMINAL_NX[cfg] if args.nx is None else args.nx
    if args.scaling == "strong" and world > 1:
        if nx_all < world:
            raise SystemExit(f"bench.py: config {cfg} has {nx_all} spatial cell(s), fewer than {world} ranks; use --scaling weak")
        w = workloads.make(cfg, nx=args.nx, sampler=args.sampler, cells=cell_range(nx_all, rank, world))
        ix_offset = w["ix_offset"]
    else:
        w = workloads.make(cfg, nx=args.nx, sampler=args.sampler)
        ix_offset = rank * w["problem"]["nx"]              # weak: every rank sweeps one copy at its own global offset
    if args.nx is not None:
        w["name"] += f" [nx overridden to {args.nx}]"
    sym = args.estimator == "symmetric"
    if sym:
        w["name"] += " [conservative estimator]"
        w["dt"] = 0.0
    prob = w["problem"]
    col = rbg.Collision(prob, fp32_kinematics=w["fp32"], ix_offset=ix_offset)
    for kv in args.opt:
        k, v = kv.split("=")
        col.set_option(k, int(v))
    n_evals = col.sample_evals(w["n_samples"])
    f = torch.from_numpy(w["f"]).cuda()
    out = torch.empty_like(f)
    flag = torch.zeros(1, dtype=torch.int32, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2
    stream = torch.cuda.current_stream()

    def step():
        if w["dt"] > 0:
            col.collision_update(f, w["dt"], w["n_samples"], w["seed"], out=out, neg_flag=flag, stream=stream)
        elif sym:
            col.collision_symmetric(f, w["n_samples"], w["seed"], out=out, stream=stream)
        else:
            col.collision(f, w["n_samples"], w["seed"], out=out, stream=stream)

    import torch.distributed as dist
    grouped = dist.is_available() and dist.is_initialized()      # N > 1, or N = 1 with --force-dist

    def barrier():
        if grouped:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warmup):
        step()
    barrier()
    launches_per_step = col.last_launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    with ClockSampler(local) as cs:
        barrier()
        for e0, e1 in ev:
            flush.fill_(1)                     # L2 flush between timed iterations (inputs < L2 for configs 1-3)
            e0.record(stream)
            step()
            e1.record(stream)
        barrier()
    clocks = cs.summary()
    times_ms = [e0.elapsed_time(e1) for e0, e1 in ev]
    t_step = max_over_ranks(sum(times_ms) / len(times_ms)) * 1e-3
    total_evals = n_evals
    if grouped:
        t = torch.tensor([float(n_evals)], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        total_evals = int(t.item())
    res = {"w": w, "t_step": t_step, "n_evals_total": total_evals, "n_evals_rank": n_evals, "launches_per_step": launches_per_step,
           "clocks": clocks, "times_ms": times_ms, "fl_rank": flops_per_sweep(prob, w["n_samples"], w["fp32"])}

    if e2e:
        # the same sweep through the C ABI with HOST buffers (pinned): copies inside the timed region
        f_host = torch.from_numpy(w["f"]).pin_memory()
        c_host = torch.empty_like(f_host).pin_memory()

        def host_call():
            if sym:                              # no host entry point for this one: pinned copies around the device call
                fd = f_host.cuda(non_blocking=True)
                r = col.collision_symmetric(fd, w["n_samples"], w["seed"])
                c_host.copy_(r, non_blocking=True)
                torch.cuda.synchronize()
            elif w["dt"] > 0:
                col.collision_update_host(f_host, w["dt"], w["n_samples"], w["seed"], out=c_host)
            else:
                col.collision_host(f_host, w["n_samples"], w["seed"], out=c_host)
        host_call()                              # warm: allocates scratch
        barrier()
        e2e_steps = max(1, min(steps, 3))
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            host_call()
        res["t_e2e"] = max_over_ranks((time.perf_counter() - t0) / e2e_steps)
        res["same"] = bool(torch.equal(c_host.cuda(), out)) if not sym else None
        res["bytes"] = int(w["f"].nbytes)
        del f_host, c_host
    del f, out, flush, col
    torch.cuda.empty_cache()
    return res


def roofline_of(rbg, torch, res, args, local, probe_cache):
    """ALU roofline of the dominant kernel (every role launch of a sweep is an instance of one template)."""
    w = res["w"]
    t_launch = res["t_step"] / res["launches_per_step"]
    achieved = res["fl_rank"] / res["launches_per_step"] / t_launch / 1e12      # this rank's flops over the max-over-ranks time
    sms = torch.cuda.get_device_properties(local).multi_processor_count
    try:
        max_mhz = float(json.loads((ROOT / "MEASURED_PEAKS.json").read_text()).get("sm_max_mhz", 1965.0))
    except (OSError, ValueError):
        max_mhz = 1965.0
    lanes = FP64_LANES_PER_SM * (2 if w["fp32"] else 1)       # 128 fp32 lanes per SM
    peak_nominal = sms * lanes * 2 * max_mhz * 1e6 / 1e12
    what = 1 if w["fp32"] else 0
    if what not in probe_cache:
        probe_cache[what] = rbg.probe_alu_peak(what, 1 << 17) * 2 / 1e12
    probe = probe_cache[what]
    if "ctx" not in probe_cache:        # operand-pattern context (profiles/r2_collision.md): instructions/s per SM sub-partition-cycle
        probe_cache["ctx"] = {"dfma_3_distinct_operands_tflops": rbg.probe_alu_peak(3, 1 << 16) * 2 / 1e12,
                              "widemul_u32_gops": rbg.probe_alu_peak(4, 1 << 16) / 1e9}
    sym = args.estimator == "symmetric"
    traffic = (None, "not a full-size default run of the standard estimator")
    if args.nx is None and not args.sampler and not sym and not args.opt:
        traffic = ncu_traffic("collision", w["cfg"])
    return {"bound": "alu", "achieved": achieved, "peak": peak_nominal, "unit": "TFLOP/s", "frac": achieved / peak_nominal,
            "traffic": traffic[0], "traffic_unit": traffic[1],
            "peak_source": f"{sms} SM x {lanes} FMA/clk x 2 x {max_mhz:.0f} MHz ({'FP32' if w['fp32'] else 'FP64'} FMA pipe; DESIGN.md section 8)",
            "peak_probe_tflops": probe, "frac_of_probe": achieved / probe, "probe_context": probe_cache["ctx"],
            # FP64 chain: a DFMA whose three operands are distinct registers is limited by register-file operand bandwidth
            # to 2/3 of the lane peak; the fraction of THAT rate is context, `frac` stays the headline
            "frac_of_3_operand_dfma_rate": None if w["fp32"] else achieved / probe_cache["ctx"]["dfma_3_distinct_operands_tflops"],
            "kernel": "rbg::collision_symmetric_kernel" if sym else "rbg::collision_role_kernel", "launch_ms": t_launch * 1e3,
            "flops_per_sample": res["fl_rank"] / res["n_evals_rank"]}


def evolve_measure(rbg, torch, w, n_steps, n_evals_per_step):
    """The paper's collision-dominated run: n Euler steps f <- f + dt C[f] in place, every step a full sweep with its own
    seed (rbg_collision_evolve); wall clock around the call, device synchronised on both sides."""
    col = rbg.Collision(w["problem"], fp32_kinematics=w["fp32"])
    fe = torch.from_numpy(w["f"]).cuda()
    dt_e = w["dt"] if w["dt"] > 0 else 1e-3
    col.collision_evolve(fe, dt_e, 3, w["n_samples"], w["seed"])             # warm-up
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    _, negf = col.collision_evolve(fe, dt_e, n_steps, w["n_samples"], w["seed"])
    torch.cuda.synchronize()
    t_ev = time.perf_counter() - t0
    return {"steps": n_steps, "seconds": t_ev, "ms_per_step": 1e3 * t_ev / n_steps, "dt": dt_e,
            "samples_per_s": n_evals_per_step * n_steps / t_ev,
            "negative_cells_counted": int(negf.item()), "f_finite": bool(torch.isfinite(fe).all())}


def next_block(rbg, torch, args, local, probe_cache):
    """The rows SURVEY.md section 8(f) marks "next", each at full size and timed like the headline (3 warm-up sweeps, L2
    flushed between timed sweeps, CUDA events, clocks sampled during the timed region), so that the driver's own N = 1 run
    carries them: the paper's QGP sweep (workload 7, 70 roles, Table III kinds, inelastic roles), the conservative
    estimator on the headline workload, the t-channel importance sampler on config 2, the paper's own collision test
    (config 6: one Euler step, and 2 500 steps of rbg_collision_evolve), and the moments / drift / Vlasov kernels against
    the HBM roofline on config 4 and on workload 7's odd 11^3 grid."""
    import copy

    def collision(cfg, steps, **over):
        a = copy.copy(args)
        a.nx, a.opt, a.sampler, a.estimator = None, [], 0, "standard"
        for k, v in over.items():
            setattr(a, k, v)
        r = time_config(rbg, torch, cfg, a, steps, 3, 0, 1, local, e2e=False)
        roof = roofline_of(rbg, torch, r, a, local, probe_cache)
        return r, {"workload": r["w"]["name"], "value": r["n_evals_total"] / r["t_step"], "unit": UNIT,
                   "ms_per_step": r["t_step"] * 1e3, "steps": steps, "warmup": 3, "sample_evals_per_sweep": r["n_evals_total"],
                   "gpu_launches_per_step": r["launches_per_step"], "dtype": "f32" if r["w"]["fp32"] else "f64",
                   "roofline": {k: roof[k] for k in ("bound", "achieved", "peak", "unit", "frac", "flops_per_sample", "launch_ms",
                                                     "kernel")},
                   "clocks": r["clocks"]}

    def be(cfg, steps):
        a = copy.copy(args)
        a.nx, a.opt = None, []
        line = measure_be_steps(a, cfg, None, steps, cpu_baseline=False, e2e=False)
        return {"workload": line["config"]["workload"], "cells": line["config"]["cells"], "ms_per_step": line["ms_per_step"],
                "steps": steps, "warmup": line["warmup"], "gpu_launches": line["gpu_launches"], "clocks": line["clocks"],
                "peak_gbs": line["roofline"]["peak"], "peak_source": line["roofline"]["peak_source"],
                "kernels": {k: {kk: v[kk] for kk in ("ms", "achieved_gbs", "frac", "algorithmic_bytes_per_cell")}
                            for k, v in line["kernels"].items() if k != "drift_pfl"}}

    out = {}
    _, out["qgp_workload7_sweep"] = collision(7, 2)
    _, out["conservative_estimator_config4"] = collision(HEADLINE_CONFIG, 2, estimator="symmetric")
    _, out["tchannel_sampler_config2"] = collision(2, 3, sampler=1)
    r6, out["papers_collision_test_config6_euler_step"] = collision(6, 10)
    out["papers_collision_test_config6_evolve"] = evolve_measure(rbg, torch, r6["w"], 2500, r6["n_evals_total"])
    del r6
    out["be_steps_config4"] = be(4, 5)
    out["be_steps_workload7"] = be(7, 5)
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--path", default="collision", choices=["collision", "be"], help="collision: the hot path "
                    "(default); be: the NEXT-4 kernels (moments, UPFD drift, UPFD Vlasov)")
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=HEADLINE_CONFIG, help="BASELINE.json config number (1-5; default 4, the "
                    "largest single-GPU fp64 config); 6, 7 = the paper's own workloads")
    ap.add_argument("--scaling", default="strong", choices=["strong", "weak"], help="N > 1: strong = the workload's spatial "
                    "cells sharded over the ranks (default); weak = one copy of the workload per rank")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-seconds", type=float, default=3.0, help="CPU wall time per step of the reference arm (bounded sample)")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="CPU wall time of the cpu_baseline leg (bounded sample)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-config-block", action="store_true", help="skip the per-config block (configs 1, 2, 3, 5) of the N = 1 line")
    ap.add_argument("--no-next", action="store_true", help="skip the `next` object (SURVEY 8(f) rows: workload 7, conservative "
                    "estimator, t-channel sampler, config 6 step + evolve, moments / drift / Vlasov) of the default N = 1 line")
    ap.add_argument("--block-steps", type=int, default=3, help="timed sweeps per config of the per-config block")
    ap.add_argument("--nx", type=int, default=None, help="override the number of spatial cells (profiling runs; "
                    "the JSON line then names the reduced workload)")
    ap.add_argument("--sampler", type=int, default=0, choices=[0, 1], help="1: t-channel importance sampler on the "
                    "t-channel processes (configs 2, 3, 5); the JSON line then names it")
    ap.add_argument("--estimator", default="standard", choices=["standard", "symmetric"], help="symmetric: the conservative "
                    "estimator rbg_collision_symmetric (NEXT-3); the JSON line then names it")
    ap.add_argument("--opt", action="append", default=[], help="librbg option key=value (launch geometry)")
    ap.add_argument("--evolve-steps", type=int, default=0, help="also time rbg_collision_evolve over this many explicit Euler steps "
                    "in place (the paper's collision test, config 6: 25 000 steps, PAPER.md:469-506) and add an `evolve` object")
    ap.add_argument("--force-dist", action="store_true", help="N = 1: initialise the NCCL process group with one rank and run the "
                    "same barrier / MAX / SUM reductions as N > 1 (exercises the multi-GPU plumbing on one GPU)")
    ap.add_argument("--launch-check", action="store_true", help="launcher / rank plumbing only (gloo, no GPU work)")
    args = ap.parse_args()
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return self_launch(args)
    if args.launch_check:
        return launch_check(args)
    if args.path == "be":
        return run_be_steps(args)

    import torch
    import paper_2308_04869_b200 as rbg

    rank, world, local = rank_env(args)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    if torch.cuda.device_count() <= local:
        raise SystemExit(f"bench.py: rank {rank} needs CUDA device {local}, only {torch.cuda.device_count()} visible")
    torch.cuda.set_device(local)
    grouped = world > 1 or args.force_dist
    json_out = sys.stdout
    if grouped:
        # --force-dist at N = 1: the same NCCL process group, barrier, MAX and SUM reductions as N > 1, with one rank, so
        # that a one-GPU run executes the multi-GPU plumbing (the communicator lines go to stderr)
        import torch.distributed as dist
        os.environ.setdefault("NCCL_DEBUG", "INFO")
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")     # NCCL logs to stdout by default: stdout carries the JSON line only
        if "MASTER_ADDR" not in os.environ:
            os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(free_port()), RANK="0", WORLD_SIZE="1", LOCAL_RANK="0")
        # NCCL writes its version banner (and, without NCCL_DEBUG_FILE, its log) to file descriptor 1.  stdout must carry the one
        # JSON line and nothing else, so for the rest of this process fd 1 points at stderr and the line goes to the saved stdout.
        sys.stdout.flush()
        json_out = os.fdopen(os.dup(1), "w")
        os.dup2(2, 1)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    warmup = max(args.warmup, 3)
    res = time_config(rbg, torch, args.config, args, args.steps, warmup, rank, world, local)
    w = res["w"]
    value = res["n_evals_total"] / res["t_step"]
    probe_cache = {}

    if rank == 0:
        cfgd = config_block(w, args, world)
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warmup,
                "ms_per_step": res["t_step"] * 1e3, "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None,
                "dtype": "f32" if w["fp32"] else "f64", "data": "synthetic", "config": cfgd,
                "workload_detail": {"sample_evals_per_sweep": res["n_evals_total"], "f_bytes_per_rank": res["bytes"],
                                    "nx_per_rank": w["problem"]["nx"], "roles": len(wl.roles(w["problem"]))},
                "clocks": res["clocks"], "gpu_launches": res["launches_per_step"] * args.steps,
                "process_group": f"nccl, {world} rank(s)" if grouped else None,
                "e2e": {"value": res["n_evals_total"] / res["t_e2e"], "unit": UNIT, "h2d_bytes_per_step": res["bytes"] * world,
                        "d2h_bytes_per_step": res["bytes"] * world, "ms_per_step": res["t_e2e"] * 1e3,
                        "matches_device_path": res["same"],
                        "api": ("pinned host -> device copy, rbg_collision_symmetric, device -> pinned host copy" if args.estimator != "standard"
                                else "rbg_collision_update_host (pinned host buffers in and out)" if w["dt"] > 0
                                else "rbg_collision_host (pinned host buffers in and out)")},
                "roofline": roofline_of(rbg, torch, res, args, local, probe_cache)}
        # ---- every other BASELINE config in the same record (N = 1 only) -------------------------------------------
        if (world == 1 and not args.no_config_block and args.config == HEADLINE_CONFIG and args.nx is None and not args.opt
                and args.estimator == "standard" and not args.sampler):
            block = {}
            for cfg in BLOCK_CONFIGS:
                r = time_config(rbg, torch, cfg, args, args.block_steps, 3, 0, 1, local, e2e=False)
                roof = roofline_of(rbg, torch, r, args, local, probe_cache)
                block[str(cfg)] = {"workload": r["w"]["name"], "dtype": "f32" if r["w"]["fp32"] else "f64",
                                   "value": r["n_evals_total"] / r["t_step"], "unit": UNIT, "ms_per_step": r["t_step"] * 1e3,
                                   "steps": args.block_steps, "warmup": 3, "sample_evals_per_sweep": r["n_evals_total"],
                                   "gpu_launches_per_step": r["launches_per_step"],
                                   "roofline": {k: roof[k] for k in ("bound", "achieved", "peak", "unit", "frac", "frac_of_probe",
                                                                     "flops_per_sample", "launch_ms", "traffic")},
                                   "clocks": r["clocks"]}
            line["configs"] = block
            if not args.no_next:
                line["next"] = next_block(rbg, torch, args, local, probe_cache)
        if args.evolve_steps > 0 and world == 1:
            line["evolve"] = evolve_measure(rbg, torch, w, args.evolve_steps, res["n_evals_total"])
        if not args.no_cpu_baseline and world == 1:          # rank 0 at N = 1 only
            cb = oracle_leg(w, args.cpu_seconds)
            cb.pop("seconds")
            line["cpu_baseline"] = cb
        print(json.dumps(line), file=json_out, flush=True)
    if grouped:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
