#!/usr/bin/env python
"""bench.py -- one JSON line for the collision-term hot path (contract: task prompt, section 4).

A "step" is one full collision-term sweep (rbg_collision: every role, spatial cell, momentum cell,
sample) of BASELINE.json configs[1] (e-/H+, screened Coulomb, 8^3 x 20^3 x 2 species, 1024 samples).
  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference]
N > 1: launched by torchrun, one rank per GPU; each rank sweeps its own copy of the workload with a
distinct global cell offset (weak scaling; the path has no collective).
"""
from __future__ import annotations

import argparse
import json
import os
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

# Algorithmic FP64 work per sample of chain O1-O12 (FMA = 2 flops, every other
# add/mul/compare/sqrt/divide = 1), by |M|^2 kind, classical statistics (+12 with quantum factors).
FLOPS_PER_SAMPLE = {0: 141.0, 1: 155.0, 2: 157.0, 3: 142.0,
                    # Table III kinds: 138 (O2-O7, O10-O12) + t 11 + u 2 + T, U 2 + squares 3 + weight 3 + the row's
                    # rational function (5 / 14 / 14 / 5 / 12 / 12 / 16; a reciprocal = 1)
                    4: 164.0, 5: 173.0, 6: 173.0, 7: 164.0, 8: 171.0, 9: 171.0, 10: 175.0}
QUANTUM_EXTRA_FLOPS = 10.0
# the same count for the t-channel importance sampler (steps S1-S7), kinds 1 and 2
FLOPS_PER_SAMPLE_TCHANNEL = {1: 185.0, 2: 187.0}
FP64_LANES_PER_SM = 64          # FMA/clk/SM; confirmed by the live probe
# dram__bytes_read.sum + dram__bytes_write.sum of one role launch from the committed `ncu --set full`
# capture (profiles/r1c_chain_v2_cfg2.md: 32.87 MB + 2.15 MB, config 2 at full size); null elsewhere.
NCU_TRAFFIC_BYTES_PER_LAUNCH = {2: 35.02e6}


def flops_per_sweep(problem, n_samples):
    tot = 0.0
    for r, p in zip(wl.roles(problem), wl.role_processes(problem)):
        q = any(problem["species"][s]["stat"] != 0 for s in r)
        table = FLOPS_PER_SAMPLE_TCHANNEL if p.get("sampler", 0) == 1 else FLOPS_PER_SAMPLE
        per = table[p["kind"]] + (QUANTUM_EXTRA_FLOPS if q else 0.0)
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
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}


def oracle_leg(w, cells, label):
    """Time the oracle, as it stands, on the given spatial cells (host cores of this box)."""
    import oracle
    orc = oracle.Oracle(w["problem"], use_float=w["fp32"])
    per_cell = wl.sample_evals(dict(w["problem"], nx=1), w["n_samples"])
    t0 = time.perf_counter()
    for ix in cells:
        orc.collision(w["f"], w["n_samples"], w["seed"], ix_begin=ix, ix_end=ix + 1)
    dt = time.perf_counter() - t0
    return {"value": per_cell * len(cells) / dt, "unit": UNIT, "cores": oracle.threads(), "kind": "oracle",
            "sample": f"{len(cells)} of {w['problem']['nx']} spatial cells ({label}); every role, momentum cell "
                      f"and sample of those cells", "seconds": dt}


def run_reference(args):
    """--impl reference: the oracle on this box's host cores, same config/metric (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    w = workloads.make(args.config, sampler=args.sampler)
    nx = w["problem"]["nx"]
    ncell = max(1, min(nx, args.ref_cells))
    cells = [int(i) for i in np.linspace(0, nx - 1, ncell).astype(int)]
    import oracle
    oracle.build()
    for _ in range(args.warmup):
        oracle_leg(w, cells[:1], "warm-up")
    times, vals = [], []
    for _ in range(args.steps):
        r = oracle_leg(w, cells, "evenly spaced")
        times.append(r["seconds"]); vals.append(r["value"])
    value = float(np.mean(vals))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(times)), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32" if w["fp32"] else "f64", "data": "synthetic",
            "config": {"workload": w["name"], "cfg": args.config},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"]},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# dram__bytes_read.sum + dram__bytes_write.sum per launch of the NEXT-4 kernels on config 4 at full size, from the committed
# `ncu --set full` captures (profiles/r1d_be_steps_and_qgp.md, captures D and F); null for other workloads.
NCU_TRAFFIC_BE_CFG4 = {"moments": 2.097e9 + 7.1e6, "drift": 2.460e9 + 2.087e9, "vlasov": 2.099e9 + 2.042e9,
                       "drift_pfl": 5.233e9 + 2.083e9}


def run_be_steps(args):
    """--path be: the NEXT-4 kernels (rbg_moments, rbg_drift_step, rbg_vlasov_step) on the chosen config, one JSON line.
    A step = moments + one drift step + one Vlasov step over every phase-space cell.  HBM roofline: algorithmic bytes
    are 8 B per cell for the moments (f read once) and 16 B per cell for each stencil (f read once, f_out written once);
    peak = MEASURED_PEAKS.json hbm_gbs (sustained copy bandwidth), else the profiling guide's fallback 6500 GB/s."""
    import torch
    import paper_2308_04869_b200 as rbg
    if int(os.environ.get("RANK", "0")) != 0:
        return
    torch.cuda.set_device(0)
    w = workloads.make(args.config, nx=args.nx)
    prob = w["problem"]
    nx = prob["nx"]
    side = round(nx ** (1.0 / 3.0))
    nxyz = (side, side, side) if side ** 3 == nx else (nx, 1, 1)
    charges = (-1.0, 1.0, 2.0, 0.5, -0.5, 0.0, 1.5)
    for sp, q in zip(prob["species"], charges):
        if sp.get("charge", 0.0) == 0.0:
            sp["charge"] = q                       # the Vlasov step needs charged species
    col = rbg.Collision(dict(prob, nx=nxyz))
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
    try:
        peaks = json.loads((ROOT / "MEASURED_PEAKS.json").read_text())
        peak, peak_src = float(peaks["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    except (OSError, ValueError, KeyError):
        peak, peak_src = 6500.0, "B200_PROFILING.md fallback"
    res, launches = {}, 0
    with ClockSampler(0) as cs:
        for name, (fn, bytes_per_cell) in kernels.items():
            for _ in range(max(args.warmup, 3)):
                fn()
            torch.cuda.synchronize()
            ts = []
            for _ in range(args.steps):
                flush.fill_(1)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream); fn(); e1.record(stream)
                torch.cuda.synchronize()
                ts.append(e0.elapsed_time(e1))
            launches += col.last_launch_count() * args.steps
            ms = sum(ts) / len(ts)
            gbs = bytes_per_cell * cells / (ms * 1e-3) / 1e9
            res[name] = {"ms": ms, "algorithmic_bytes_per_cell": bytes_per_cell, "achieved_gbs": gbs, "frac": gbs / peak,
                         "traffic": NCU_TRAFFIC_BE_CFG4.get(name) if (args.config == 4 and args.nx is None) else None}
    clocks = cs.summary()
    t_step = sum(r["ms"] for k, r in res.items() if k != "drift_pfl") * 1e-3
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
    dom = max(("drift", "vlasov"), key=lambda k: res[k]["ms"])
    line = {"metric": "be_step_phase_space_cells_per_s", "value": cells / t_step, "unit": "cells/s", "n_gpus": 1, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": t_step * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w["name"] + " [moments + UPFD drift + UPFD Vlasov, NEXT-4]", "cfg": args.config, "nxyz": list(nxyz),
                       "cells": cells, "f_bytes": int(w["f"].nbytes), "l2": "L2 flushed (256 MB write) between timed iterations"},
            "clocks": clocks, "gpu_launches": launches,
            "e2e": {"value": cells / t_e2e, "unit": "cells/s", "h2d_bytes_per_step": int(w["f"].nbytes),
                    "d2h_bytes_per_step": int(w["f"].nbytes) + int(em.numel() * 8), "ms_per_step": t_e2e * 1e3},
            "roofline": {"bound": "hbm", "achieved": res[dom]["achieved_gbs"], "peak": peak, "unit": "GB/s", "frac": res[dom]["frac"],
                         "traffic": res[dom]["traffic"], "kernel": f"rbg::{dom}_upfd_kernel", "peak_source": peak_src},
            "kernels": res}
    if not args.no_cpu_baseline:
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
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--path", default="collision", choices=["collision", "be"], help="collision: the hot path "
                    "(default); be: the NEXT-4 kernels (moments, UPFD drift, UPFD Vlasov)")
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number (1-5); 2 = configs[1]; 6, 7 = the paper's own workloads")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-cells", type=int, default=6, help="spatial cells per step of the reference arm")
    ap.add_argument("--cpu-cells", type=int, default=48, help="spatial cells of the cpu_baseline leg")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--nx", type=int, default=None, help="override the number of spatial cells (profiling runs; "
                    "the JSON line then names the reduced workload)")
    ap.add_argument("--sampler", type=int, default=0, choices=[0, 1], help="1: t-channel importance sampler on the "
                    "t-channel processes (configs 2, 3, 5); the JSON line then names it")
    ap.add_argument("--estimator", default="standard", choices=["standard", "symmetric"], help="symmetric: the conservative "
                    "estimator rbg_collision_symmetric (NEXT-3); the JSON line then names it")
    ap.add_argument("--opt", action="append", default=[], help="librbg option key=value (launch geometry)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.path == "be":
        return run_be_steps(args)

    import torch
    import torch.distributed as dist
    import paper_2308_04869_b200 as rbg
    from paper_2308_04869_b200.sharding import max_over_ranks

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    w = workloads.make(args.config, nx=args.nx, sampler=args.sampler)
    if args.nx is not None:
        w["name"] += f" [nx overridden to {args.nx}]"
    sym = args.estimator == "symmetric"
    if sym:
        w["name"] += " [conservative (symmetric) estimator]"
        w["dt"] = 0.0
    prob = w["problem"]
    # weak scaling: every rank sweeps one copy of the workload; rank r holds global cells [r*Nx, (r+1)*Nx)
    col = rbg.Collision(prob, fp32_kinematics=w["fp32"], ix_offset=rank * prob["nx"])
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

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    launches_per_step = col.last_launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
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
    value = world * n_evals / t_step

    # ---- e2e: the same sweep through the C ABI with HOST buffers (pinned), copies inside the timing
    f_host = torch.from_numpy(w["f"]).pin_memory()
    c_host = torch.empty_like(f_host).pin_memory()
    def host_call():
        if sym:                                  # no host entry point for this estimator: pinned copies around the device call
            fd = f_host.cuda(non_blocking=True)
            c_host.copy_(col.collision_symmetric(fd, w["n_samples"], w["seed"]), non_blocking=True)
            torch.cuda.synchronize()
        else:
            col.collision_host(f_host, w["n_samples"], w["seed"], out=c_host)
    host_call()                                  # warm: allocates scratch
    barrier()
    e2e_steps = max(1, min(args.steps, 3))
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        host_call()
    t_e2e = max_over_ranks((time.perf_counter() - t0) / e2e_steps)
    same = bool(torch.equal(c_host.cuda(), out)) if (w["dt"] == 0 and not sym) else None

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (all role launches are the same template here) ---------
    fl = flops_per_sweep(prob, w["n_samples"])
    t_launch = t_step / launches_per_step
    achieved = fl / launches_per_step / t_launch / 1e12
    sms = torch.cuda.get_device_properties(local).multi_processor_count
    try:
        peaks = json.loads((ROOT / "MEASURED_PEAKS.json").read_text())
        max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    except (OSError, ValueError):
        max_mhz = 1965.0
    peak_nominal = sms * FP64_LANES_PER_SM * 2 * max_mhz * 1e6 / 1e12
    probe = rbg.probe_alu_peak(0 if not w["fp32"] else 1, 1 << 17) * 2 / 1e12
    if w["fp32"]:
        peak_nominal *= 2                       # 128 fp32 lanes per SM
    roof = {"bound": "alu", "achieved": achieved, "peak": peak_nominal, "unit": "TFLOP/s", "frac": achieved / peak_nominal,
            "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH.get(args.config) if args.nx is None and not args.sampler and not sym else None,
            "traffic_unit": "bytes per launch (ncu capture, profiles/r1c_chain_v2_cfg2.md)", "peak_source": f"{sms} SM x {FP64_LANES_PER_SM * (2 if w['fp32'] else 1)} FMA/clk x 2 x "
                                            f"{max_mhz:.0f} MHz (DESIGN.md section 8)",
            "peak_probe_tflops": probe, "frac_of_probe": achieved / probe,
            "kernel": "rbg::collision_symmetric_kernel" if sym else "rbg::collision_role_kernel", "launch_ms": t_launch * 1e3,
            "flops_per_sample": fl / n_evals}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": t_step * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if w["fp32"] else "f64", "data": "synthetic",
            "config": {"workload": w["name"], "cfg": args.config, "nx": prob["nx"], "n_samples": w["n_samples"],
                       "sample_evals_per_sweep": n_evals, "f_bytes": int(w["f"].nbytes),
                       "l2": "L2 flushed (256 MB write) between timed iterations", "parallelism": f"spatial-shard x{world}"},
            "clocks": clocks, "gpu_launches": launches_per_step * args.steps,
            "e2e": {"value": world * n_evals / t_e2e, "unit": UNIT, "h2d_bytes_per_step": int(w["f"].nbytes),
                    "d2h_bytes_per_step": int(w["f"].nbytes), "ms_per_step": t_e2e * 1e3, "matches_device_path": same},
            "roofline": roof}
    if not args.no_cpu_baseline:
        import oracle
        oracle.build()
        nx = prob["nx"]
        cells = [int(i) for i in np.linspace(0, nx - 1, max(1, min(nx, args.cpu_cells))).astype(int)]
        cb = oracle_leg(w, cells, "evenly spaced")
        cb.pop("seconds")
        line["cpu_baseline"] = cb
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
