"""Smallest cases that reach every kernel family, for `compute-sanitizer` (one tool per run):

    compute-sanitizer --tool memcheck  python tests/sanitizer_cases.py
    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py
    compute-sanitizer --tool synccheck python tests/sanitizer_cases.py
    compute-sanitizer --tool initcheck python tests/sanitizer_cases.py

and, where compute-sanitizer is not available (it is closed on the pool this repo is developed on, profiles/r2_sanitizers.md),
with the library's own device-side checks:

    python tests/sanitizer_cases.py --checked      # librbg_checked.so; prints the eight failure counters, all must be 0

Not a pytest module (correctness against the oracle is tests/test_gpu_*.py); it only drives the CUDA path through the C ABI
so that the tool sees every staging / synchronisation pattern: TMA bulk copy + mbarrier, cooperative staging, global (L2)
gathers, the fused update, shared-memory and global atomics of the conservative estimator with its CTA-end flush, the
mbarrier stage ring of the persistent moments / Vlasov kernels under slot reuse, and the drift stencils.  Prints one line
per case and exits 0; the tool's summary line ("ERROR SUMMARY: 0 errors" / "RACECHECK SUMMARY: 0 hazards") is the result.
"""
import sys
from pathlib import Path

import numpy as np
import torch

sys.path.insert(0, str(Path(__file__).resolve().parent.parent))

import paper_2308_04869_b200 as rbg  # noqa: E402
import workloads  # noqa: E402


def _finite(t, what):
    torch.cuda.synchronize()
    assert bool(torch.isfinite(t).all()), what
    print(f"ok  {what}", flush=True)


def collision_cases():
    for what, cfg, kw, fp32, opts in (
            ("collision: TMA-staged tables (8^3, 16-byte multiples), 2 species", 2, dict(nx=2, np_side=8, n_samples=40), False, ()),
            ("collision: cooperative staging (7^3 tables, odd byte counts)", 2, dict(nx=2, np_side=7, n_samples=33), False, ()),
            ("collision: global (L2) gathers forced", 2, dict(nx=2, np_side=8, n_samples=40), False, (("gather", 2),)),
            ("collision: 35^3 tables do not fit shared memory (the paper's grid)", 6, dict(nx=1, n_samples=2), False, ()),
            ("collision: fp32 kinematics, cooperative float staging", 2, dict(nx=2, np_side=8, n_samples=40), True, ()),
            ("collision: quantum statistics, t-channel kind, 5 species", 3, dict(nx=1, np_side=6, n_samples=32), False, ()),
            ("collision: Table III kinds with inelastic roles (three tables)", 7, dict(nx=2, np_side=4, n_samples=16), False, ()),
            ("collision: 2 samples per lane, 12 warps", 4, dict(nx=2, np_side=8, n_samples=70), False, (("samples_per_lane", 2),)),
            ("collision: 1 sample per lane, 32 warps", 4, dict(nx=2, np_side=8, n_samples=70), False, (("warps_per_cta", 32),)),
            ("collision: t-channel importance sampler", 2, dict(nx=2, np_side=8, n_samples=40, sampler=1), False, ())):
        w = workloads.make(cfg, **kw)
        col = rbg.Collision(w["problem"], fp32_kinematics=fp32)
        for k, v in opts:
            col.set_option(k, v)
        f = torch.from_numpy(w["f"]).cuda()
        _finite(col.collision(f, w["n_samples"], w["seed"]), what)
        out, flag = col.collision_update(f, 1e-3, w["n_samples"], w["seed"])
        _finite(out, what + " [fused update]")


def symmetric_cases():
    for what, cfg, kw, tables in (
            ("conservative estimator: global atomics (default)", 2, dict(nx=2, np_side=8, n_samples=40), 0),
            ("conservative estimator: shared-memory accumulators (red.shared + CTA-end flush)", 2, dict(nx=2, np_side=8, n_samples=40), 1),
            ("conservative estimator: inelastic roles", 7, dict(nx=2, np_side=4, n_samples=16), 0),
            ("conservative estimator: inelastic roles, shared-memory accumulators", 7, dict(nx=2, np_side=4, n_samples=16), 1),
            ("conservative estimator: 31^3 tables do not fit, global atomics although tables were asked for", 6, dict(nx=1, np_side=31, n_samples=2), 1)):
        w = workloads.make(cfg, **kw)
        col = rbg.Collision(w["problem"])
        col.set_option("sym_tables", tables)
        _finite(col.collision_symmetric(torch.from_numpy(w["f"]).cuda(), w["n_samples"], w["seed"]), what)


def be_step_cases():
    rng = np.random.default_rng(3)
    for what, cfg, kw, nxyz in (
            # 20^3: one cell per stage, two stages per CTA: 600 cells over 148 CTAs reuse every slot twice
            ("moments / Vlasov: stage ring with slot reuse, one 64 KB cell per stage", 2, dict(np_side=20), (600, 1, 1)),
            # 11^3 (odd cell count): groups of several cells per stage, leading single cell, 7 species
            ("moments / Vlasov: grouped stages, odd momentum-cell count", 7, dict(np_side=11), (10, 10, 9)),
            ("moments / Vlasov: 35^3 blocks (direct kernels)", 6, dict(), (2, 1, 1)),
            ("moments / Vlasov: tiny momentum grid", 1, dict(np_side=2), (37, 1, 1))):
        nx = int(np.prod(nxyz))
        w = workloads.make(cfg, nx=nx, **kw)
        prob = w["problem"]
        for i, sp in enumerate(prob["species"]):
            sp["charge"] = (-1.0, 1.0, 2.0, 0.5, -0.5, 1.5, -2.0)[i % 7]
        col = rbg.Collision(dict(prob, nx=nxyz))
        f = torch.from_numpy(w["f"]).cuda()
        M, tot, em = col.moments(f)
        _finite(M, what + " [moments]")
        # the general staged kernel as well where the symmetric-grid kernel (three stages, two teams) was taken above
        col.set_option("moments_path", 1)
        M, tot, em = col.moments(f)
        _finite(M, what + " [moments, general staged kernel]")
        col.set_option("moments_path", 0)
        E = torch.from_numpy(rng.normal(size=(nx, 3))).cuda()
        B = torch.from_numpy(rng.normal(size=(nx, 3))).cuda()
        _finite(col.vlasov_step(f, 0.01, E, B), what + " [vlasov]")
        col.set_option("vlasov_path", 1)
        _finite(col.vlasov_step(f, 0.01, E, B), what + " [vlasov, general staged kernel]")
        col.set_option("vlasov_path", 0)
    for what, cfg, kw, nxyz, bc, zeta in (("drift: periodic", 2, dict(np_side=8), (5, 4, 3), (1, 1, 1), 0.0),
                                          ("drift: reflecting and absorbing walls", 7, dict(np_side=5), (3, 6, 4), (0, 1, 0), 0.6)):
        nx = int(np.prod(nxyz))
        w = workloads.make(cfg, nx=nx, **kw)
        col = rbg.Collision(dict(w["problem"], nx=nxyz))
        f = torch.from_numpy(w["f"]).cuda()
        _finite(col.drift_step(f, 0.02, (0.5, 0.8, 0.3), bc=bc, zeta=zeta), what + " [first order]")
        _finite(col.drift_step_pfl(f, 0.02, (0.5, 0.8, 0.3)), what + " [second order, periodic]")
    w = workloads.make(2, nx=12, np_side=8, n_samples=24)
    col = rbg.Collision(dict(w["problem"], nx=(3, 2, 2)))
    f = torch.from_numpy(w["f"]).cuda()
    E = torch.ones((12, 3), dtype=torch.float64, device="cuda")
    for mode in (True, "symmetric"):
        col.be_step(f, 0.002, dx=(0.5, 0.5, 0.5), E=E, B=E, n_samples=24, seed=5, collision=mode)
        _finite(f, f"rbg_be_step, collision={mode}")


if __name__ == "__main__":
    checked = "--checked" in sys.argv
    if checked:
        from paper_2308_04869_b200.build import build
        build(checked=True)
        rbg.use_checked_build()
    torch.cuda.set_device(0)
    collision_cases()
    symmetric_cases()
    be_step_cases()
    print("all sanitizer cases ran")
    if checked:
        counts = rbg.selfcheck_failures()
        names = ("f-table index", "tile index", "direction-table index", "output index", "shared-memory layout",
                 "ring-slot contents", "stencil / moment index", "conservative-estimator index")
        for n, c in zip(names, counts):
            print(f"checked build: {n}: {c} failures")
        assert not any(counts), counts
        print("CHECKED BUILD SUMMARY: 0 failures")
