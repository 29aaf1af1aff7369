"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element on the same
seeded inputs.  Bar (north_star): |C_gpu - C_oracle| <= 1e-10 (|gain| + |loss|) per cell in fp64;
1e-4 of the same scale for the fp32-kinematics variant against the oracle's float chain."""
import numpy as np
import pytest
import torch

import oracle
import workloads

pytestmark = pytest.mark.gpu

TOL64 = 1e-10
TOL32 = 1e-4


def _rbg():
    import paper_2308_04869_b200 as rbg
    return rbg


def oracle_C_and_scale(orc, f, n_samples, seed, **kw):
    """Oracle C and the per-cell tolerance scale sum_roles (|G| + |L|).  With ix_begin / ix_end / ix_stride only the
    visited spatial cells are touched (the detail arrays of a full-size problem are gigabytes of untouched zeros)."""
    C_ref, d = orc.collision(f, n_samples, seed, detail=True, **kw)
    mag = np.zeros_like(C_ref)
    cells = range(kw.get("ix_begin", 0), kw.get("ix_end", None) or orc.nx, kw.get("ix_stride", 1))
    for r in range(orc.n_roles):
        s1 = orc.roles[r]["s"][0]
        n = orc.np[s1]
        if len(cells) == orc.nx:
            sl_c, sl_d = slice(orc.sp_off[s1], orc.sp_off[s1] + orc.nx * n), slice(orc.role_off[r], orc.role_off[r] + orc.nx * n)
            mag[sl_c] += np.abs(d["G"][sl_d]) + np.abs(d["L"][sl_d])
            continue
        for ix in cells:
            sl_c = slice(orc.sp_off[s1] + ix * n, orc.sp_off[s1] + (ix + 1) * n)
            sl_d = slice(orc.role_off[r] + ix * n, orc.role_off[r] + (ix + 1) * n)
            mag[sl_c] += np.abs(d["G"][sl_d]) + np.abs(d["L"][sl_d])
    return C_ref, mag


def gpu_C(problem, f, n_samples, seed, fp32=False, options=(), ix_offset=0):
    rbg = _rbg()
    col = rbg.Collision(problem, fp32_kinematics=fp32, ix_offset=ix_offset)
    for k, v in options:
        col.set_option(k, v)
    ft = torch.from_numpy(np.ascontiguousarray(f)).cuda()
    C = col.collision(ft, n_samples, seed)
    torch.cuda.synchronize()
    return C.cpu().numpy(), col


def assert_parity(C, C_ref, mag, tol, what):
    err = np.abs(C - C_ref)
    bad = err > tol * mag
    worst = np.max(err / np.maximum(mag, 1e-300))
    assert not bad.any(), f"{what}: {bad.sum()} cells off, worst err/(G+L) = {worst:.3e}"
    assert np.any(C_ref != 0), what


CASES = [
    # (config, overrides): sizes the oracle finishes in seconds that still span several p1 tiles,
    # ragged tile tails, sample counts that are not a multiple of the warp size, odd grid sizes
    # (7^3 = 343 cells: table size not a multiple of 16 bytes -> non-TMA staging path)
    (1, dict()),                                             # BASELINE configs[0] at full size
    (1, dict(nx=3, np_side=7, n_samples=100)),
    (2, dict(nx=3, np_side=20, n_samples=64)),
    (2, dict(nx=2, np_side=7, n_samples=33)),
    (3, dict(nx=2, np_side=8, n_samples=96)),
    (3, dict(nx=1, np_side=20, n_samples=16)),
    (4, dict(nx=5, np_side=20, n_samples=100)),
    (6, dict(nx=2, np_side=9, n_samples=64)),               # kind ISO_DSIGMA (the paper's collision test)
    (6, dict(n_samples=16)),                                # 35^3 tables (343 KB each): global/L2 gather path
]


@pytest.mark.parametrize("cfg,kw", CASES)
def test_parity_fp64(cfg, kw):
    w = workloads.make(cfg, **kw)
    orc = oracle.Oracle(w["problem"])
    C_ref, mag = oracle_C_and_scale(orc, w["f"], w["n_samples"], w["seed"])
    C, col = gpu_C(w["problem"], w["f"], w["n_samples"], w["seed"])
    assert_parity(C, C_ref, mag, TOL64, f"cfg{cfg} {kw}")
    assert col.last_launch_count() == orc.n_roles
    assert col.sample_evals(w["n_samples"]) == workloads.configs.sample_evals(w["problem"], w["n_samples"])


@pytest.mark.parametrize("cfg,kw", [(1, dict(nx=2, np_side=8, n_samples=128)), (2, dict(nx=2, np_side=10, n_samples=64)),
                                    (3, dict(nx=1, np_side=8, n_samples=64)), (6, dict(nx=1, np_side=10, n_samples=64))])
def test_parity_fp32_kinematics(cfg, kw):
    w = workloads.make(cfg, **kw)
    orc = oracle.Oracle(w["problem"], use_float=True)
    C_ref, mag = oracle_C_and_scale(orc, w["f"], w["n_samples"], w["seed"])
    C, _ = gpu_C(w["problem"], w["f"], w["n_samples"], w["seed"], fp32=True)
    assert_parity(C, C_ref, mag, TOL32, f"fp32 cfg{cfg}")


def test_result_independent_of_launch_geometry_and_gather_path():
    """Determinism contract of include/rbg.h: each p1 is reduced by one warp in a fixed lane order, so
    the result is bit-identical for any tile size, CTA size and gather path."""
    w = workloads.make(2, nx=2, np_side=12, n_samples=80)
    base, _ = gpu_C(w["problem"], w["f"], w["n_samples"], w["seed"])
    for opts in ([("warps_per_cta", 3), ("p1_per_cta", 5)], [("warps_per_cta", 8), ("p1_per_cta", 1000)],
                 [("gather", 2)], [("gather", 2), ("warps_per_cta", 1), ("p1_per_cta", 1)],
                 [("samples_per_lane", 1)], [("warps_per_cta", 32)], [("samples_per_lane", 1), ("gather", 2), ("warps_per_cta", 5)]):
        other, _ = gpu_C(w["problem"], w["f"], w["n_samples"], w["seed"], options=opts)
        assert np.array_equal(base, other), opts
    # more than two 32-sample blocks per lane, a ragged last block, fp32 kinematics: the lane sums must not depend on SPL
    for fp32, N in ((False, 200), (True, 333)):
        base, _ = gpu_C(w["problem"], w["f"], N, 9, fp32=fp32)
        for opts in ([("samples_per_lane", 1)], [("warps_per_cta", 32)], [("samples_per_lane", 2), ("warps_per_cta", 7)]):
            other, _ = gpu_C(w["problem"], w["f"], N, 9, fp32=fp32, options=opts)
            assert np.array_equal(base, other), (fp32, N, opts)


def test_spatial_sharding_reproduces_the_single_device_result():
    """Section 8(e): spatial cells are independent; the stream is keyed by the global cell index."""
    w = workloads.make(2, nx=5, np_side=8, n_samples=48)
    full, _ = gpu_C(w["problem"], w["f"], w["n_samples"], w["seed"])
    offs, total = workloads.f_layout(w["problem"])
    for lo, hi in ((0, 2), (2, 5)):
        prob = dict(w["problem"], nx=hi - lo)
        parts_in, parts_ref = [], []
        for s, g in enumerate(w["problem"]["grids"]):
            npc = int(np.prod(g["n"]))
            blk = w["f"][offs[s]:offs[s] + 5 * npc].reshape(5, npc)
            parts_in.append(blk[lo:hi].reshape(-1))
            parts_ref.append(full[offs[s]:offs[s] + 5 * npc].reshape(5, npc)[lo:hi].reshape(-1))
        shard, _ = gpu_C(prob, np.concatenate(parts_in), w["n_samples"], w["seed"], ix_offset=lo)
        assert np.array_equal(shard, np.concatenate(parts_ref))


@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs two CUDA devices")
def test_two_device_shards_concatenate_to_the_single_device_result():
    """What `bench.py --gpus 2` does, in one process: each device holds half of the spatial cells (workloads.make(cells=...)),
    the handle is created on that device with the shard's global offset; the pieces concatenate bit-identically.  Also
    exercises the device guard: the second handle is called while device 0 is current."""
    rbg = _rbg()
    from paper_2308_04869_b200 import sharding
    w = workloads.make(2, nx=6, np_side=8, n_samples=48)
    full, _ = gpu_C(w["problem"], w["f"], w["n_samples"], w["seed"])
    pieces = []
    for r in range(2):
        ws = workloads.make(2, nx=6, np_side=8, n_samples=48, cells=sharding.cell_range(6, r, 2))
        with torch.cuda.device(r):
            col = rbg.Collision(ws["problem"], ix_offset=ws["ix_offset"])
            ft = torch.from_numpy(ws["f"]).cuda()
        torch.cuda.set_device(0)
        C = col.collision(ft, ws["n_samples"], ws["seed"], stream=torch.cuda.current_stream(r))
        torch.cuda.synchronize(r)
        pieces.append(C.cpu().numpy())
    assert np.array_equal(sharding.unshard(w["problem"], pieces), full)


def test_fused_update_and_negativity_flag():
    """rbg_collision_update: f_out = f + dt*C (Eq. 27) and the count of negative cells."""
    rbg = _rbg()
    w = workloads.make(2, nx=2, np_side=8, n_samples=64)
    orc = oracle.Oracle(w["problem"])
    C_ref, mag = oracle_C_and_scale(orc, w["f"], w["n_samples"], w["seed"])
    col = rbg.Collision(w["problem"])
    f = torch.from_numpy(w["f"]).cuda()
    for dt in (1e-3, 5e3):                      # the large step drives some cells negative
        ref, neg_ref = oracle.update(w["f"], C_ref, dt)
        out, flag = col.collision_update(f, dt, w["n_samples"], w["seed"])
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        assert np.all(np.abs(got - ref) <= dt * TOL64 * mag + 4 * np.finfo(float).eps * np.abs(ref))
        margin = dt * TOL64 * mag + 4 * np.finfo(float).eps * np.abs(ref)
        sure_neg = int(np.sum(ref < -margin)); maybe_neg = int(np.sum(ref < margin))
        assert sure_neg <= int(flag.item()) <= maybe_neg
        assert int(flag.item()) == int(np.sum(got < 0))
        if dt > 1:
            assert neg_ref > 0 and flag.item() > 0
        else:
            assert flag.item() == 0
    # the flag accumulates (caller zeroes it)
    out, flag2 = col.collision_update(f, 5e3, w["n_samples"], w["seed"], neg_flag=flag.clone())
    torch.cuda.synchronize()
    assert flag2.item() == 2 * flag.item()
    with pytest.raises(rbg.RbgError):
        col.collision_update(f, 1e-3, 8, 1, out=f)          # f_out must not alias f


def test_outputs_that_overlap_f_partly_are_refused():
    """include/rbg.h, "Overlap": the byte ranges are compared, so an output that starts inside f (or ends inside it) is an
    error just like out == f; buffers that merely touch are fine."""
    rbg = _rbg()
    w = workloads.make(1, nx=2, np_side=6, n_samples=8)
    col = rbg.Collision(w["problem"])
    n = col.f_elems
    buf = torch.zeros(3 * n, dtype=torch.float64, device="cuda")
    buf[n:2 * n] = torch.from_numpy(w["f"]).cuda()
    f = buf[n:2 * n]
    for lo in (n - 1, n + 1, 1, 2 * n - 1):                 # ends one element inside f / starts one element inside f / ...
        out = buf[lo:lo + n]
        for call in (lambda: col.collision(f, 8, 1, out=out), lambda: col.collision_update(f, 1e-3, 8, 1, out=out),
                     lambda: col.collision_symmetric(f, 8, 1, out=out), lambda: col.collision_evolve(f, 1e-3, 1, 8, 1, scratch=out)):
            with pytest.raises(rbg.RbgError, match="overlaps"):
                call()
    ref = col.collision(f, 8, 1).clone()
    for lo in (0, 2 * n):                                   # adjacent, not overlapping
        assert torch.equal(col.collision(f, 8, 1, out=buf[lo:lo + n]), ref)
    host = np.zeros(2 * n)
    with pytest.raises(rbg.RbgError, match="overlaps"):
        col.collision_host(host[:n], 8, 1, out=host[n - 1:2 * n - 1])


def test_host_entry_point_matches_device_entry_point():
    w = workloads.make(1, nx=2, np_side=8, n_samples=64)
    C_dev, col = gpu_C(w["problem"], w["f"], w["n_samples"], w["seed"])
    C_host = col.collision_host(w["f"], w["n_samples"], w["seed"])
    assert np.array_equal(C_dev, C_host)
    pinned = torch.from_numpy(w["f"]).pin_memory()
    assert np.array_equal(col.collision_host(pinned, w["n_samples"], w["seed"]).numpy(), C_dev)


def test_update_host_entry_point_matches_the_device_update():
    """rbg_collision_update_host = rbg_collision_update with host buffers: same bits, and the count of negative cells is set
    (not accumulated).  Two species, fp32 kinematics and fp64; a step large enough to drive cells negative; then a problem
    above 128 MB so that the sweep is pipelined over two chunks and the count sums over them."""
    rbg = _rbg()
    for fp32 in (False, True):
        w = workloads.make(2, nx=3, np_side=8, n_samples=32)
        col = rbg.Collision(w["problem"], fp32_kinematics=fp32)
        f = torch.from_numpy(w["f"]).cuda()
        for dt in (1e-3, 5e4):
            ref, flag = col.collision_update(f, dt, w["n_samples"], w["seed"])
            torch.cuda.synchronize()
            for _ in range(2):                                   # twice: the count must not accumulate
                out, neg = col.collision_update_host(w["f"], dt, w["n_samples"], w["seed"])
                assert np.array_equal(out, ref.cpu().numpy())
                assert neg == int(flag.item()) == int(np.sum(out < 0))
        assert neg > 0
    w = workloads.make(2, nx=1201, np_side=20, n_samples=4)
    assert w["f"].nbytes > (128 << 20)
    col = rbg.Collision(w["problem"])
    ref, flag = col.collision_update(torch.from_numpy(w["f"]).cuda(), 3e4, w["n_samples"], w["seed"])
    out, neg = col.collision_update_host(torch.from_numpy(w["f"]).pin_memory(), 3e4, w["n_samples"], w["seed"])
    assert torch.equal(out, ref.cpu()) and neg == int(flag.item()) and neg > 0
    with pytest.raises(rbg.RbgError, match="overlaps"):
        buf = np.zeros(2 * col.f_elems)
        col.collision_update_host(buf[:col.f_elems], 1e-3, 4, 1, out=buf[1:col.f_elems + 1])


def test_host_entry_point_pipelined_over_cell_chunks_is_bit_identical():
    """rbg_collision_host pipelines copy-in / kernels / copy-out over chunks of spatial cells once f exceeds 128 MB
    (include/rbg.h); two species so that every chunk is two H2D copies, an odd cell count so that the chunks are unequal.
    The sample stream is keyed by the global cell index, so the result must equal the one-launch device path bit for bit."""
    w = workloads.make(2, nx=1201, np_side=20, n_samples=8)           # 2 x 1201 x 8000 doubles = 154 MB -> 2 chunks
    assert w["f"].nbytes > (128 << 20)
    C_dev, col = gpu_C(w["problem"], w["f"], w["n_samples"], w["seed"])
    n_device_launches = col.last_launch_count()
    pinned = torch.from_numpy(w["f"]).pin_memory()
    C_host = col.collision_host(pinned, w["n_samples"], w["seed"]).numpy()
    assert col.last_launch_count() == 2 * n_device_launches            # two chunks, every role in each
    assert np.array_equal(C_host, C_dev)


def test_edge_cases():
    rbg = _rbg()
    # single sample; fewer samples than lanes; one momentum cell; a species that takes part in no process
    w = workloads.make(2, nx=1, np_side=4, n_samples=1)
    for N in (1, 5, 31, 32, 33):
        orc = oracle.Oracle(w["problem"])
        C_ref, mag = oracle_C_and_scale(orc, w["f"], N, 77)
        C, _ = gpu_C(w["problem"], w["f"], N, 77)
        assert_parity(C, C_ref, mag, TOL64, f"N={N}")
    prob = dict(w["problem"], processes=[w["problem"]["processes"][0]])      # only e-e: H+ has no role
    orc = oracle.Oracle(prob)
    C_ref, mag = oracle_C_and_scale(orc, w["f"], 16, 3)
    C, col = gpu_C(prob, w["f"], 16, 3)
    assert_parity(C, C_ref, mag, TOL64, "idle species")
    assert np.all(C[orc.sp_off[1]:] == 0)
    out, flag = col.collision_update(torch.from_numpy(w["f"]).cuda(), 1e-3, 16, 3)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy()[orc.sp_off[1]:], w["f"][orc.sp_off[1]:])
    # one-cell momentum grid and no processes at all
    one = dict(nx=2, species=[dict(mass=1.0, charge=0, stat=0, g=1.0)],
               grids=[dict(n=[1, 1, 1], pmin=[-1.0] * 3, pmax=[1.0] * 3)],
               processes=[dict(a=0, b=0, c=0, d=0, kind=0, par=[1.0], sym=-1.0)], hbar=1.0)
    f1 = np.array([0.5, 0.25])
    orc = oracle.Oracle(one)
    C_ref, mag = oracle_C_and_scale(orc, f1, 64, 1)
    C, _ = gpu_C(one, f1, 64, 1)
    assert_parity(C, C_ref, mag, TOL64, "1-cell grid")
    none = dict(one, processes=[])
    C, col = gpu_C(none, f1, 64, 1)
    assert np.all(C == 0) and col.n_roles == 0
    # massless species (T = q/(E+0), h > 0 guard)
    w0 = workloads.make(3, nx=1, np_side=6, n_samples=40)
    w0["problem"]["species"][3]["mass"] = 0.0
    orc = oracle.Oracle(w0["problem"])
    C_ref, mag = oracle_C_and_scale(orc, w0["f"], 40, 5)
    C, _ = gpu_C(w0["problem"], w0["f"], 40, 5)
    assert_parity(C, C_ref, mag, TOL64, "massless")
    assert np.all(np.isfinite(C))
    # a massless species with a cell centre at p = 0 (odd grid, symmetric box): 1/p0 of Eq. 16 diverges -> refused, as the
    # oracle refuses it; with a mass, or when the species takes part in no process, the same grid is accepted
    w1 = workloads.make(3, nx=1, np_side=7, n_samples=8)
    w1["problem"]["species"][3]["mass"] = 0.0
    with pytest.raises(rbg.RbgError, match="zero energy"):
        rbg.Collision(w1["problem"])
    with pytest.raises(ValueError):
        oracle.Oracle(w1["problem"])
    idle = dict(w1["problem"], processes=[p for p in w1["problem"]["processes"] if 3 not in (p["a"], p["b"])])
    assert rbg.Collision(idle).n_roles == oracle.Oracle(idle).n_roles
    w1["problem"]["species"][3]["mass"] = 0.01
    f1 = np.nan_to_num(w1["f"], nan=0.1)             # the generator's anisotropy factor p_z/|p| is 0/0 at the centre cell
    orc = oracle.Oracle(w1["problem"])
    C_ref, mag = oracle_C_and_scale(orc, f1, 8, 5)
    C, _ = gpu_C(w1["problem"], f1, 8, 5)
    assert np.all(np.isfinite(C))
    assert_parity(C, C_ref, mag, TOL64, "odd grid, light species")


def test_hbar_enters_the_prefactor_squared_and_the_occupation_number():
    """Eq. 16: hbar^2 c |M|^2 / (64 pi^2 ...); Eq. 18: nbar = (2 pi hbar)^3 f / g.  Parity at hbar != 1 for a
    quantum problem, and C(hbar) = hbar^2 C(1) exactly (a power of two) for a classical one."""
    w = workloads.make(3, nx=2, np_side=8, n_samples=64)
    prob = dict(w["problem"], hbar=0.25)
    orc = oracle.Oracle(prob)
    C_ref, mag = oracle_C_and_scale(orc, w["f"], 64, 11)
    C, _ = gpu_C(prob, w["f"], 64, 11)
    assert_parity(C, C_ref, mag, TOL64, "hbar = 0.25, quantum")
    w = workloads.make(1, nx=2, np_side=8, n_samples=64)
    C1, _ = gpu_C(w["problem"], w["f"], 64, 11)
    Ch, _ = gpu_C(dict(w["problem"], hbar=0.25), w["f"], 64, 11)
    assert np.array_equal(Ch, 0.0625 * C1) and np.any(C1 != 0)


def test_argument_errors():
    rbg = _rbg()
    w = workloads.make(1, np_side=4)
    P = w["problem"]
    bads = [dict(P, nx=0),
            dict(P, species=[dict(mass=-1.0, charge=0, stat=0, g=1.0)]),
            dict(P, species=[dict(mass=1.0, charge=0, stat=2, g=1.0)]),
            dict(P, species=[dict(mass=1.0, charge=0, stat=0, g=0.0)]),
            dict(P, grids=[dict(n=[4, 0, 4], pmin=[-1.0] * 3, pmax=[1.0] * 3)]),
            dict(P, grids=[dict(n=[4, 4, 4], pmin=[1.0] * 3, pmax=[1.0] * 3)]),
            dict(P, processes=[dict(a=0, b=1, c=0, d=1, kind=0, par=[1.0], sym=-1.0)]),
            dict(P, processes=[dict(a=0, b=0, c=0, d=0, kind=11, par=[1.0], sym=-1.0)])]
    for bad in bads:
        with pytest.raises(rbg.RbgError):
            rbg.Collision(bad)
    two = dict(P, species=P["species"] * 2, grids=P["grids"] * 2)
    with pytest.raises(rbg.RbgError, match="ambiguous"):          # a + b -> b + a must be written a + b -> a + b
        rbg.Collision(dict(two, processes=[dict(a=0, b=1, c=1, d=0, kind=0, par=[1.0], sym=-1.0)]))
    with pytest.raises(rbg.RbgError, match="elastic"):            # the t-channel sampler is for elastic processes
        rbg.Collision(dict(two, processes=[dict(a=0, b=0, c=1, d=1, kind=1, par=[1.0, 0.1], sym=-1.0, sampler=1)]))
    assert rbg.Collision(dict(two, processes=[dict(a=0, b=0, c=1, d=1, kind=0, par=[1.0], sym=-1.0)])).n_roles == 2
    col = rbg.Collision(P)
    f = torch.from_numpy(w["f"]).cuda()
    with pytest.raises(rbg.RbgError):
        col.collision(f, 0, 1)
    with pytest.raises(rbg.RbgError):
        col.collision(f[:-1], 8, 1)
    with pytest.raises(rbg.RbgError):
        col.set_option("no_such_option", 1)
    with pytest.raises(rbg.RbgError):
        col.set_option("warps_per_cta", 99)


def test_evolve_is_repeated_update():
    """rbg_collision_evolve = n_steps x rbg_collision_update with seeds seed + k, result in place."""
    rbg = _rbg()
    w = workloads.make(6, nx=2, np_side=8, n_samples=48)
    orc = oracle.Oracle(w["problem"])
    dt = 2e-4                                    # small enough that f stays non-negative (the scale G + L assumes it)
    ref, mags = w["f"].copy(), []
    for k in range(3):
        C_ref, mag = oracle_C_and_scale(orc, ref, w["n_samples"], w["seed"] + k)
        ref, neg = oracle.update(ref, C_ref, dt)
        assert neg == 0
        mags.append(mag)
    col = rbg.Collision(w["problem"])
    for steps in (3, 2, 1, 0):
        f = torch.from_numpy(w["f"]).cuda()
        got, flag = col.collision_evolve(f, dt, steps, w["n_samples"], w["seed"])
        torch.cuda.synchronize()
        assert got.data_ptr() == f.data_ptr()
        assert col.last_launch_count() == steps * orc.n_roles
        chain = torch.from_numpy(w["f"]).cuda()
        for k in range(steps):
            chain, _ = col.collision_update(chain, dt, w["n_samples"], w["seed"] + k)
        torch.cuda.synchronize()
        assert torch.equal(got, chain), steps
        if steps == 3:
            # each step's C agrees to TOL64 (G + L); a 1e-16 difference in f after step k feeds into step k+1
            tol = dt * TOL64 * sum(mags) + 1e-13 * np.abs(ref).max()
            assert np.all(np.abs(got.cpu().numpy() - ref) <= tol)
    f = torch.from_numpy(w["f"]).cuda()
    with pytest.raises(rbg.RbgError):
        col.collision_evolve(f, dt, 1, 8, 1, scratch=f)
    with pytest.raises(rbg.RbgError):
        col.collision_evolve(f, dt, -1, 8, 1)


@pytest.mark.parametrize("cfg,kw,fp32", [(2, dict(nx=3, np_side=20, n_samples=64), False), (2, dict(nx=2, np_side=7, n_samples=33), False),
                                         (3, dict(nx=2, np_side=8, n_samples=96), False), (2, dict(nx=2, np_side=10, n_samples=64), True),
                                         (3, dict(nx=1, np_side=8, n_samples=64), True)])
def test_parity_tchannel_importance_sampler(cfg, kw, fp32):
    """sampler = 1: same bar as the uniform sampler, both precisions, and a result that
    differs from the uniform sampler's (the two draw different directions from the same words)."""
    w = workloads.make(cfg, sampler=1, **kw)
    assert all(p.get("sampler") == 1 for p in w["problem"]["processes"])
    orc = oracle.Oracle(w["problem"], use_float=fp32)
    C_ref, mag = oracle_C_and_scale(orc, w["f"], w["n_samples"], w["seed"])
    C, col = gpu_C(w["problem"], w["f"], w["n_samples"], w["seed"], fp32=fp32)
    assert_parity(C, C_ref, mag, TOL32 if fp32 else TOL64, f"tchannel cfg{cfg} {kw}")
    w0 = workloads.make(cfg, **kw)
    C0, _ = gpu_C(w0["problem"], w0["f"], w0["n_samples"], w0["seed"], fp32=fp32)
    assert not np.array_equal(C, C0)
    if not fp32:
        other, _ = gpu_C(w["problem"], w["f"], w["n_samples"], w["seed"], options=[("gather", 2), ("warps_per_cta", 5)])
        assert np.array_equal(C, other)


def test_sampler_argument_errors():
    rbg = _rbg()
    P = workloads.make(1, np_side=4)["problem"]
    for bad in (dict(P, processes=[dict(P["processes"][0], sampler=1)]),                     # CONST kind
                dict(P, processes=[dict(P["processes"][0], kind=1, par=[1.0, 0.0], sampler=1)]),   # no regulator
                dict(P, processes=[dict(P["processes"][0], kind=1, par=[1.0, 0.1], sampler=7)])):
        with pytest.raises(rbg.RbgError):
            rbg.Collision(bad)


# ---------------------------------------------------------------------------------------------------------------
# NEXT-2(ii): Table III kinds and inelastic roles (workload 7 = the paper's quark-gluon plasma scenario, 70 roles)
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kw", [dict(nx=2, np_side=6, n_samples=48),       # 216-cell tables: TMA staging
                                dict(nx=3, np_side=5, n_samples=33),       # 125 cells: odd size, cooperative staging
                                dict(nx=1, np_side=11, n_samples=16)])     # the paper's 11^3 momentum grid
def test_parity_fp64_qgp_all_table3_processes(kw):
    w = workloads.make(7, **kw)
    orc = oracle.Oracle(w["problem"])
    assert orc.n_roles == 70
    C_ref, mag = oracle_C_and_scale(orc, w["f"], w["n_samples"], w["seed"])
    C, col = gpu_C(w["problem"], w["f"], w["n_samples"], w["seed"])
    assert_parity(C, C_ref, mag, TOL64, f"cfg7 {kw}")
    assert col.last_launch_count() == 70
    assert col.sample_evals(w["n_samples"]) == workloads.configs.sample_evals(w["problem"], w["n_samples"])
    # the global-memory gather path gives the same numbers
    C2, _ = gpu_C(w["problem"], w["f"], w["n_samples"], w["seed"], options=(("gather", 2),))
    assert np.array_equal(C, C2)


def test_parity_fp32_qgp():
    w = workloads.make(7, nx=2, np_side=6, n_samples=48)
    orc = oracle.Oracle(w["problem"], use_float=True)
    C_ref, mag = oracle_C_and_scale(orc, w["f"], w["n_samples"], w["seed"])
    C, _ = gpu_C(w["problem"], w["f"], w["n_samples"], w["seed"], fp32=True)
    assert_parity(C, C_ref, mag, TOL32, "fp32 cfg7")


def test_parity_inelastic_role_with_four_species_four_grids_and_a_threshold():
    """a + b -> c + d with four masses, four different momentum grids (three tables in shared memory) and unequal
    degrees of freedom: the heavy pair is below threshold for part of the samples."""
    species = [dict(mass=m, charge=0.0, stat=st, g=g) for m, st, g in
               ((0.2, -1, 2.0), (0.35, 1, 3.0), (0.9, 0, 1.0), (1.4, -1, 4.0))]
    grids = [dict(n=[6, 5, 7], pmin=[-2.0, -2.5, -2.0], pmax=[2.0, 2.5, 2.2]),
             dict(n=[4, 8, 6], pmin=[-3.0] * 3, pmax=[3.0] * 3),
             dict(n=[7, 7, 7], pmin=[-2.5] * 3, pmax=[2.5] * 3),
             dict(n=[8, 4, 6], pmin=[-3.5] * 3, pmax=[3.5] * 3)]
    procs = [dict(a=0, b=1, c=2, d=3, kind=0, par=[1.5], sym=-1.0),
             dict(a=2, b=2, c=0, d=3, kind=2, par=[1.3, 0.7], sym=-1.0)]
    prob = dict(nx=3, species=species, grids=grids, processes=procs, hbar=0.2)      # occupation numbers below 1
    rng = np.random.default_rng(77)
    orc = oracle.Oracle(prob)
    assert orc.n_roles == 7
    f = rng.random(orc.f_elems) * 0.2
    C_ref, mag = oracle_C_and_scale(orc, f, 80, 4321)
    C, col = gpu_C(prob, f, 80, 4321)
    assert_parity(C, C_ref, mag, TOL64, "four-species inelastic")
    # fused update over inelastic roles: several roles accumulate into one species block
    out_ref, neg_ref = oracle.update(f, C_ref, 0.05)
    ft = torch.from_numpy(f).cuda()
    out, flag = col.collision_update(ft, 0.05, 80, 4321)
    torch.cuda.synchronize()
    assert np.all(np.abs(out.cpu().numpy() - out_ref) <= 0.05 * TOL64 * mag + 1e-15)
    assert int(flag.item()) == neg_ref
