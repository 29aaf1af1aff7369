"""Parity of the NEXT-4 kernels (rbg_moments, rbg_drift_step, rbg_vlasov_step) against oracle/be_steps.py through
the C ABI, element by element on the same seeded inputs.

Tolerances (fp64, derived from the arithmetic): a moment is a sum of Np products, compared within
1e-12 of the sum of the absolute values of its terms (summation order differs); a stencil output is a ratio of two
short sums of non-negative terms, compared within 1e-14 relative (a few roundings)."""
import numpy as np
import pytest
import torch

import workloads
from oracle import be_steps as bs

pytestmark = pytest.mark.gpu


def _rbg():
    import paper_2308_04869_b200 as rbg
    return rbg


def _with_grid(problem, nxyz):
    return dict(problem, nx=tuple(nxyz))


CASES = [(2, dict(np_side=20), (3, 2, 2)),          # two species, 8000-cell grids
         (7, dict(np_side=11), (2, 3, 2)),          # seven species, the paper's 11^3 grid (odd: a cell at p = 0)
         (3, dict(np_side=8), (1, 1, 5)),           # includes an almost massless species
         (1, dict(np_side=16), (1, 1, 1))]


@pytest.mark.parametrize("path", [0, 1])             # 0: symmetric-grid kernel where it applies, 1: general staged kernel
@pytest.mark.parametrize("cfg,kw,nxyz", CASES + [(4, dict(np_side=20), (1, 1, 7)),     # one species, odd number of units
                                                 (1, dict(np_side=7), (2, 1, 1))])    # odd np: the symmetric kernel does not apply
def test_moments_parity(cfg, kw, nxyz, path):
    rbg = _rbg()
    w = workloads.make(cfg, nx=int(np.prod(nxyz)), **kw)
    prob = w["problem"]
    for s, q in zip(prob["species"], (-1.0, 1.0, 2.0, 0.5, -0.5, 0.0, 1.5)):
        s["charge"] = q
    M_ref, tot_ref, em_ref = bs.moments(prob, w["f"])
    Mabs, totabs, _ = bs.moments(prob, np.abs(w["f"]))
    # scale of a term sum: moments of |f| with |weights| are bounded by E-weighted ones; use n and T00 of |f|
    col = rbg.Collision(_with_grid(prob, nxyz))
    col.set_option("moments_path", path)
    M, tot, em = col.moments(torch.from_numpy(w["f"]).cuda())
    torch.cuda.synchronize()
    M, tot, em = M.cpu().numpy(), tot.cpu().numpy(), em.cpu().numpy()
    assert M.shape == M_ref.shape
    pmax = max(max(abs(v) for v in g["pmin"] + g["pmax"]) for g in prob["grids"])
    scale = np.maximum(Mabs[..., 0:1], Mabs[..., 4:5]) * max(1.0, pmax) ** 2
    assert np.all(np.abs(M - M_ref) <= 1e-12 * scale), np.max(np.abs(M - M_ref) / scale)
    assert np.all(np.abs(tot - tot_ref) <= 1e-12 * scale.sum(0))
    assert np.all(np.abs(em - em_ref) <= 3e-12 * scale.sum(0)[:, :1])
    assert np.any(M_ref[..., 1:4] != 0) and np.all(M_ref[..., 0] > 0)
    assert col.last_launch_count() == len(prob["species"]) + 1


@pytest.mark.parametrize("cfg,kw,nxyz,bc,zeta", [
    (2, dict(np_side=8), (5, 4, 3), (1, 1, 1), 0.0),
    (2, dict(np_side=8), (5, 4, 3), (0, 1, 0), 0.0),          # absorbing walls in x and z
    (7, dict(np_side=5), (3, 6, 4), (0, 0, 0), 0.6),          # partially reflecting walls, odd momentum grid
    (4, dict(np_side=20), (2, 2, 19), (1, 0, 1), 1.0),        # slab boundary inside the z rows (19 cells per row, slabs of 16)
    (1, dict(np_side=16), (1, 1, 1), (1, 1, 1), 0.0)])        # one cell: every neighbour is the cell itself
def test_drift_step_parity(cfg, kw, nxyz, bc, zeta):
    rbg = _rbg()
    w = workloads.make(cfg, nx=int(np.prod(nxyz)), **kw)
    prob = w["problem"]
    dt, dx = 0.07, (0.5, 0.8, 0.3)
    ref = bs.drift_upfd(prob, w["f"], nxyz, dt, dx, bc=bc, zeta=zeta)
    col = rbg.Collision(_with_grid(prob, nxyz))
    out = col.drift_step(torch.from_numpy(w["f"]).cuda(), dt, dx, bc=bc, zeta=zeta)
    torch.cuda.synchronize()
    out = out.cpu().numpy()
    assert np.all(np.abs(out - ref) <= 1e-14 * np.abs(ref)), np.max(np.abs(out - ref) / np.abs(ref))
    assert np.all(out >= 0)
    # a single periodic cell is its own neighbour: the step leaves it unchanged; everything else moves
    assert np.allclose(out, w["f"], rtol=1e-13) == (int(np.prod(nxyz)) == 1)


@pytest.mark.parametrize("path", [0, 1])             # 0: symmetric-grid kernel where it applies, 1: general staged kernel
@pytest.mark.parametrize("cfg,kw,nx", [(2, dict(np_side=8), 7), (7, dict(np_side=5), 20), (2, dict(np_side=20), 3),
                                       (3, dict(np_side=6), 17),
                                       (4, dict(np_side=20), 301),    # several units per CTA: every ring slot is re-armed
                                       (1, dict(np_side=10), 5),      # 100 columns: 5 segments of 2 planes per column
                                       (1, dict(np_side=28), 2)])     # 784 columns: one segment, 800 threads
def test_vlasov_step_parity(cfg, kw, nx, path):
    rbg = _rbg()
    w = workloads.make(cfg, nx=nx, **kw)
    prob = w["problem"]
    for s, q in zip(prob["species"], (-1.0, 1.0, 2.0, 0.5, -0.5, 0.0, 1.5)):
        s["charge"] = q
    rng = np.random.default_rng(11)
    E = rng.normal(size=(nx, 3)); B = rng.normal(size=(nx, 3))
    E[0] = 0.0; B[0] = 0.0                                   # a field-free cell: f unchanged
    B[1] = 0.0
    dt = 0.02
    ref = bs.vlasov_upfd(prob, w["f"], dt, E, B)
    col = rbg.Collision(prob)
    col.set_option("vlasov_path", path)
    out = col.vlasov_step(torch.from_numpy(w["f"]).cuda(), dt, torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda())
    torch.cuda.synchronize()
    out = out.cpu().numpy()
    assert np.all(np.abs(out - ref) <= 1e-14 * np.abs(ref)), np.max(np.abs(out - ref) / np.abs(ref))
    assert np.all(out >= 0) and not np.allclose(out, w["f"])


def test_be_step_argument_errors():
    rbg = _rbg()
    w = workloads.make(1, np_side=4)
    col = rbg.Collision(w["problem"])
    f = torch.from_numpy(w["f"]).cuda()
    with pytest.raises(rbg.RbgError):
        col.drift_step(f, 0.1, (1.0, 1.0, 1.0), out=f)               # aliasing
    # partial overlap: the output starts one element before the end of f
    n = col.f_elems
    buf = torch.zeros(2 * n, dtype=torch.float64, device="cuda")
    buf[:n] = f
    EB = torch.zeros((1, 3), dtype=torch.float64, device="cuda")
    for call in (lambda: col.drift_step(buf[:n], 0.1, (1.0, 1.0, 1.0), out=buf[n - 1:2 * n - 1]),
                 lambda: col.drift_step_pfl(buf[:n], 0.1, (1.0, 1.0, 1.0), out=buf[n - 1:2 * n - 1]),
                 lambda: col.vlasov_step(buf[:n], 0.1, EB, EB, out=buf[1:n + 1])):
        with pytest.raises(rbg.RbgError, match="overlaps"):
            call()
    with pytest.raises(rbg.RbgError):
        col.drift_step(f, 0.1, (0.0, 1.0, 1.0))                      # dx = 0
    with pytest.raises(rbg.RbgError):
        col.drift_step(f, 0.1, (1.0, 1.0, 1.0), bc=(2, 1, 1))
    with pytest.raises(rbg.RbgError):
        col.drift_step(f, 0.1, (1.0, 1.0, 1.0), bc=(0, 1, 1), zeta=1.5)
    off = rbg.Collision(w["problem"], ix_offset=3)
    with pytest.raises(rbg.RbgError, match="ghost"):
        off.drift_step(f, 0.1, (1.0, 1.0, 1.0))
    skew = dict(w["problem"], grids=[dict(n=[4, 4, 4], pmin=[-1.0, -1.0, -1.0], pmax=[2.0, 1.0, 1.0])])
    with pytest.raises(rbg.RbgError, match="symmetric"):
        rbg.Collision(skew).drift_step(f, 0.1, (1.0, 1.0, 1.0), bc=(0, 1, 1), zeta=0.5)
    with pytest.raises(rbg.RbgError):
        col.vlasov_step(f, 0.1, torch.zeros(2, dtype=torch.float64, device="cuda"), torch.zeros(3, dtype=torch.float64, device="cuda"))


def test_be_step_validates_everything_before_the_first_launch():
    """A refused rbg_be_step must leave f untouched: the collision arguments are checked before the drift and Vlasov
    launches are queued."""
    rbg = _rbg()
    w = workloads.make(2, nx=4, np_side=6, n_samples=8)
    col = rbg.Collision(dict(w["problem"], nx=(4, 1, 1)))
    f0 = torch.from_numpy(w["f"]).cuda()
    E = torch.ones((4, 3), dtype=torch.float64, device="cuda"); B = torch.ones((4, 3), dtype=torch.float64, device="cuda")
    for kw in (dict(n_samples=0), dict(n_samples=8, dx=(1.0, 0.0, 1.0)), dict(n_samples=8, zeta=2.0, bc=(0, 1, 1))):
        f = f0.clone()
        with pytest.raises(rbg.RbgError):
            col.be_step(f, 0.01, E=E, B=B, seed=1, **kw)
        torch.cuda.synchronize()
        assert torch.equal(f, f0), kw
    tch = workloads.make(2, nx=4, np_side=6, n_samples=8, sampler=1)
    col2 = rbg.Collision(dict(tch["problem"], nx=(4, 1, 1)))
    f = f0.clone()
    with pytest.raises(rbg.RbgError, match="uniform sampler"):
        col2.be_step(f, 0.01, E=E, B=B, n_samples=8, seed=1, collision="symmetric")
    torch.cuda.synchronize()
    assert torch.equal(f, f0)


def test_be_step_is_drift_then_vlasov_then_collision_with_3dt():
    """rbg_be_step against the composition of the three oracles (Eq. 25-27; order: DESIGN.md reading R24)."""
    import oracle
    from test_gpu_parity import oracle_C_and_scale
    rbg = _rbg()
    nxyz = (3, 2, 2)
    w = workloads.make(2, nx=12, np_side=6, n_samples=48)
    prob = w["problem"]
    rng = np.random.default_rng(4)
    E = rng.normal(size=(12, 3)); B = rng.normal(size=(12, 3))
    dt, dx = 0.004, (0.5, 0.7, 0.9)
    f1 = bs.drift_upfd(prob, w["f"], nxyz, dt, dx, bc=(1, 0, 1), zeta=0.5)
    f2 = bs.vlasov_upfd(prob, f1, dt, E, B)
    orc = oracle.Oracle(prob)
    C_ref, mag = oracle_C_and_scale(orc, f2, 48, 777)
    ref, neg_ref = oracle.update(f2, C_ref, 3 * dt)
    col = rbg.Collision(_with_grid(prob, nxyz))
    f = torch.from_numpy(w["f"]).cuda()
    out, flag = col.be_step(f, dt, dx=dx, bc=(1, 0, 1), zeta=0.5, E=torch.from_numpy(E).cuda(), B=torch.from_numpy(B).cuda(),
                            n_samples=48, seed=777)
    torch.cuda.synchronize()
    assert out.data_ptr() == f.data_ptr()
    got = out.cpu().numpy()
    assert np.all(np.abs(got - ref) <= 3 * dt * 1e-10 * mag + 1e-13 * np.abs(ref))
    assert int(flag.item()) == neg_ref
    assert col.last_launch_count() == 2 + 2 + 4
    # sub-steps can be switched off; two of them leave the result in f as well
    g = torch.from_numpy(w["f"]).cuda()
    col.be_step(g, dt, dx=dx, bc=(1, 0, 1), zeta=0.5, collision=False, E=torch.from_numpy(E).cuda(), B=torch.from_numpy(B).cuda())
    torch.cuda.synchronize()
    assert np.all(np.abs(g.cpu().numpy() - f2) <= 1e-13 * np.abs(f2))
    with pytest.raises(rbg.RbgError):
        col.be_step(g, dt, dx=dx, E=None, B=None)


@pytest.mark.parametrize("cfg,kw,nx", [(2, dict(np_side=20), 1300),      # one cell per stage, two stages: every CTA reuses its slots 4-5 times
                                       (7, dict(np_side=11), 2500),      # four cells per stage, odd np: leading cell, cooperative tails
                                       (1, dict(np_side=16), 1000)])     # two cells per stage (4096-cell grid)
@pytest.mark.parametrize("path", [0, 1])
def test_staged_kernels_are_race_free_under_ring_reuse(cfg, kw, nx, path):
    """The persistent moments / Vlasov kernels recycle their shared-memory stages through mbarrier phases and warp
    arrival counters.  Many units per CTA, repeated runs: every run must equal the oracle and, bit for bit, every
    other run (both kernels add in a fixed order)."""
    rbg = _rbg()
    w = workloads.make(cfg, nx=nx, **kw)
    prob = w["problem"]
    for s, q in zip(prob["species"], (-1.0, 1.0, 2.0, 0.5, -0.5, 0.3, 1.5)):
        s["charge"] = q
    rng = np.random.default_rng(8)
    E = rng.normal(size=(nx, 3)); B = rng.normal(size=(nx, 3))
    M_ref, _, _ = bs.moments(prob, w["f"])
    V_ref = bs.vlasov_upfd(prob, w["f"], 0.02, E, B)
    col = rbg.Collision(prob)
    col.set_option("moments_path", path)       # 0: the symmetric-grid moments kernel (three stages, two teams) for cfg 2 and 1
    col.set_option("vlasov_path", path)        # 0: the symmetric-grid Vlasov kernel (three stages, 800 / 768 threads)
    f = torch.from_numpy(w["f"]).cuda()
    Ed, Bd = torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda()
    first = None
    for rep in range(6):
        M, _, _ = col.moments(f)
        V = col.vlasov_step(f, 0.02, Ed, Bd)
        torch.cuda.synchronize()
        if first is None:
            first = (M.clone(), V.clone())
            Mh = M.cpu().numpy()
            scale = np.maximum(np.abs(M_ref[..., 0:1]), np.abs(M_ref[..., 4:5])) * 30.0
            assert np.all(np.abs(Mh - M_ref) <= 1e-12 * scale)
            assert np.all(np.abs(V.cpu().numpy() - V_ref) <= 1e-14 * np.abs(V_ref))
        else:
            assert torch.equal(M, first[0]) and torch.equal(V, first[1]), rep


def _tiny_problem(n, nx, asym=False):
    """asym: the first species' box is not symmetric about p_x = 0 (the symmetric-grid kernels must not be taken for it)."""
    return dict(nx=nx, species=[dict(mass=0.4, charge=-1.0, stat=0, g=1.0), dict(mass=0.0, charge=2.0, stat=0, g=1.0)],
                grids=[dict(n=list(n), pmin=[-1.0, -2.0, -1.5], pmax=[1.75 if asym else 1.0, 2.0, 1.5]),
                       dict(n=list(n[::-1]), pmin=[-2.0] * 3, pmax=[2.0] * 3)],
                processes=[], hbar=1.0)


@pytest.mark.parametrize("n,nx,asym", [((1, 1, 1), 1, False), ((1, 1, 1), 37, False), ((2, 1, 3), 5, False), ((3, 7, 1), 64, False),
                                       ((1, 40, 33), 3, False),
                                       # even cell counts with odd extents: the symmetric-grid kernels with a centre plane / row
                                       ((3, 2, 2), 40, False), ((1, 2, 2), 7, False), ((7, 6, 2), 9, False),
                                       ((5, 4, 6), 700, False),      # five units per CTA: every ring slot re-armed, centre plane
                                       ((2, 24, 32), 5, False),      # 768 columns: Vlasov one segment per column, moments general kernel
                                       ((20, 3, 1), 11, False),      # three columns: twenty one-plane segments per column
                                       ((4, 4, 4), 300, True)])      # box not symmetric about p_x = 0: general kernels
def test_be_steps_on_degenerate_momentum_grids(n, nx, asym):
    """Edge cases: one momentum cell (its own periodic neighbour), extents of 1 along some axes, a (ipy, ipz) plane wider
    than a team (1 x 40 x 33), odd extents in the symmetric-grid kernels, a box that is not symmetric, a massless species
    with a cell at p = 0, no processes at all."""
    rbg = _rbg()
    prob = _tiny_problem(n, nx, asym)
    rng = np.random.default_rng(21)
    npc = int(np.prod(n))
    f = rng.random(2 * nx * npc) + 0.05
    E = rng.normal(size=(nx, 3)); B = rng.normal(size=(nx, 3))
    col = rbg.Collision(prob)
    fd = torch.from_numpy(f).cuda()
    M, tot, em = col.moments(fd)
    V = col.vlasov_step(fd, 0.03, torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda())
    D = col.drift_step(fd, 0.03, (0.4, 0.5, 0.6), bc=(1, 1, 1))
    torch.cuda.synchronize()
    M_ref, tot_ref, em_ref = bs.moments(prob, f)
    scale = np.maximum(M_ref[..., 0:1], M_ref[..., 4:5]) * 16.0
    assert np.all(np.abs(M.cpu().numpy() - M_ref) <= 1e-12 * scale)
    assert np.all(np.abs(em.cpu().numpy() - em_ref) <= 1e-12 * scale.sum(0)[:, :1])
    V_ref = bs.vlasov_upfd(prob, f, 0.03, E, B)
    assert np.all(np.abs(V.cpu().numpy() - V_ref) <= 1e-14 * np.abs(V_ref))
    D_ref = bs.drift_upfd(prob, f, (nx, 1, 1), 0.03, (0.4, 0.5, 0.6))
    assert np.all(np.abs(D.cpu().numpy() - D_ref) <= 1e-14 * np.abs(D_ref))


def test_be_steps_massless_species_with_a_centre_that_is_zero_only_up_to_rounding():
    """A massless species on an odd grid whose box edges are not dyadic: the centre cell's momentum is ~1e-16, not 0, so
    E_p ~ 1e-16 and v = p / E_p is decided by the last bit of the centre.  The kernels must form the centre exactly as the
    1/E and v tables (and the oracle) do -- pmin + (i + 1/2) delta in two roundings; a fused form fails here."""
    rbg = _rbg()
    box = [1.8258518432329411, 1.966972915376824, 1.6607711616229521]
    for n, nx in (((3, 7, 5), 7), ((5, 2, 6), 300)):                    # general kernels (odd cell count) / symmetric-grid kernels
        prob = dict(nx=nx, species=[dict(mass=0.0, charge=-1.0, stat=0, g=1.0)],
                    grids=[dict(n=list(n), pmin=[-b for b in box], pmax=list(box))], processes=[], hbar=1.0)
        rng = np.random.default_rng(5)
        f = rng.random(nx * int(np.prod(n))) + 0.05
        E = rng.normal(size=(nx, 3)); B = rng.normal(size=(nx, 3))
        col = rbg.Collision(prob)
        fd = torch.from_numpy(f).cuda()
        M, _, _ = col.moments(fd)
        V = col.vlasov_step(fd, 0.03, torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda())
        torch.cuda.synchronize()
        M_ref, _, _ = bs.moments(prob, f)
        scale = np.maximum(M_ref[..., 0:1], M_ref[..., 4:5]) * 16.0
        assert np.all(np.abs(M.cpu().numpy() - M_ref) <= 1e-12 * scale)
        V_ref = bs.vlasov_upfd(prob, f, 0.03, E, B)
        assert np.all(np.abs(V.cpu().numpy() - V_ref) <= 1e-14 * np.abs(V_ref))


def test_be_steps_on_the_papers_35_cubed_grid_use_the_direct_kernels():
    """A 35^3 block (343 KB) does not fit in shared memory: moments and Vlasov fall back to their direct kernels."""
    rbg = _rbg()
    w = workloads.make(6, nx=3)
    prob = w["problem"]
    prob["species"][0]["charge"], prob["species"][1]["charge"] = -1.0, 1.0
    rng = np.random.default_rng(2)
    f = w["f"] + 0.01 * rng.random(w["f"].size)
    E = rng.normal(size=(3, 3)); B = rng.normal(size=(3, 3))
    col = rbg.Collision(prob)
    fd = torch.from_numpy(f).cuda()
    M = col.moments(fd)[0].cpu().numpy()
    V = col.vlasov_step(fd, 0.01, torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda()).cpu().numpy()
    M_ref = bs.moments(prob, f)[0]
    assert np.all(np.abs(M - M_ref) <= 1e-12 * np.maximum(M_ref[..., 0:1], M_ref[..., 4:5]) * 4.0)
    V_ref = bs.vlasov_upfd(prob, f, 0.01, E, B)
    assert np.all(np.abs(V - V_ref) <= 1e-14 * np.abs(V_ref))


def test_be_step_is_capturable_in_a_cuda_graph():
    """All launches of rbg_be_step go to the caller's stream back to back: a CUDA graph of one step replays to the same
    result as direct calls (launch-bound small problems are the use case)."""
    rbg = _rbg()
    nxyz = (2, 2, 2)
    w = workloads.make(2, nx=8, np_side=6, n_samples=32)
    prob = w["problem"]
    rng = np.random.default_rng(6)
    E = torch.from_numpy(rng.normal(size=(8, 3))).cuda(); B = torch.from_numpy(rng.normal(size=(8, 3))).cuda()
    col = rbg.Collision(_with_grid(prob, nxyz))
    kw = dict(dx=(0.5, 0.5, 0.5), E=E, B=B, n_samples=32, seed=5)
    ref = torch.from_numpy(w["f"]).cuda()
    for _ in range(3):
        col.be_step(ref, 0.002, **kw)
    torch.cuda.synchronize()
    f = torch.from_numpy(w["f"]).cuda()
    scratch, flag = torch.empty_like(f), torch.zeros(1, dtype=torch.int32, device="cuda")
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        col.be_step(f, 0.002, scratch=scratch, neg_flag=flag, stream=side, **kw)       # warm-up outside the capture
        f.copy_(torch.from_numpy(w["f"]).cuda())
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            col.be_step(f, 0.002, scratch=scratch, neg_flag=flag, stream=torch.cuda.current_stream(), **kw)
    torch.cuda.current_stream().wait_stream(side)
    for _ in range(3):
        graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(f, ref)


@pytest.mark.parametrize("cfg,kw,nxyz", [(2, dict(np_side=8), (5, 4, 3)), (7, dict(np_side=5), (3, 6, 4)),
                                         (4, dict(np_side=20), (2, 2, 19)), (1, dict(np_side=16), (1, 1, 1)),
                                         (1, dict(np_side=6), (2, 1, 2))])
def test_drift_step_pfl_parity(cfg, kw, nxyz):
    """Second-order flux-limited drift (Eq. 31-33) against oracle.be_steps.drift_pfl.  Tolerance: the update subtracts
    six limited face values scaled by 3 dt |v| / dx from f; 1e-13 of the local scale max(f, neighbours)."""
    rbg = _rbg()
    w = workloads.make(cfg, nx=int(np.prod(nxyz)), **kw)
    prob = w["problem"]
    f = w["f"].copy()
    f[::11] = 0.0                                              # empty cells exercise the limiter's special cases
    f[5::13] = f[4::13][:f[5::13].size]                        # equal neighbours along the momentum axis only (harmless)
    dt, dx = 0.02, (0.5, 0.8, 0.3)
    ref = bs.drift_pfl(prob, f, nxyz, dt, dx)
    col = rbg.Collision(_with_grid(prob, nxyz))
    out = col.drift_step_pfl(torch.from_numpy(f).cuda(), dt, dx)
    torch.cuda.synchronize()
    out = out.cpu().numpy()
    scale = np.abs(f).max()
    # the local scale the docstring names: per momentum cell, the largest |f| among the spatial cell itself and its
    # neighbours up to two cells away along each axis (the stencil of Eq. 32-33), periodic
    offs, _ = workloads.f_layout(dict(prob, nx=int(np.prod(nxyz))))
    tol = np.empty_like(f)
    ends = offs[1:] + [f.size]
    for o, e in zip(offs, ends):
        a = np.abs(f[o:e]).reshape(*nxyz, -1)
        loc = a.copy()
        for d in range(3):
            for k in (-2, -1, 1, 2):
                loc = np.maximum(loc, np.roll(a, k, axis=d))
        tol[o:e] = 1e-13 * loc.reshape(-1)
    assert np.all(np.abs(out - ref) <= tol + 1e-300), float(np.max(np.abs(out - ref) / (tol + 1e-300)))
    assert scale > 0
