"""Parity of rbg_collision_symmetric (NEXT-3, the conservative estimator) against the oracle's orc_collision_symmetric
on the same seeded inputs: per cell within 1e-10 of the sum of the absolute deposits (the deposits are atomic adds, so
the order of summation differs from the oracle's and from run to run), plus the property it exists for: particle
number conserved to rounding."""
import numpy as np
import pytest
import torch

import oracle
import workloads

pytestmark = pytest.mark.gpu
TOL = 1e-10


def _rbg():
    import paper_2308_04869_b200 as rbg
    return rbg


def _run(prob, f, n, seed, tables=0):
    """tables = 1: deposits through per-CTA shared-memory tables (option "sym_tables") instead of global atomics."""
    col = _rbg().Collision(prob)
    col.set_option("sym_tables", tables)
    C = col.collision_symmetric(torch.from_numpy(np.ascontiguousarray(f)).cuda(), n, seed)
    torch.cuda.synchronize()
    return C.cpu().numpy(), col


@pytest.mark.parametrize("cfg,kw", [(1, dict(nx=3, np_side=8, n_samples=100)), (2, dict(nx=3, np_side=10, n_samples=64)),
                                    (3, dict(nx=2, np_side=8, n_samples=48)), (7, dict(nx=2, np_side=6, n_samples=32)),
                                    (6, dict(nx=2, np_side=9, n_samples=64)), (1, dict())])
@pytest.mark.parametrize("tables", [0, 1])
def test_symmetric_parity(cfg, kw, tables):
    w = workloads.make(cfg, **kw)
    orc = oracle.Oracle(w["problem"])
    C_ref, mag = orc.collision_symmetric(w["f"], w["n_samples"], w["seed"])
    C, col = _run(w["problem"], w["f"], w["n_samples"], w["seed"], tables)
    err = np.abs(C - C_ref)
    assert np.all(err <= TOL * mag + 1e-300), float(np.max(err / np.maximum(mag, 1e-300)))
    assert np.any(C_ref != 0) and col.last_launch_count() == orc.n_roles
    # it is a different estimator from the standard one, of the same quantity
    C_std = col.collision(torch.from_numpy(w["f"]).cuda(), w["n_samples"], w["seed"]).cpu().numpy()
    assert not np.allclose(C, C_std, rtol=1e-6, atol=0)


def test_symmetric_four_species_inelastic_and_global_accumulators():
    species = [dict(mass=m, charge=0.0, stat=st, g=g) for m, st, g in
               ((0.2, -1, 2.0), (0.35, 1, 3.0), (0.9, 0, 1.0), (1.4, -1, 4.0))]
    grids = [dict(n=[6, 5, 7], pmin=[-2.0, -2.5, -2.0], pmax=[2.0, 2.5, 2.2]), dict(n=[4, 8, 6], pmin=[-3.0] * 3, pmax=[3.0] * 3),
             dict(n=[7, 7, 7], pmin=[-2.5] * 3, pmax=[2.5] * 3), dict(n=[8, 4, 6], pmin=[-3.5] * 3, pmax=[3.5] * 3)]
    procs = [dict(a=0, b=1, c=2, d=3, kind=0, par=[1.5], sym=-1.0), dict(a=2, b=2, c=0, d=3, kind=2, par=[1.3, 0.7], sym=-1.0)]
    prob = dict(nx=3, species=species, grids=grids, processes=procs, hbar=0.2)
    orc = oracle.Oracle(prob)
    f = np.random.default_rng(77).random(orc.f_elems) * 0.2
    C_ref, mag = orc.collision_symmetric(f, 80, 4321)
    for tables in (0, 1):
        C, _ = _run(prob, f, 80, 4321, tables)
        assert np.all(np.abs(C - C_ref) <= TOL * mag + 1e-300)
    # 35^3 tables (343 KB each) do not fit in shared memory: the deposits go to global memory whatever the option says
    w = workloads.make(6, n_samples=8)
    orc = oracle.Oracle(w["problem"])
    C_ref, mag = orc.collision_symmetric(w["f"], 8, 3)
    C, _ = _run(w["problem"], w["f"], 8, 3, tables=1)
    assert np.all(np.abs(C - C_ref) <= TOL * mag + 1e-300)


def test_symmetric_conserves_particle_number_to_rounding():
    """Config-1-like problem with f supported in |p| < 1 (m = 1, box [-2,2]^3: nothing can leave the box)."""
    w = workloads.make(1, nx=4, np_side=16, n_samples=256)
    prob = w["problem"]
    prob["grids"][0] = dict(n=[16] * 3, pmin=[-2.0] * 3, pmax=[2.0] * 3)
    P = workloads.configs.cell_centres(prob["grids"][0])
    f = (w["f"].reshape(4, -1) * ((P * P).sum(1) < 1.0)[None, :]).reshape(-1)
    C, col = _run(prob, f, 256, 9)
    C_std = col.collision(torch.from_numpy(f).cuda(), 256, 9).cpu().numpy()
    per_cell_sym = np.abs(C.reshape(4, -1).sum(1))
    per_cell_std = np.abs(C_std.reshape(4, -1).sum(1))
    scale = np.abs(C).reshape(4, -1).sum(1)
    assert np.all(per_cell_sym < 1e-12 * scale)
    assert np.all(per_cell_std > 1e-5 * scale)


def test_symmetric_argument_errors():
    rbg = _rbg()
    w = workloads.make(2, nx=1, np_side=4, sampler=1)
    f = torch.from_numpy(w["f"]).cuda()
    with pytest.raises(rbg.RbgError, match="uniform"):
        rbg.Collision(w["problem"]).collision_symmetric(f, 8, 1)
    w = workloads.make(1, np_side=4)
    f = torch.from_numpy(w["f"]).cuda()
    with pytest.raises(rbg.RbgError, match="fp64"):
        rbg.Collision(w["problem"], fp32_kinematics=True).collision_symmetric(f, 8, 1)
    with pytest.raises(rbg.RbgError):
        rbg.Collision(w["problem"]).collision_symmetric(f, 8, 1, out=f)


def test_symmetric_and_local_be_steps_shard_over_spatial_cells():
    """Spatial shards (paper_2308_04869_b200.sharding, stream keyed by the global cell index) reproduce the one-device
    result: the conservative estimator to rounding (atomic order), moments and the Vlasov step bit for bit.  The drift
    stencil is the one step that does not shard without a ghost-layer exchange (rbg_drift_step refuses ix_offset != 0)."""
    from paper_2308_04869_b200 import sharding
    rbg = _rbg()
    w = workloads.make(2, nx=5, np_side=8, n_samples=40)
    prob = w["problem"]
    full = rbg.Collision(prob)
    f = torch.from_numpy(w["f"]).cuda()
    C_full = full.collision_symmetric(f, 40, 7).cpu().numpy()
    M_full = full.moments(f)[0].cpu().numpy()
    rng = np.random.default_rng(1)
    E = rng.normal(size=(5, 3)); B = rng.normal(size=(5, 3))
    V_full = full.vlasov_step(f, 0.01, torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda()).cpu().numpy()
    C_parts, V_parts, M_parts = [], [], []
    for rank in range(2):
        lp, lf, lo = sharding.shard_problem(prob, w["f"], rank, 2)
        hi = lo + lp["nx"]
        col = rbg.Collision(lp, ix_offset=lo)
        fd = torch.from_numpy(lf).cuda()
        C_parts.append(col.collision_symmetric(fd, 40, 7).cpu().numpy())
        V_parts.append(col.vlasov_step(fd, 0.01, torch.from_numpy(E[lo:hi]).cuda(), torch.from_numpy(B[lo:hi]).cuda()).cpu().numpy())
        M_parts.append(col.moments(fd)[0].cpu().numpy())
    C_sh = sharding.unshard(prob, C_parts)
    assert np.all(np.abs(C_sh - C_full) <= 1e-13 * np.abs(C_full).max())
    assert np.array_equal(sharding.unshard(prob, V_parts), V_full)
    assert np.array_equal(np.concatenate(M_parts, axis=1), M_full)


def test_be_step_with_the_conservative_estimator():
    """rbg_be_step(do_collision = 2): f <- f + 3 dt C_sym[f] after the drift and Vlasov sub-steps, against the composed
    oracles; with the transport sub-steps off and an input that cannot leak, particle number is conserved to rounding."""
    from oracle import be_steps as bs
    rbg = _rbg()
    nxyz = (2, 2, 1)
    w = workloads.make(2, nx=4, np_side=6, n_samples=40)
    prob = w["problem"]
    rng = np.random.default_rng(3)
    E = rng.normal(size=(4, 3)); B = rng.normal(size=(4, 3))
    dt, dx = 0.003, (0.5, 0.6, 0.7)
    f1 = bs.drift_upfd(prob, w["f"], nxyz, dt, dx)
    f2 = bs.vlasov_upfd(prob, f1, dt, E, B)
    orc = oracle.Oracle(prob)
    C_ref, mag = orc.collision_symmetric(f2, 40, 11)
    ref, neg_ref = oracle.update(f2, C_ref, 3 * dt)
    col = rbg.Collision(dict(prob, nx=nxyz))
    f = torch.from_numpy(w["f"]).cuda()
    out, flag = col.be_step(f, dt, dx=dx, E=torch.from_numpy(E).cuda(), B=torch.from_numpy(B).cuda(), n_samples=40, seed=11,
                            collision="symmetric")
    torch.cuda.synchronize()
    assert out.data_ptr() == f.data_ptr()
    assert np.all(np.abs(out.cpu().numpy() - ref) <= 3 * dt * TOL * mag + 1e-13 * np.abs(ref))
    assert int(flag.item()) == neg_ref
    # collision only, compact input (config-1-like, |p| < 1 in a [-2,2]^3 box): number conserved per spatial cell
    w1 = workloads.make(1, nx=3, np_side=16, n_samples=128)
    p1 = w1["problem"]
    p1["grids"][0] = dict(n=[16] * 3, pmin=[-2.0] * 3, pmax=[2.0] * 3)
    P = workloads.configs.cell_centres(p1["grids"][0])
    f0 = (w1["f"].reshape(3, -1) * ((P * P).sum(1) < 1.0)[None, :]).reshape(-1)
    c1 = rbg.Collision(p1)
    g = torch.from_numpy(f0).cuda()
    for k in range(5):
        c1.be_step(g, 0.01, n_samples=128, seed=50 + k, drift=False, vlasov=False, collision="symmetric")
    torch.cuda.synchronize()
    n0, n1 = f0.reshape(3, -1).sum(1), g.cpu().numpy().reshape(3, -1).sum(1)
    assert np.all(np.abs(n1 - n0) <= 1e-12 * n0) and not np.allclose(g.cpu().numpy(), f0)
