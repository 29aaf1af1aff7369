"""Randomly drawn small problems (seeded): the CUDA path against the oracles on shapes nobody chose by hand -- mixed
masses (massless included), unequal and shifted momentum boxes, 1-4 species, elastic and inelastic processes of every
|M|^2 kind, both samplers, hbar != 1, random launch options; and random momentum grids for the moments / Vlasov / drift
kernels (odd and even extents, symmetric and non-symmetric boxes, non-dyadic edges, walls).  Same bars as the hand-made
cases: 1e-10 (fp64) / 1e-4 (fp32 kinematics) of |gain| + |loss| per cell, 1e-12 for a moment, 1e-14 for a stencil output.
Occupations are kept physical (fermions below 1) so that every sample's gain and loss are non-negative and |G| + |L| is the
sum of the absolute terms."""
import numpy as np
import pytest
import torch

import oracle
from oracle import be_steps as bs
from test_gpu_parity import oracle_C_and_scale

pytestmark = pytest.mark.gpu


def _rbg():
    import paper_2308_04869_b200 as rbg
    return rbg


def _random_problem(rng):
    ns = int(rng.integers(1, 5))
    hbar = float(rng.choice([1.0, 0.2, 0.5]))
    species, grids = [], []
    for _ in range(ns):
        m = float(rng.choice([0.0, 0.05, 0.3, 1.0, 7.0, 50.0]))
        species.append(dict(mass=m, charge=0.0, stat=int(rng.choice([0, 0, 1, -1])), g=float(rng.choice([1.0, 2.0, 6.0, 16.0]))))
        n = [int(rng.integers(2, 9)) for _ in range(3)]
        if m == 0.0:
            n = [2 * max(1, k // 2) for k in n]                    # massless: no cell centre at p = 0 (include/rbg.h)
        L = [float(rng.uniform(1.0, 6.0)) * (1.0 + m) for _ in range(3)]
        shift = [float(rng.uniform(-0.3, 0.3)) * l if m > 0 else 0.0 for l in L]
        grids.append(dict(n=n, pmin=[-l + sh for l, sh in zip(L, shift)], pmax=[l + sh for l, sh in zip(L, shift)]))
    procs = []
    for _ in range(int(rng.integers(1, 4))):
        a, b = int(rng.integers(ns)), int(rng.integers(ns))
        kind = int(rng.integers(0, 11))
        if rng.random() < 0.7 or ns < 3:
            c, d = a, b
        else:
            c, d = int(rng.integers(ns)), int(rng.integers(ns))
            if (c, d) == (b, a) and a != b:
                c, d = a, b
        sampler = 1 if (c, d) == (a, b) and kind in (1, 2) and rng.random() < 0.4 else 0
        procs.append(dict(a=a, b=b, c=c, d=d, kind=kind, par=[float(rng.uniform(0.5, 2.0)), float(rng.uniform(0.2, 1.0)), 0.0, 0.0],
                          sym=-1.0, sampler=sampler))
    return dict(nx=int(rng.integers(1, 4)), species=species, grids=grids, processes=procs, hbar=hbar)


def _physical_f(rng, prob):
    parts = []
    for sp, g in zip(prob["species"], prob["grids"]):
        kappa = (2.0 * np.pi * prob["hbar"]) ** 3 / sp["g"]
        top = 0.9 / kappa if sp["stat"] == -1 else float(rng.choice([0.05, 1.0, 20.0]))     # fermions: occupation below 1
        parts.append(rng.random(prob["nx"] * int(np.prod(g["n"]))) * top)
    return np.concatenate(parts)


@pytest.mark.parametrize("seed", [101, 102, 103, 104])
def test_random_collision_problems(seed):
    rbg = _rbg()
    rng = np.random.default_rng(seed)
    for case in range(6):
        prob = _random_problem(rng)
        f = _physical_f(rng, prob)
        N = int(rng.choice([1, 7, 32, 33, 64, 100]))
        mc_seed = int(rng.integers(1, 2 ** 62))
        nx = prob["nx"]
        for fp32 in (False, True):
            orc = oracle.Oracle(prob, use_float=fp32)
            C_ref, mag = oracle_C_and_scale(orc, f, N, mc_seed)
            col = rbg.Collision(prob, fp32_kinematics=fp32)
            if rng.random() < 0.3:
                col.set_option("gather", 2)
            if rng.random() < 0.3:
                col.set_option("warps_per_cta", int(rng.choice([1, 5, 8, 12, 16, 20, 32])))
            if rng.random() < 0.3:
                col.set_option("p1_per_cta", int(rng.choice([1, 7, 33, 100])))
            fd = torch.from_numpy(f).cuda()
            C = col.collision(fd, N, mc_seed).cpu().numpy()
            tol = 1e-4 if fp32 else 1e-10
            assert np.all(np.abs(C - C_ref) <= tol * mag + 1e-300), (seed, case, fp32, float(np.max(np.abs(C - C_ref) / np.maximum(mag, 1e-300))))
            if fp32:
                continue
            # fused Euler update
            dt = float(rng.choice([1e-3, 5.0]))
            out, _ = col.collision_update(fd, dt, N, mc_seed)
            assert np.all(np.abs(out.cpu().numpy() - (f + dt * C_ref)) <= 1e-10 * dt * mag + 1e-15 * np.abs(f)), (seed, case)
            # the upper half of the spatial cells as a shard: bit-identical
            if nx >= 2:
                lo, parts, refs, off = nx // 2, [], [], 0
                for g in prob["grids"]:
                    npc = int(np.prod(g["n"]))
                    parts.append(f[off:off + nx * npc].reshape(nx, npc)[lo:].reshape(-1))
                    refs.append(C[off:off + nx * npc].reshape(nx, npc)[lo:].reshape(-1))
                    off += nx * npc
                shard = rbg.Collision(dict(prob, nx=nx - lo), ix_offset=lo)
                C2 = shard.collision(torch.from_numpy(np.concatenate(parts)).cuda(), N, mc_seed).cpu().numpy()
                assert np.array_equal(C2, np.concatenate(refs)), (seed, case)
            # this repo's conservative estimator (uniform sampler only), both accumulator variants
            if all(p["sampler"] == 0 for p in prob["processes"]):
                Cs_ref, smag = orc.collision_symmetric(f, N, mc_seed)
                for tables in (0, 1):
                    col.set_option("sym_tables", tables)
                    Cs = col.collision_symmetric(fd, N, mc_seed).cpu().numpy()
                    assert np.all(np.abs(Cs - Cs_ref) <= 1e-10 * smag + 1e-300), (seed, case, tables)


@pytest.mark.parametrize("seed", [201, 202, 203])
def test_random_momentum_grids_for_moments_vlasov_drift(seed):
    rbg = _rbg()
    rng = np.random.default_rng(seed)
    for case in range(12):
        n = [int(rng.integers(1, 13)) for _ in range(3)]
        asym = rng.random() < 0.25
        L = [float(rng.uniform(0.5, 3.0)) for _ in range(3)]                                  # non-dyadic edges
        g0 = dict(n=n, pmin=[-l for l in L], pmax=[l * (1.3 if (asym and d == 1) else 1.0) for d, l in enumerate(L)])
        g1 = dict(n=[int(rng.integers(1, 25)) for _ in range(3)], pmin=[-2.0] * 3, pmax=[2.0] * 3)
        nxyz = (int(rng.integers(1, 6)), int(rng.integers(1, 6)), int(rng.integers(1, 40)))
        nx = int(np.prod(nxyz))
        prob = dict(nx=nx, species=[dict(mass=float(rng.choice([0.0, 0.4, 2.0])), charge=-1.0, stat=0, g=1.0),
                                    dict(mass=0.3, charge=2.0, stat=0, g=1.0)], grids=[g0, g1], processes=[], hbar=1.0)
        f = rng.random(nx * (int(np.prod(n)) + int(np.prod(g1["n"])))) + 0.05
        E = rng.normal(size=(nx, 3)); B = rng.normal(size=(nx, 3))
        bc = (1, 1, 1) if asym else tuple(int(v) for v in rng.integers(0, 2, size=3))          # reflecting walls need symmetric grids
        zeta = float(rng.choice([0.0, 0.5, 1.0]))
        col = rbg.Collision(dict(prob, nx=nxyz))
        fd = torch.from_numpy(f).cuda()
        M, _, _ = col.moments(fd)
        V = col.vlasov_step(fd, 0.03, torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda())
        D = col.drift_step(fd, 0.03, (0.4, 0.5, 0.6), bc=bc, zeta=zeta)
        torch.cuda.synchronize()
        M_ref, _, _ = bs.moments(prob, f)
        Mabs, _, _ = bs.moments(prob, np.abs(f))
        scale = np.maximum(Mabs[..., 0:1], Mabs[..., 4:5]) * 16.0
        assert np.all(np.abs(M.cpu().numpy() - M_ref) <= 1e-12 * scale), (seed, case, n, g1["n"], nxyz)
        V_ref = bs.vlasov_upfd(prob, f, 0.03, E, B)
        assert np.all(np.abs(V.cpu().numpy() - V_ref) <= 1e-14 * np.abs(V_ref)), (seed, case, n, g1["n"], nxyz)
        D_ref = bs.drift_upfd(prob, f, nxyz, 0.03, (0.4, 0.5, 0.6), bc=bc, zeta=zeta)
        assert np.all(np.abs(D.cpu().numpy() - D_ref) <= 1e-14 * np.abs(D_ref)), (seed, case, n, g1["n"], nxyz, bc, zeta)
