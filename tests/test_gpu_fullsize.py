"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times: the CUDA path
runs the whole sweep; the oracle recomputes a deterministic sample of spatial cells (cells are
independent and the stream is keyed by the global cell index, so a subset is exact evidence)."""
import numpy as np
import pytest
import torch

import oracle
import workloads
from test_gpu_parity import TOL32, TOL64, oracle_C_and_scale

pytestmark = pytest.mark.gpu


def _check_cells(w, C, cells, fp32):
    orc = oracle.Oracle(w["problem"], use_float=fp32)
    tol = TOL32 if fp32 else TOL64
    for ix in cells:
        C_ref, mag = oracle_C_and_scale(orc, w["f"], w["n_samples"], w["seed"], ix_begin=ix, ix_end=ix + 1)
        for s in range(orc.n_species):
            sl = slice(orc.sp_off[s] + ix * orc.np[s], orc.sp_off[s] + (ix + 1) * orc.np[s])
            err = np.abs(C[sl] - C_ref[sl])
            assert np.all(err <= tol * mag[sl]), (w["cfg"], ix, s, float(np.max(err / np.maximum(mag[sl], 1e-300))))
            assert np.any(C_ref[sl] != 0)


def _sample_cells(problem, n=16):
    """At least n spatial cells of a full-size problem: the first and the last two (both ends of every species block in the
    species-major layout), the two cells either side of the first CTA-wave boundary (one CTA per SM, 148 SMs, tiles of at
    most 512 momentum cells of the first species), the two in the middle, and an even spread over the rest."""
    nx = problem["nx"]
    tiles = -(-int(np.prod(problem["grids"][0]["n"])) // 512)
    wave = max(1, 148 // tiles)
    want = {0, 1, wave - 1, wave, nx // 2 - 1, nx // 2, nx - 2, nx - 1}
    want |= {int(v) for v in np.linspace(0, nx - 1, n)}
    return sorted(c for c in want if 0 <= c < nx)


@pytest.mark.parametrize("cfg", [2, 3, 4])
def test_fullsize_sampled_parity(cfg):
    import paper_2308_04869_b200 as rbg
    w = workloads.make(cfg)
    col = rbg.Collision(w["problem"])
    f = torch.from_numpy(w["f"]).cuda()
    C = col.collision(f, w["n_samples"], w["seed"])
    torch.cuda.synchronize()
    cells = _sample_cells(w["problem"])
    assert len(cells) >= 16
    _check_cells(w, C.cpu().numpy(), cells, False)
    # properties that hold at any size: finite everywhere, every spatial cell written
    assert bool(torch.isfinite(C).all())
    offs, _ = workloads.f_layout(w["problem"])
    npc = int(np.prod(w["problem"]["grids"][0]["n"]))
    per_cell = C[offs[0]:offs[0] + w["problem"]["nx"] * npc].view(w["problem"]["nx"], npc).abs().sum(1)
    assert bool((per_cell > 0).all())


def test_fullsize_config5_fused_update_fp32():
    import paper_2308_04869_b200 as rbg
    w = workloads.make(5)
    col = rbg.Collision(w["problem"], fp32_kinematics=True)
    f = torch.from_numpy(w["f"]).cuda()
    out, flag = col.collision_update(f, w["dt"], w["n_samples"], w["seed"])
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    orc = oracle.Oracle(w["problem"], use_float=True)
    cells = _sample_cells(w["problem"])
    assert len(cells) >= 16
    for ix in cells:
        C_ref, mag = oracle_C_and_scale(orc, w["f"], w["n_samples"], w["seed"], ix_begin=ix, ix_end=ix + 1)
        for s in range(orc.n_species):
            sl = slice(orc.sp_off[s] + ix * orc.np[s], orc.sp_off[s] + (ix + 1) * orc.np[s])
            ref = w["f"][sl] + w["dt"] * C_ref[sl]
            assert np.all(np.abs(got[sl] - ref) <= w["dt"] * TOL32 * mag[sl] + 4e-16 * np.abs(ref))
    assert int(flag.item()) == int((out < 0).sum().item())


def test_paper_collision_test_thermalises_species_b():
    """The paper's own collision workload at its full grid (35^3) through
    rbg_collision_evolve: species b (dsigma/dOmega = 20) reaches exp(-E/T) with the T its conserved energy per
    particle dictates, species a (dsigma/dOmega = 1) is still far from it (Fig. 9)."""
    import paper_2308_04869_b200 as rbg
    from test_oracle_thermalisation import boltzmann_fit, temperature_from_energy_per_particle
    from workloads.configs import cell_centres
    w = workloads.make(6)
    col = rbg.Collision(w["problem"])
    P = cell_centres(w["problem"]["grids"][0])
    E = np.sqrt((P * P).sum(1) + 0.3 ** 2)
    npc, dp3 = P.shape[0], (4.0 / 35) ** 3
    f0 = w["f"]
    f = torch.from_numpy(f0).cuda()
    _, flag = col.collision_evolve(f, w["dt"], 60, w["n_samples"], w["seed"])
    torch.cuda.synchronize()
    got = f.cpu().numpy()
    assert int(flag.item()) == int((got < 0).sum()) == 0
    fa, fb = got[:npc], got[npc:]
    (Ta, rms_a), (Tb, rms_b) = boltzmann_fit(fa, E), boltzmann_fit(fb, E)
    T_pred = temperature_from_energy_per_particle((f0[npc:] * E).sum() / f0[npc:].sum(), 0.3)
    assert rms_b < 0.12 and rms_a > 4 * rms_b, (rms_a, rms_b)
    assert abs(Tb - T_pred) < 0.05 * T_pred, (Tb, T_pred)
    assert abs(fa.sum() / f0[:npc].sum() - 1) < 5e-3
    assert 0.93 < fb.sum() / f0[npc:].sum() < 1.01
    # one step of it against the oracle, on the cells the oracle is asked for (every cell: nx = 1)
    C = col.collision(torch.from_numpy(f0).cuda(), 16, w["seed"])
    torch.cuda.synchronize()
    _check_cells(dict(w, n_samples=16), C.cpu().numpy(), (0,), False)


def test_fullsize_config2_tchannel_sampler():
    """Config 2 at full size with the t-channel importance sampler: sampled parity, and the per-cell scatter of
    C across spatial cells (which differ only by their density factor and their random streams) is far below
    the uniform sampler's."""
    import paper_2308_04869_b200 as rbg
    res = {}
    for sampler in (1, 0):
        w = workloads.make(2, sampler=sampler)
        col = rbg.Collision(w["problem"])
        C = col.collision(torch.from_numpy(w["f"]).cuda(), w["n_samples"], w["seed"])
        torch.cuda.synchronize()
        if sampler == 1:
            _check_cells(w, C.cpu().numpy(), (3, 508), False)
        res[sampler] = C
    # H+ block: C(x, p) / n(x)^2 is the same function of p in every spatial cell up to Monte Carlo noise
    offs, _ = workloads.f_layout(w["problem"])
    nx, npc = w["problem"]["nx"], 8000
    dens = torch.from_numpy(w["f"][offs[1]:offs[1] + nx * npc].reshape(nx, npc)[:, 0] / w["f"][offs[1]]).cuda()
    noise = {}
    for sampler, C in res.items():
        blk = C[offs[1]:offs[1] + nx * npc].view(nx, npc) / (dens * dens)[:, None]
        noise[sampler] = float(blk.std(0).mean())
    assert noise[1] < 0.2 * noise[0], noise


def test_fullsize_config7_qgp_sampled_parity():
    """Workload 7 (the paper's quark-gluon-plasma scenario, 21^3 x 11^3, 70 roles) at full size: the oracle recomputes
    16+ spatial cells; every cell is finite and written."""
    import paper_2308_04869_b200 as rbg
    w = workloads.make(7)
    col = rbg.Collision(w["problem"])
    C = col.collision(torch.from_numpy(w["f"]).cuda(), w["n_samples"], w["seed"])
    torch.cuda.synchronize()
    assert col.last_launch_count() == 70
    _check_cells(w, C.cpu().numpy(), _sample_cells(w["problem"]), False)
    assert bool(torch.isfinite(C).all())


def test_fullsize_be_steps_config4_and_config7():
    """NEXT-4 kernels at the sizes bench.py --path be times: sampled spatial cells against oracle/be_steps.py, plus
    properties that hold at any size (positivity, particle number of a periodic drift / uniform-force Vlasov step,
    totals = sum over species)."""
    import paper_2308_04869_b200 as rbg
    from oracle import be_steps as bs
    for cfg, nxyz in ((4, (32, 32, 32)), (7, (21, 21, 21))):
        w = workloads.make(cfg)
        prob = w["problem"]
        nx = prob["nx"]
        for sp, q in zip(prob["species"], (-1.0, 1.0, 2.0, 0.5, -0.5, 0.3, 1.5)):
            sp["charge"] = q
        col = rbg.Collision(dict(prob, nx=nxyz))
        f = torch.from_numpy(w["f"]).cuda()
        offs, _ = workloads.f_layout(prob)
        npcs = [int(np.prod(g["n"])) for g in prob["grids"]]
        # ---- moments: three sampled cells per species against the oracle (moments are local in x)
        M, tot, em = col.moments(f)
        torch.cuda.synchronize()
        Mh = M.cpu().numpy()
        cells = [0, nx // 2 + 1, nx - 1]
        sub = dict(prob, nx=len(cells))
        fsub = np.concatenate([w["f"][o:o + nx * n].reshape(nx, n)[cells].reshape(-1) for o, n in zip(offs, npcs)])
        M_ref, tot_ref, em_ref = bs.moments(sub, fsub)
        scale = np.maximum(np.abs(M_ref[..., 0:1]), np.abs(M_ref[..., 4:5])) * 25.0
        assert np.all(np.abs(Mh[:, cells] - M_ref) <= 1e-12 * scale)
        assert bool(((tot - M.sum(0)).abs() <= 1e-13 * M.abs().sum(0)).all())
        # ---- Vlasov: same sampled cells (the stencil is local in x); uniform E only: particle number conserved
        rng = np.random.default_rng(3)
        E = rng.normal(size=(nx, 3)); B = rng.normal(size=(nx, 3))
        out = col.vlasov_step(f, 0.01, torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda())
        torch.cuda.synchronize()
        ref = bs.vlasov_upfd(sub, fsub, 0.01, E[cells], B[cells])
        got = np.concatenate([out[o:o + nx * n].view(nx, n)[cells].reshape(-1).cpu().numpy() for o, n in zip(offs, npcs)])
        assert np.all(np.abs(got - ref) <= 1e-14 * np.abs(ref))
        assert bool((out > 0).all())
        outE = col.vlasov_step(f, 0.01, torch.from_numpy(E).cuda(), torch.zeros_like(torch.from_numpy(B)).cuda())
        for o, n in zip(offs, npcs):
            a, b = f[o:o + nx * n].view(nx, n).sum(1), outE[o:o + nx * n].view(nx, n).sum(1)
            assert torch.allclose(a, b, rtol=1e-12, atol=0)
        # ---- drift, periodic: per momentum cell the particle number is conserved.  Oracle check: the 3 x 3 x nz block
        # of rows (0..2, 0..2, :) run as its own periodic domain has the same x, y, z neighbours for its centre row
        # (1, 1, :) as the full domain
        dx = (0.5, 0.4, 0.3)
        out = col.drift_step(f, 0.02, dx)
        torch.cuda.synchronize()
        assert bool((out > 0).all())
        for o, n in zip(offs, npcs):
            a, b = f[o:o + nx * n].view(nx, n).sum(0), out[o:o + nx * n].view(nx, n).sum(0)
            assert torch.allclose(a, b, rtol=1e-12, atol=0)
        nz = nxyz[2]
        fsub = np.concatenate([w["f"][o:o + nx * n].reshape(*nxyz, n)[0:3, 0:3].reshape(-1) for o, n in zip(offs, npcs)])
        ref = bs.drift_upfd(dict(prob, nx=9 * nz), fsub, (3, 3, nz), 0.02, dx)
        o_sub = 0
        for o, n in zip(offs, npcs):
            r = ref[o_sub:o_sub + 9 * nz * n].reshape(3, 3, nz, n)[1, 1]
            g = out[o:o + nx * n].view(*nxyz, n)[1, 1].cpu().numpy()
            assert np.all(np.abs(g - r) <= 1e-14 * np.abs(r))
            o_sub += 9 * nz * n
        del f, out, outE, M, tot, em
        torch.cuda.empty_cache()
