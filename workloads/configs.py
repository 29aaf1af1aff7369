"""The five BASELINE.json configs as seeded synthetic phase-space grids (recipe: DESIGN.md section 6).

The paper uses no public dataset; its collision workloads are self-defined momentum boxes
(PAPER.md:469, :510).  The configs take their shape from them: uniform Cartesian momentum grid,
layout [species][ix][ipx][ipy][ipz] with ipz fastest, thermal-like f.
"""
from __future__ import annotations

import numpy as np

KIND_CONST = 0              # |M|^2 = par[0]
KIND_COULOMB_SCREENED = 1   # |M|^2 = par[0] / (t - par[1]^2)^2
KIND_TCHAN_S2 = 2           # |M|^2 = par[0]^4 s^2 / (t - par[1]^2)^2
KIND_ISO_DSIGMA = 3         # |M|^2 = 64 pi^2 s par[0]  (constant CM-frame dsigma/dOmega = par[0])

INPUT_SEED_BASE = 0x5EED0000
MC_SEED_BASE = 20230810


def _grid(n, lo, hi):
    return dict(n=[int(n)] * 3, pmin=[float(lo)] * 3, pmax=[float(hi)] * 3)


def cell_centres(grid):
    """(np, 3) array of cell-centre momenta, ipz fastest."""
    ax = []
    for d in range(3):
        n, lo, hi = grid["n"][d], grid["pmin"][d], grid["pmax"][d]
        ax.append(lo + (np.arange(n) + 0.5) * ((hi - lo) / n))
    P = np.stack(np.meshgrid(*ax, indexing="ij"), axis=-1).reshape(-1, 3)
    return P


def f_layout(problem):
    """Offsets of each species' block and the total element count of the f / C arrays."""
    offs, off = [], 0
    for g in problem["grids"]:
        offs.append(off)
        off += problem["nx"] * int(np.prod(g["n"]))
    return offs, off


def equilibrium_nbar(E, T, stat, mu=0.0):
    """Occupation number at equilibrium (Eq. 11 PAPER.md:140-145 for stat=0; FD/BE for -1/+1)."""
    return 1.0 / (np.exp((E - mu) / T) - stat)


def _elastic(a, b, kind, par):
    return dict(a=a, b=b, c=a, d=b, kind=kind, par=list(par), sym=-1.0)


def make(cfg: int, nx: int | None = None, n_samples: int | None = None, np_side: int | None = None,
         sampler: int = 0):
    """Return dict(name, problem, f, n_samples, seed, dt, fp32).  ``nx``/``n_samples``/``np_side``
    override the config's spatial cell count / sample count / momentum cells per axis (tests use
    reduced sizes; bench.py uses the defaults).  ``sampler`` = 1 asks for the t-channel importance
    sampler on every process whose |M|^2 kind has the t-channel shape (configs 2, 3, 5)."""
    rng = np.random.Generator(np.random.PCG64(INPUT_SEED_BASE + cfg))
    seed = MC_SEED_BASE + cfg
    dt, fp32 = 0.0, False
    if cfg == 1:
        nxd, N, side = 1, 256, 16
        nx = nxd if nx is None else nx
        side = side if np_side is None else np_side
        species = [dict(mass=1.0, charge=0.0, stat=0, g=1.0)]
        grids = [_grid(side, -5.0, 5.0)]
        procs = [_elastic(0, 0, KIND_CONST, [1.0])]
        P = cell_centres(grids[0])
        E = np.sqrt((P * P).sum(1) + 1.0)
        f = np.exp(-E / 1.0)[None, :] * (1.0 + 0.1 * (2.0 * rng.random((nx, P.shape[0])) - 1.0))
        fs = [f]
        name = "cfg1: 1 classical species, const |M|^2, MJ T=1 + 10% noise"
    elif cfg in (2, 5):
        nxd, N, side = (512, 1024, 20) if cfg == 2 else (4096, 2048, 20)
        nx = nxd if nx is None else nx
        side = side if np_side is None else np_side
        species = [dict(mass=1.0, charge=-1.0, stat=0, g=1.0), dict(mass=1836.0, charge=1.0, stat=0, g=1.0)]
        grids = [_grid(side, -5.0, 5.0), _grid(side, -50.0, 50.0)]
        par = [1.0, 0.1]
        procs = [_elastic(0, 0, KIND_COULOMB_SCREENED, par), _elastic(0, 1, KIND_COULOMB_SCREENED, par),
                 _elastic(1, 1, KIND_COULOMB_SCREENED, par)]
        fs = []
        for s, g in zip(species, grids):
            P = cell_centres(g)
            E = np.sqrt((P * P).sum(1) + s["mass"] ** 2)
            dens = 1.0 + 0.1 * (2.0 * rng.random(nx) - 1.0)          # seeded density perturbation n(x)
            fs.append(dens[:, None] * np.exp(-(E - s["mass"]) / 1.0)[None, :])   # rest mass subtracted
        name = "cfg2: e-/H+ screened Coulomb" if cfg == 2 else "cfg5: e-/H+ fused Euler update, fp32 kinematics"
        if cfg == 5:
            dt, fp32 = 1e-3, True
    elif cfg == 3:
        nxd, N, side = 64, 1024, 20
        nx = nxd if nx is None else nx
        side = side if np_side is None else np_side
        masses = [0.05, 0.05, 0.2, 0.01, 0.5]
        stats = [-1, -1, -1, 1, 1]
        species = [dict(mass=m, charge=0.0, stat=st, g=1.0) for m, st in zip(masses, stats)]
        grids = [_grid(side, -3.0, 3.0) for _ in masses]
        par = [2.0, 0.6]                                    # g = 2, m_D = g T = 0.6
        pairs = [(0, 0), (1, 1), (2, 2), (3, 3), (0, 1), (0, 2), (0, 3), (2, 4)]
        procs = [_elastic(a, b, KIND_TCHAN_S2, par) for a, b in pairs]
        kappa = (2.0 * np.pi) ** 3                          # (2 pi hbar)^3 / g, hbar = g = 1
        fs = []
        for s, g in zip(species, grids):
            P = cell_centres(g)
            pabs = np.sqrt((P * P).sum(1))
            E = np.sqrt(pabs ** 2 + s["mass"] ** 2)
            nbar = equilibrium_nbar(E, 0.3, s["stat"])
            aniso = 1.0 + 0.2 * (P[:, 2] / pabs)[None, :] * (2.0 * rng.random((nx, P.shape[0])) - 1.0)
            fs.append(nbar[None, :] / kappa * aniso)
        name = "cfg3: 3 fermions + 2 bosons, t-channel g^4 s^2/(t-mD^2)^2"
    elif cfg == 4:
        nxd, N, side = 32 ** 3, 512, 20
        nx = nxd if nx is None else nx
        side = side if np_side is None else np_side
        species = [dict(mass=1.0, charge=0.0, stat=0, g=1.0)]
        grids = [_grid(side, -5.0, 5.0)]
        procs = [_elastic(0, 0, KIND_CONST, [1.0])]
        P = cell_centres(grids[0])
        def mj(shift):
            Q = P.copy(); Q[:, 2] -= shift
            return np.exp(-np.sqrt((Q * Q).sum(1) + 1.0) / 0.5)
        prof = 0.5 * (mj(2.0) + mj(-2.0))                    # two counter-streaming beams along z
        dens = 1.0 + 0.1 * (2.0 * rng.random(nx) - 1.0)
        fs = [dens[:, None] * prof[None, :]]
        name = "cfg4: 1 classical species, two counter-streaming beams, const |M|^2"
    elif cfg == 6:
        # The paper's own collision test (Eq. 46-48, Fig. 9): two classical species of
        # mass 0.3, 1x1x1 spatial cell, 35^3 momentum cells on [-2,2]^3, step-function input with Q_s = 1,
        # f_0 = 0.2 / 0.4, constant differential cross sections 1 (aa), 20 (bb), 0.01 (ab),
        # dt = 0.0002/0.197, 25 000 steps.  Readings (R17-R19): the cross sections are taken as
        # CM-frame isotropic; the occupied region is |p| < Q_s (Eq. 46-47 print the opposite inequality,
        # which would fill the box to its corners); samples per cell and step are not stated (256 here).
        nxd, N, side = 1, 256, 35
        nx = nxd if nx is None else nx
        side = side if np_side is None else np_side
        species = [dict(mass=0.3, charge=0.0, stat=0, g=1.0), dict(mass=0.3, charge=0.0, stat=0, g=1.0)]
        grids = [_grid(side, -2.0, 2.0), _grid(side, -2.0, 2.0)]
        procs = [_elastic(0, 0, KIND_ISO_DSIGMA, [1.0]), _elastic(1, 1, KIND_ISO_DSIGMA, [20.0]),
                 _elastic(0, 1, KIND_ISO_DSIGMA, [0.01])]
        P = cell_centres(grids[0])
        inside = ((P * P).sum(1) < 1.0).astype(np.float64)
        fs = [np.tile(f0 * inside, (nx, 1)) for f0 in (0.2, 0.4)]
        dt = 0.0002 / 0.197
        name = "cfg6: paper's collision test (Eq. 46-48): 2 classical species m=0.3, const dsigma/dOmega 1/20/0.01"
    else:
        raise ValueError(f"unknown config {cfg}")
    if sampler:
        for p in procs:
            if p["kind"] in (KIND_COULOMB_SCREENED, KIND_TCHAN_S2):
                p["sampler"] = int(sampler)
        name += " [t-channel importance sampler]"
    problem = dict(nx=int(nx), species=species, grids=grids, processes=procs, hbar=1.0)
    f = np.concatenate([np.ascontiguousarray(a, dtype=np.float64).reshape(-1) for a in fs])
    return dict(cfg=cfg, name=name, problem=problem, f=f, n_samples=int(N if n_samples is None else n_samples),
                seed=int(seed), dt=float(dt), fp32=bool(fp32))


def n_roles(problem) -> int:
    return sum(1 if p["a"] == p["b"] else 2 for p in problem["processes"])


def sample_evals(problem, n_samples) -> int:
    """roles * Nx * Np * N: the 'collision samples' one sweep evaluates (BASELINE.json metric)."""
    tot = 0
    for p in problem["processes"]:
        for s in ([p["a"]] if p["a"] == p["b"] else [p["a"], p["b"]]):
            tot += problem["nx"] * int(np.prod(problem["grids"][s]["n"])) * n_samples
    return tot
