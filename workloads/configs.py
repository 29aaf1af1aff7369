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
# Table III of the paper, par = [g, m_g]
(KIND_QCD_Q1Q2, KIND_QCD_Q1Q1, KIND_QCD_Q1QB1, KIND_QCD_Q1QB1_Q2QB2, KIND_QCD_QQB_GG, KIND_QCD_QG,
 KIND_QCD_GG) = 4, 5, 6, 7, 8, 9, 10

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


def _process(a, b, c, d, kind, par):
    return dict(a=a, b=b, c=c, d=d, kind=kind, par=list(par), sym=-1.0)


def qgp_processes(par, n_flavours=3):
    """Every row of Table III among n_flavours quarks (species 0..nf-1), their antiquarks
    (nf..2nf-1) and the gluon (2nf): "seven particle species ... u, d, and s quarks, their anti-quarks, and gluons"
    (PAPER.md:510).  With 3 flavours: 34 processes, 70 roles."""
    nf = n_flavours
    q, qb, G = list(range(nf)), list(range(nf, 2 * nf)), 2 * nf
    procs = []
    for i in range(nf):
        for j in range(i + 1, nf):
            procs.append(_elastic(q[i], q[j], KIND_QCD_Q1Q2, par))
            procs.append(_elastic(qb[i], qb[j], KIND_QCD_Q1Q2, par))
        for j in range(nf):
            if j != i:
                procs.append(_elastic(q[i], qb[j], KIND_QCD_Q1Q2, par))
    for i in range(nf):
        procs.append(_elastic(q[i], q[i], KIND_QCD_Q1Q1, par))
        procs.append(_elastic(qb[i], qb[i], KIND_QCD_Q1Q1, par))
        procs.append(_elastic(q[i], qb[i], KIND_QCD_Q1QB1, par))
    for i in range(nf):
        for j in range(i + 1, nf):
            procs.append(_process(q[i], qb[i], q[j], qb[j], KIND_QCD_Q1QB1_Q2QB2, par))
    for i in range(nf):
        procs.append(_process(q[i], qb[i], G, G, KIND_QCD_QQB_GG, par))
    for i in range(nf):
        procs.append(_elastic(q[i], G, KIND_QCD_QG, par))
        procs.append(_elastic(qb[i], G, KIND_QCD_QG, par))
    procs.append(_elastic(G, G, KIND_QCD_GG, par))
    return procs


NOMINAL_NX = {1: 1, 2: 8 ** 3, 3: 4 ** 3, 4: 32 ** 3, 5: 16 ** 3, 6: 1, 7: 21 ** 3}


def make(cfg: int, nx: int | None = None, n_samples: int | None = None, np_side: int | None = None,
         sampler: int = 0, cells: tuple | None = None):
    """Return dict(name, problem, f, n_samples, seed, dt, fp32, ix_offset, nx_global).  ``nx``/``n_samples``/``np_side``
    override the config's spatial cell count / sample count / momentum cells per axis (tests use
    reduced sizes; bench.py uses the defaults).  ``sampler`` = 1 asks for the t-channel importance
    sampler on every process whose |M|^2 kind has the t-channel shape (configs 2, 3, 5).
    ``cells`` = (lo, hi) builds only spatial cells [lo, hi) of the workload (a rank's shard): the
    per-cell random numbers are drawn for the whole domain and sliced, so the shards of any partition concatenate to
    the unsharded f bit for bit; problem["nx"] is then hi - lo and ix_offset = lo."""
    rng = np.random.Generator(np.random.PCG64(INPUT_SEED_BASE + cfg))
    nx_all = NOMINAL_NX[cfg] if nx is None else int(nx)
    lo, hi = (0, nx_all) if cells is None else (int(cells[0]), int(cells[1]))
    if not (0 <= lo < hi <= nx_all):
        raise ValueError(f"cells {cells} outside [0, {nx_all})")
    sl = slice(lo, hi)
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
        f = np.exp(-E / 1.0)[None, :] * (1.0 + 0.1 * (2.0 * rng.random((nx, P.shape[0]))[sl] - 1.0))
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
            dens = 1.0 + 0.1 * (2.0 * rng.random(nx)[sl] - 1.0)      # seeded density perturbation n(x)
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
            aniso = 1.0 + 0.2 * (P[:, 2] / pabs)[None, :] * (2.0 * rng.random((nx, P.shape[0]))[sl] - 1.0)
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
        dens = 1.0 + 0.1 * (2.0 * rng.random(nx)[sl] - 1.0)
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
        fs = [np.tile(f0 * inside, (hi - lo, 1)) for f0 in (0.2, 0.4)]
        dt = 0.0002 / 0.197
        name = "cfg6: paper's collision test (Eq. 46-48): 2 classical species m=0.3, const dsigma/dOmega 1/20/0.01"
    elif cfg == 7:
        # The paper's multi-GPU performance scenario (Table II :484-491): quark-gluon plasma, seven
        # species (u, d, s, their antiquarks, gluons), every process of Table III, the recommended per-run grid
        # 21^3 spatial x 11^3 momentum cells.  Not in BASELINE.json (NEXT-2(ii)).  The paper gives no masses, coupling,
        # regulator, box or initial state for that run (reading R22): quarks m = 0.3, 0.3, 0.45 with g = 6
        # (Fermi-Dirac), gluon m = 0.5 with g = 16 (Bose-Einstein), coupling 2, regulator m_g = 0.8,
        # box [-2,2]^3, hbar = 1, f = nbar/kappa at T = 0.4 with a seeded anisotropy and the gluons under-populated
        # by a factor 1/2 (so that q qbar <-> g g has a net rate); 256 samples per cell and role.
        nxd, N, side = 21 ** 3, 256, 11
        nx = nxd if nx is None else nx
        side = side if np_side is None else np_side
        masses = [0.3, 0.3, 0.45, 0.3, 0.3, 0.45, 0.5]
        stats = [-1] * 6 + [1]
        gs = [6.0] * 6 + [16.0]
        species = [dict(mass=m, charge=0.0, stat=st, g=g) for m, st, g in zip(masses, stats, gs)]
        grids = [_grid(side, -2.0, 2.0) for _ in masses]
        procs = qgp_processes([2.0, 0.8])
        fs = []
        for s, g in zip(species, grids):
            P = cell_centres(g)
            E = np.sqrt((P * P).sum(1) + s["mass"] ** 2)
            kappa = (2.0 * np.pi) ** 3 / s["g"]
            nbar = equilibrium_nbar(E, 0.4, s["stat"]) * (0.5 if s["stat"] == 1 else 1.0)
            aniso = 1.0 + 0.2 * (P[:, 2] / E)[None, :] * (2.0 * rng.random((nx, P.shape[0]))[sl] - 1.0)
            fs.append(nbar[None, :] / kappa * aniso)
        name = "cfg7: quark-gluon plasma, 7 species, all Table III processes (34 processes, 70 roles)"
    else:
        raise ValueError(f"unknown config {cfg}")
    if sampler:
        for p in procs:
            if p["kind"] in (KIND_COULOMB_SCREENED, KIND_TCHAN_S2):
                p["sampler"] = int(sampler)
        name += " [t-channel importance sampler]"
    problem = dict(nx=int(hi - lo), species=species, grids=grids, processes=procs, hbar=1.0)
    f = np.concatenate([np.ascontiguousarray(a, dtype=np.float64).reshape(-1) for a in fs])
    return dict(cfg=cfg, name=name, problem=problem, f=f, n_samples=int(N if n_samples is None else n_samples),
                seed=int(seed), dt=float(dt), fp32=bool(fp32), ix_offset=int(lo), nx_global=int(nx_all))


def roles(problem):
    """(s1, s2, s3, s4) of every role, in role order: a + b -> c + d is seen from a, from b (if
    b != a) and, if it is inelastic, from c and from d (if d != c)."""
    out = []
    for p in problem["processes"]:
        a, b, c, d = p["a"], p["b"], p["c"], p["d"]
        out.append((a, b, c, d))
        if b != a:
            out.append((b, a, d, c))
        if not (c == a and d == b):
            out.append((c, d, a, b))
            if d != c:
                out.append((d, c, b, a))
    return out


def role_processes(problem):
    """The process each role comes from, in role order."""
    out = []
    for p in problem["processes"]:
        a, b, c, d = p["a"], p["b"], p["c"], p["d"]
        out += [p] * ((1 if b == a else 2) + (0 if (c == a and d == b) else (1 if d == c else 2)))
    return out


def n_roles(problem) -> int:
    return len(roles(problem))


def sample_evals(problem, n_samples) -> int:
    """roles * Nx * Np * N: the 'collision samples' one sweep evaluates (BASELINE.json metric)."""
    return sum(problem["nx"] * int(np.prod(problem["grids"][r[0]]["n"])) * n_samples for r in roles(problem))
