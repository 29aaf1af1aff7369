"""P6 / P9: the Monte Carlo oracle against two independent evaluations of the same integral:
the paper's own 5-D form Eq. 37 (oracle/eq37.py) and a deterministic brute-force
quadrature of the reduced form (R) (oracle/quadrature.py).  Analytic-f mode, smooth inputs."""
import math

import numpy as np
import pytest

import oracle
from oracle.eq37 import eq37_mc
from oracle.quadrature import collision_quadrature

KAPPA = (2 * math.pi) ** 3


def thermal_np(row):
    scale, T, mu, m, theta, ux, uy, uz = row

    def f(p):
        q = np.asarray(p, float) - np.array([ux, uy, uz])
        return scale / (np.exp((np.sqrt((q * q).sum(-1) + m * m) - mu) / T) - theta)
    return f


CASES = {
    # name: (masses (a,b), stats, kind, par, rows(a,b))
    "classical_const": ((0.7, 0.7), (0, 0), 0, [1.3],
                        [[0.8, 0.9, 0.0, 0.7, 0, 0.4, 0, -0.3], [0.8, 0.9, 0.0, 0.7, 0, 0.4, 0, -0.3]]),
    "two_species_coulomb": ((0.3, 1.1), (0, 0), 1, [1.0, 0.8],
                            [[0.5, 0.8, 0.0, 0.3, 0, 0.0, 0.3, 0.0], [1.2, 1.1, 0.0, 1.1, 0, -0.4, 0.0, 0.2]]),
    "fermion_boson_tchan": ((0.2, 0.6), (-1, 1), 2, [1.2, 0.7],
                            [[1 / KAPPA, 0.8, 0.1, 0.2, -1, 0.3, 0, 0], [1 / KAPPA, 0.6, -0.3, 0.6, 1, 0, -0.2, 0.3]]),
}


def _setup(name, same_species=False):
    (ma, mb), (sa, sb), kind, par, rows = CASES[name]
    if same_species:
        species = [dict(mass=ma, charge=0, stat=sa, g=1.0)]
        grids = [dict(n=[6] * 3, pmin=[-3.0] * 3, pmax=[3.0] * 3)]
        procs = [dict(a=0, b=0, c=0, d=0, kind=kind, par=par, sym=-1.0)]
        rows = rows[:1]
    else:
        species = [dict(mass=ma, charge=0, stat=sa, g=1.0), dict(mass=mb, charge=0, stat=sb, g=1.0)]
        grids = [dict(n=[6] * 3, pmin=[-3.0] * 3, pmax=[3.0] * 3), dict(n=[4, 5, 6], pmin=[-3.5, -3.0, -2.5], pmax=[3.0, 3.5, 3.5])]
        procs = [dict(a=0, b=1, c=0, d=1, kind=kind, par=par, sym=-1.0)]
    prob = dict(nx=1, species=species, grids=grids, processes=procs, hbar=1.0)
    return prob, rows


def _quad_for_role(o, prob, rows, role, p1, n=(6, 16, 16), panels=4):
    s4 = o.roles[role]["s"]
    masses = [prob["species"][s]["mass"] for s in s4]
    fs = [thermal_np(rows[s]) for s in s4]
    tk = [prob["species"][s]["stat"] * KAPPA for s in s4]
    g2 = prob["grids"][s4[1]]
    pr = prob["processes"][o.roles[role]["process"]]
    return collision_quadrature(p1, masses, fs, tk, pr["kind"], pr["par"], o.roles[role]["sym"],
                                (g2["pmin"], g2["pmax"]), *n, panels=panels), (masses, fs, tk, g2, pr)


@pytest.mark.parametrize("name,same", [("classical_const", True), ("two_species_coulomb", False),
                                       ("fermion_boson_tchan", False)])
def test_p9_monte_carlo_converges_to_brute_force_quadrature(name, same):
    prob, rows = _setup(name, same)
    o = oracle.Oracle(prob)
    fcb = ("thermal", rows)
    for role in range(o.n_roles):
        ip1 = 4 * 36 + 2 * 6 + 3 if o.np[o.roles[role]["s"][0]] == 216 else 50
        p1 = o.trace(None, role, 0, ip1, 0, 1, fcb=fcb, box_cut=False)["p1"]
        (Cq, Gq, Lq), _ = _quad_for_role(o, prob, rows, role, p1)
        (Cq2, Gq2, Lq2), _ = _quad_for_role(o, prob, rows, role, p1, n=(5, 14, 14), panels=4)
        assert abs(Gq - Gq2) < 2e-3 * Gq and abs(Lq - Lq2) < 2e-3 * Lq      # quadrature itself converged
        N = 1 << 20
        G, L, Lin, Q = o.point(None, role, 0, ip1, N, 2468, fcb=fcb, box_cut=False)
        se = math.sqrt(max(Q - (G - L) ** 2 / N, 0.0))
        assert abs((G - L) - Cq) < 4 * se + 2e-3 * abs(Cq) + 2e-4 * Lq, (G - L, Cq, se)
        assert abs(G - Gq) < 0.01 * Gq and abs(L - Lq) < 0.01 * Lq, (G, Gq, L, Lq)
        assert abs(G - L) > 5 * se          # the case really is off equilibrium


def test_p9_error_decays_like_inverse_sqrt_n():
    prob, rows = _setup("classical_const", True)
    o = oracle.Oracle(prob)
    fcb = ("thermal", rows)
    ip1 = 4 * 36 + 2 * 6 + 3
    p1 = o.trace(None, 0, 0, ip1, 0, 1, fcb=fcb, box_cut=False)["p1"]
    (Cq, Gq, Lq), _ = _quad_for_role(o, prob, rows, 0, p1, n=(6, 16, 16), panels=5)
    Ns = [1 << k for k in (8, 10, 12, 14, 16)]
    rms = []
    for N in Ns:
        err = [o.point(None, 0, 0, ip1, N, 1000 + 17 * j, fcb=fcb, box_cut=False)[1] - Lq for j in range(24)]
        rms.append(math.sqrt(np.mean(np.square(err))))
    slope = np.polyfit(np.log(Ns), np.log(rms), 1)[0]
    assert -0.62 < slope < -0.38, (slope, rms)
    assert rms[-1] < 0.01 * Lq


@pytest.mark.parametrize("name,same", [("classical_const", True), ("fermion_boson_tchan", False)])
def test_p6_reduced_form_equals_papers_eq37(name, same):
    """(R) sampled by the oracle == Eq. 37 sampled by oracle/eq37.py, both by Monte Carlo."""
    prob, rows = _setup(name, same)
    o = oracle.Oracle(prob)
    fcb = ("thermal", rows)
    role = 0
    ip1 = 4 * 36 + 2 * 6 + 3
    p1 = o.trace(None, role, 0, ip1, 0, 1, fcb=fcb, box_cut=False)["p1"]
    _, (masses, fs, tk, g2, pr) = _quad_for_role(o, prob, rows, role, p1, n=(2, 4, 4), panels=1)
    runs = np.array([o.point(None, role, 0, ip1, 1 << 17, 97 + 13 * j, fcb=fcb, box_cut=False)[:2] for j in range(8)])
    G, L = runs.mean(0)
    seG, seL = runs.std(0, ddof=1) / math.sqrt(len(runs))
    (g37, sg37), (l37, sl37) = eq37_mc(p1, masses, fs, tk, pr["kind"], pr["par"], o.roles[role]["sym"],
                                       (g2["pmin"], g2["pmax"]), 3_000_000, np.random.default_rng(5))
    assert math.hypot(seG, sg37) < 0.02 * G and math.hypot(seL, sl37) < 0.02 * L
    assert abs(G - g37) < 4 * math.hypot(seG, sg37), (G, seG, g37, sg37)
    assert abs(L - l37) < 4 * math.hypot(seL, sl37), (L, seL, l37, sl37)
    assert abs(G - L) > 0.01 * L                        # off equilibrium: the two brackets differ
