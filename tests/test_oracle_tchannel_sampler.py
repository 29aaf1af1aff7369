"""Pins of the t-channel importance sampler (sampler = 1, steps S1..S7 of oracle/rbg_oracle.cpp; DESIGN.md
section 4b): the CM polar angle about the direction of particle 1 is drawn from the shape 1/(t - mD^2)^2 of the
screened t-channel matrix elements (Table III form) by its inverse CDF.  It must estimate the
same integral (R) as the uniform sampler -- Eq. 16 -- only with less variance."""
import math

import numpy as np
import pytest
from scipy import integrate, stats

import oracle
from oracle.quadrature import collision_quadrature
from test_oracle_integral import CASES, KAPPA, thermal_np


def _problem(ma, mb, sa, sb, kind, par, sampler, same=False, n=6, box=3.0):
    if same:
        species = [dict(mass=ma, charge=0, stat=sa, g=1.0)]
        grids = [dict(n=[n] * 3, pmin=[-box] * 3, pmax=[box] * 3)]
        procs = [dict(a=0, b=0, c=0, d=0, kind=kind, par=par, sym=-1.0, sampler=sampler)]
    else:
        species = [dict(mass=ma, charge=0, stat=sa, g=1.0), dict(mass=mb, charge=0, stat=sb, g=1.0)]
        grids = [dict(n=[n] * 3, pmin=[-box] * 3, pmax=[box] * 3),
                 dict(n=[4, 5, 6], pmin=[-3.5, -3.0, -2.5], pmax=[3.0, 3.5, 3.5])]
        procs = [dict(a=0, b=1, c=0, d=1, kind=kind, par=par, sym=-1.0, sampler=sampler)]
    return dict(nx=1, species=species, grids=grids, processes=procs, hbar=1.0)


def _to_cm(p, E, P, Et, rs):
    """Textbook boost of (E, p) into the rest frame of (Et, P)."""
    beta = P / Et
    gamma = Et / rs
    bp = float(beta @ p)
    return p + ((gamma - 1.0) * bp / float(beta @ beta) - gamma * E) * beta


@pytest.mark.parametrize("use_float,tol", [(False, 1e-12), (True, 2e-5)])
def test_per_sample_kinematics_and_angle_distribution(use_float, tol):
    ma, mb, mD = 0.3, 1.1, 0.25
    prob = _problem(ma, mb, 0, 0, 1, [1.0, mD], 1)
    o = oracle.Oracle(prob, use_float=use_float)
    rows = [[0.5, 0.8, 0.0, ma, 0, 0, 0, 0], [1.2, 1.1, 0.0, mb, 0, 0, 0, 0]]
    fcb = ("thermal", rows)
    for role, (m1, m2) in ((0, (ma, mb)), (1, (mb, ma))):
        us, perp = [], []
        for n in range(1500):
            tr = o.trace(None, role, 0, 77, n, 31, fcb=fcb, box_cut=False)
            assert tr["status"] == 0
            p1, p2, p3, p4 = tr["p1"], tr["p2"], tr["p3"], tr["p4"]
            E1, E2 = math.sqrt(p1 @ p1 + m1 * m1), math.sqrt(p2 @ p2 + m2 * m2)
            E3, E4 = math.sqrt(p3 @ p3 + m1 * m1), math.sqrt(p4 @ p4 + m2 * m2)
            s = (E1 + E2) ** 2 - (p1 + p2) @ (p1 + p2)
            scale = max(E1 + E2, 1.0)
            assert np.allclose(p3 + p4, p1 + p2, atol=tol * scale)
            assert abs(E3 + E4 - E1 - E2) < 20 * tol * scale ** 2
            assert abs(tr["E3"] - E3) < 20 * tol * scale ** 2
            assert abs(tr["s"] - s) < 20 * tol * scale ** 2
            # the sampled t = -2 pf^2 (1 - cos) is the lab-frame t = (p1 - p3)^2
            t_lab = (E1 - E3) ** 2 - (p1 - p3) @ (p1 - p3)
            assert abs(tr["t"] - t_lab) < 50 * tol * scale ** 2, (tr["t"], t_lab)
            # weight: |M|^2 pf / (E2 sqrt s) times D^2 / (mD^2 (mD^2 + 4 pf^2)) -- no angle left in it
            q = tr["pf"] ** 2
            assert tr["w"] == pytest.approx(tr["pf"] / (E2 * math.sqrt(s)) / (mD * mD * (mD * mD + 4 * q)), rel=200 * tol)
            om = -tr["t"] / (2 * q)
            us.append(om * (mD * mD + 4 * q) / (2 * (mD * mD + 2 * q * om)))      # CDF of the t-channel shape
            # azimuth about the CM direction of particle 1: unit vector of p3* perpendicular to p1*
            P, Et, rs = p1 + p2, E1 + E2, math.sqrt(s)
            a1, a3 = _to_cm(p1, E1, P, Et, rs), _to_cm(p3, E3, P, Et, rs)
            assert abs(math.sqrt(a3 @ a3) - tr["pf"]) < 50 * tol * scale
            e = a1 / math.sqrt(a1 @ a1)
            pr = a3 - (a3 @ e) * e
            perp.append(pr / math.sqrt(pr @ pr))
        assert stats.kstest(us, "uniform").pvalue > 1e-3
        perp = np.array(perp)
        assert np.all(np.abs(perp.mean(0)) < 4.5 / math.sqrt(len(perp)))


@pytest.mark.parametrize("name", ["two_species_coulomb", "fermion_boson_tchan"])
def test_importance_sampled_estimator_converges_to_brute_force_quadrature(name):
    (ma, mb), (sa, sb), kind, par, rows = CASES[name]
    prob = _problem(ma, mb, sa, sb, kind, par, 1)
    o = oracle.Oracle(prob)
    fcb = ("thermal", rows)
    for role in range(o.n_roles):
        ip1 = 4 * 36 + 2 * 6 + 3 if o.np[o.roles[role]["s"][0]] == 216 else 50
        p1 = o.trace(None, role, 0, ip1, 0, 1, fcb=fcb, box_cut=False)["p1"]
        s4 = o.roles[role]["s"]
        masses = [prob["species"][s]["mass"] for s in s4]
        fs = [thermal_np(rows[s]) for s in s4]
        tk = [prob["species"][s]["stat"] * KAPPA for s in s4]
        g2 = prob["grids"][s4[1]]
        Cq, Gq, Lq = collision_quadrature(p1, masses, fs, tk, kind, par, o.roles[role]["sym"], (g2["pmin"], g2["pmax"]),
                                          6, 16, 16, panels=4)
        N = 1 << 19
        G, L, Lin, Q = o.point(None, role, 0, ip1, N, 1357, fcb=fcb, box_cut=False)
        se = math.sqrt(max(Q - (G - L) ** 2 / N, 0.0))
        assert abs((G - L) - Cq) < 4 * se + 2e-3 * abs(Cq) + 2e-4 * Lq, (G - L, Cq, se)
        assert abs(G - Gq) < 0.01 * Gq and abs(L - Lq) < 0.01 * Lq, (G, Gq, L, Lq)


def _coulomb_loss_rate(p1, m1, m2, T, par0, mD):
    """Int d3p2 f2 [Int dOmega* |M|^2] pf / (64 pi^2 E1 E2 sqrt s) with the angular integral done analytically:
    Int dOmega* par0 / (mD^2 + 2 pf^2 (1 - cos))^2 = 4 pi par0 / (mD^2 (mD^2 + 4 pf^2))."""
    a1 = math.sqrt(p1 @ p1)
    E1 = math.sqrt(a1 * a1 + m1 * m1)

    def integrand(c, q):
        E2 = math.sqrt(q * q + m2 * m2)
        s = m1 * m1 + m2 * m2 + 2 * (E1 * E2 - a1 * q * c)
        pf2 = max((s - (m1 + m2) ** 2) * (s - (m1 - m2) ** 2), 0.0) / (4 * s)
        ang = 4 * math.pi * par0 / (mD * mD * (mD * mD + 4 * pf2))
        return 2 * math.pi * q * q * math.exp(-E2 / T) * ang * math.sqrt(pf2) / (64 * math.pi ** 2 * E1 * E2 * math.sqrt(s))
    return integrate.dblquad(integrand, 0.0, 40.0 * T, -1.0, 1.0, epsabs=1e-13, epsrel=1e-10)[0]


def test_small_screening_mass_loss_rate_and_variance_reduction():
    """mD = 0.1 as in BASELINE config 2: the loss rate against a quadrature whose angular integral is analytic;
    the uniform sampler needs orders of magnitude more samples for the same error."""
    m, T, mD = 1.0, 0.8, 0.1
    errs = {}
    for sampler in (1, 0):
        prob = _problem(m, m, 0, 0, 1, [1.0, mD], sampler, same=True, n=120, box=12.0)
        prob["processes"][0]["sym"] = 1.0
        o = oracle.Oracle(prob)
        thermal = ("thermal", [[1.0, T, 0.0, m, 0.0, 0, 0, 0]])
        ip1 = (61 * 120 + 56) * 120 + 65
        tr = o.trace(None, 0, 0, ip1, 0, 1, fcb=thermal, box_cut=False)
        ref = _coulomb_loss_rate(tr["p1"], m, m, T, 1.0, mD) * tr["f1"]
        Ls = np.array([o.point(None, 0, 0, ip1, 1 << 18, 50 + 7 * i, fcb=thermal, box_cut=False)[1] for i in range(16)])
        errs[sampler] = Ls.std(ddof=1)
        if sampler == 1:
            se = Ls.std(ddof=1) / 4
            assert se < 0.02 * ref
            assert abs(Ls.mean() - ref) < 4 * se + 1e-3 * ref, (Ls.mean(), ref, se)
    assert errs[0] > 5 * errs[1], errs


def test_grid_mode_agrees_with_the_uniform_sampler_within_the_monte_carlo_error():
    import workloads
    w = workloads.make(2, nx=1, np_side=6, n_samples=1 << 15)
    for p in w["problem"]["processes"]:
        p["par"] = [1.0, 1.5]                     # a screening mass the uniform sampler can resolve
    C = {}
    for sampler in (0, 1):
        prob = dict(w["problem"], processes=[dict(p, sampler=sampler) for p in w["problem"]["processes"]])
        o = oracle.Oracle(prob)
        Cs, d = o.collision(w["f"], w["n_samples"], w["seed"], detail=True)
        var = np.zeros_like(Cs)
        for r in range(o.n_roles):
            s1 = o.roles[r]["s"][0]
            n = o.np[s1]
            sl = slice(o.role_off[r], o.role_off[r] + n)
            c_r = d["G"][sl] - d["L"][sl]
            var[o.sp_off[s1]:o.sp_off[s1] + n] += np.maximum(d["Q"][sl] - c_r ** 2 / w["n_samples"], 0.0)
        C[sampler] = (Cs, var)
    diff = C[0][0] - C[1][0]
    sig = np.sqrt(C[0][1] + C[1][1])
    m = sig > 0
    z = diff[m] / sig[m]
    assert np.sqrt(np.mean(z ** 2)) < 1.3 and np.max(np.abs(z)) < 5.5, (np.sqrt(np.mean(z ** 2)), np.max(np.abs(z)))
    assert np.mean(C[1][1][m]) < np.mean(C[0][1][m])


def test_sampler_argument_checks():
    with pytest.raises(ValueError):
        oracle.Oracle(_problem(1.0, 1.0, 0, 0, 0, [1.0], 1, same=True))          # CONST kind has no t-channel shape
    with pytest.raises(ValueError):
        oracle.Oracle(_problem(1.0, 1.0, 0, 0, 1, [1.0, 0.0], 1, same=True))     # needs a regulator
    with pytest.raises(ValueError):
        oracle.Oracle(_problem(1.0, 1.0, 0, 0, 1, [1.0, 0.1], 2, same=True))
