"""P15-P17: Table III matrix elements and inelastic roles (Eq. 16 with c,d != a,b).

P15  the |M|^2 kinds against textbook values (tests/golden/qcd_90deg.txt), crossing symmetry, the small-angle
     colour factors, and the regulator limits; the sample loop uses them with the sample's own (s,t,u).
P16  inelastic roles: role list and symmetry factors, per-sample kinematics with four different masses
     (on-shell, energy conservation, threshold), exact detailed balance at equilibrium, brute-force quadrature.
P17  bookkeeping across species for q qbar <-> g g: dn_g/dt = -2 dn_q/dt and energy conservation.
"""
import math

import numpy as np
import pytest

import oracle
from oracle.quadrature import collision_quadrature
from conftest import read_golden

K = dict(Q1Q2=4, Q1Q1=5, Q1QB1=6, Q1QB1_Q2QB2=7, QQB_GG=8, QG=9, GG=10)


def _problem(masses, procs, n=8, lo=-3.0, hi=3.0, stats=None, gs=None, hbar=1.0):
    ns = len(masses)
    stats = stats or [0] * ns
    gs = gs or [1.0] * ns
    return dict(nx=1, species=[dict(mass=m, charge=0, stat=st, g=g) for m, st, g in zip(masses, stats, gs)],
                grids=[dict(n=[n] * 3, pmin=[lo] * 3, pmax=[hi] * 3) for _ in range(ns)], processes=procs, hbar=hbar)


def _proc(a, b, c, d, kind, par=(1.0, 0.0), sym=-1.0):
    return dict(a=a, b=b, c=c, d=d, kind=kind, par=list(par), sym=sym)


def _m2(kind, s, t, u, g=1.0, mg=0.0):
    """First role of a one-process problem of that kind (species content does not enter |M|^2)."""
    o = oracle.Oracle(_problem([0.0, 0.0, 0.0], [_proc(0, 1, 0, 1, kind, (g, mg))]))
    return o.m2_qcd(0, s, t, u)


# ------------------------------------------------------------------------------------------ P15
def test_p15_textbook_values_at_90_degrees():
    gold = {k: float(v) for k, v in read_golden("qcd_90deg.txt").items()}
    s = 7.3
    t = u = -s / 2
    q, g = 6.0, 16.0
    got = dict(q1q2_q1q2=_m2(K["Q1Q2"], s, t, u) / (q * q), q1q1_q1q1=_m2(K["Q1Q1"], s, t, u) / (q * q),
               q1qb1_q2qb2=_m2(K["Q1QB1_Q2QB2"], s, t, u) / (q * q), q1qb1_q1qb1=_m2(K["Q1QB1"], s, t, u) / (q * q),
               q1qb1_gg=_m2(K["QQB_GG"], s, t, u) / (q * q), gg_q1qb1=_m2(K["QQB_GG"], s, t, u) / (g * g),
               q1g_q1g=_m2(K["QG"], s, t, u) / (q * g), gg_gg=_m2(K["GG"], s, t, u) / (g * g))
    for k, v in got.items():
        tol = 0.051 if k == "gg_gg" else 0.0051          # the table prints 3 significant digits
        assert abs(v - gold[k]) < tol, (k, v, gold[k])


def test_p15_g4_scaling_and_homogeneity():
    s, t = 5.0, -1.2
    u = -s - t
    for k in K.values():
        a = _m2(k, s, t, u, g=1.0)
        assert _m2(k, s, t, u, g=1.7) == pytest.approx(a * 1.7 ** 4, rel=1e-13)
        assert _m2(k, 3 * s, 3 * t, 3 * u) == pytest.approx(a, rel=1e-13)      # dimensionless without a regulator


def test_p15_crossing_symmetry():
    rng = np.random.default_rng(5)
    for _ in range(50):
        s = rng.uniform(0.5, 20.0)
        t = -s * rng.uniform(0.02, 0.98)
        u = -s - t
        # q1 qb1 -> q2 qb2 is q1 q2 -> q1 q2 with s <-> t
        assert _m2(K["Q1QB1_Q2QB2"], s, t, u) == pytest.approx(_m2(K["Q1Q2"], t, s, u), rel=1e-12)
        # q1 qb1 -> q1 qb1 is q1 q1 -> q1 q1 with s <-> u
        assert _m2(K["Q1QB1"], s, t, u) == pytest.approx(_m2(K["Q1Q1"], u, t, s), rel=1e-12)
        # q g -> q g is q qb -> g g with s <-> t and an overall sign (one fermion line crossed)
        assert _m2(K["QG"], s, t, u) == pytest.approx(-_m2(K["QQB_GG"], t, s, u), rel=1e-12)
        # identical particles: q1 q1 and q qb -> g g are t <-> u symmetric, g g -> g g fully symmetric
        assert _m2(K["Q1Q1"], s, t, u) == pytest.approx(_m2(K["Q1Q1"], s, u, t), rel=1e-12)
        assert _m2(K["QQB_GG"], s, t, u) == pytest.approx(_m2(K["QQB_GG"], s, u, t), rel=1e-12)
        for perm in ((s, u, t), (t, s, u), (u, t, s), (t, u, s)):
            assert _m2(K["GG"], s, t, u) == pytest.approx(_m2(K["GG"], *perm), rel=1e-12)
        # every physical-region value is positive
        for k in K.values():
            assert _m2(k, s, t, u) > 0


def test_p15_small_angle_colour_factors():
    gold = {k: float(v) for k, v in read_golden("qcd_90deg.txt").items()}
    s, t = 10.0, -1e-5
    u = -s - t
    lim = lambda k, dof: _m2(k, s, t, u) / dof * t * t / (2 * s * s)
    assert lim(K["Q1Q2"], 36.0) == pytest.approx(gold["small_angle_qq"], rel=1e-4)
    assert lim(K["Q1Q1"], 36.0) == pytest.approx(gold["small_angle_qq"], rel=1e-4)
    assert lim(K["Q1QB1"], 36.0) == pytest.approx(gold["small_angle_qq"], rel=1e-4)
    assert lim(K["QG"], 96.0) == pytest.approx(gold["small_angle_qg"], rel=1e-4)
    assert lim(K["GG"], 256.0) == pytest.approx(gold["small_angle_gg"], rel=1e-4)


def test_p15_regulator_sits_in_the_t_and_u_denominators_only():
    s, t = 6.0, -2.5
    u = -s - t
    big = 1e6
    z = lambda k: _m2(k, s, t, u, mg=big)
    # m_g -> infinity removes every t- and u-channel term and leaves the s-channel ones
    assert abs(z(K["Q1Q2"])) < 1e-15 and abs(z(K["Q1Q1"])) < 1e-15
    assert z(K["Q1QB1_Q2QB2"]) == pytest.approx(_m2(K["Q1QB1_Q2QB2"], s, t, u), rel=1e-13)
    assert z(K["Q1QB1"]) == pytest.approx(_m2(K["Q1QB1_Q2QB2"], s, t, u), rel=1e-9)         # A (t^2+u^2)/s^2
    assert z(K["QQB_GG"]) == pytest.approx(-6.0 * _m2(K["Q1QB1_Q2QB2"], s, t, u), rel=1e-9)  # -D/A = -96/16
    assert z(K["QG"]) == pytest.approx(-(128.0 / 3.0) * u / s, rel=1e-9)
    assert z(K["GG"]) == pytest.approx(1152.0 * (3.0 - t * u / (s * s)), rel=1e-9)
    # sign of the regulator: t - m_g^2 never vanishes for t <= 0; at t = 0 the t-channel term is 2 A s^2 / m_g^4
    mg = 0.7
    assert _m2(K["Q1Q2"], s, 0.0, -s, mg=mg) == pytest.approx(2 * 16.0 * s * s / mg ** 4, rel=1e-13)
    # and a regulated value is the unregulated formula with t -> t - m_g^2, u -> u - m_g^2 in the denominators:
    # for the pure t-channel kind the ratio is (t / (t - m_g^2))^2
    assert _m2(K["Q1Q2"], s, t, u, mg=mg) == pytest.approx(_m2(K["Q1Q2"], s, t, u) * (t / (t - mg * mg)) ** 2, rel=1e-13)


def test_p15_sample_loop_uses_the_samples_own_invariants():
    """w = |M|^2 pf / (E2 sqrt s) with (s,t,u) recomputed here from the traced four-momenta."""
    masses = [0.3, 0.5, 0.2]
    for kind in K.values():
        o = oracle.Oracle(_problem(masses, [_proc(0, 1, 0, 1, kind, (1.3, 0.6))], n=6))
        checked = 0
        for n in range(40):
            tr = o.trace(None, 0, 0, 77, n, 99, fcb=lambda s_, p: 1.0, box_cut=False)
            if tr["status"] != 0:
                continue
            m1, m2, m3, m4 = masses[0], masses[1], masses[0], masses[1]
            E = lambda p, m: math.sqrt(p @ p + m * m)
            E1, E2, E3, E4 = E(tr["p1"], m1), E(tr["p2"], m2), E(tr["p3"], m3), E(tr["p4"], m4)
            s = (E1 + E2) ** 2 - np.sum((tr["p1"] + tr["p2"]) ** 2)
            t = (E1 - E3) ** 2 - np.sum((tr["p1"] - tr["p3"]) ** 2)
            u = (E1 - E4) ** 2 - np.sum((tr["p1"] - tr["p4"]) ** 2)
            assert s + t + u == pytest.approx(m1 ** 2 + m2 ** 2 + m3 ** 2 + m4 ** 2, abs=1e-11 * s)
            assert tr["s"] == pytest.approx(s, rel=1e-12) and tr["t"] == pytest.approx(t, abs=1e-12 * s)
            assert tr["u"] == pytest.approx(u, abs=1e-11 * s)
            m2v = tr["w"] * E2 * math.sqrt(s) / tr["pf"]
            assert m2v == pytest.approx(o.m2_qcd(0, s, t, u), rel=1e-9)
            checked += 1
        assert checked > 20


# ------------------------------------------------------------------------------------------ P16
def test_p16_role_expansion_and_symmetry_factors():
    # q(0) qbar(1) -> g(2) g(2)
    o = oracle.Oracle(_problem([0.3, 0.3, 0.5], [_proc(0, 1, 2, 2, K["QQB_GG"])]))
    got = [(r["s"], r["sym"]) for r in o.roles]
    assert got == [((0, 1, 2, 2), 0.5), ((1, 0, 2, 2), 0.5), ((2, 2, 0, 1), 1.0)]
    # the same process written the other way round gives the same set of roles
    o2 = oracle.Oracle(_problem([0.3, 0.3, 0.5], [_proc(2, 2, 0, 1, K["QQB_GG"])]))
    assert sorted((r["s"], r["sym"]) for r in o2.roles) == sorted(got)
    # q1 qb1 -> q2 qb2: four roles, no symmetry factor
    o3 = oracle.Oracle(_problem([0.1, 0.1, 0.2, 0.2], [_proc(0, 1, 2, 3, K["Q1QB1_Q2QB2"])]))
    assert [(r["s"], r["sym"]) for r in o3.roles] == [((0, 1, 2, 3), 1.0), ((1, 0, 3, 2), 1.0), ((2, 3, 0, 1), 1.0),
                                                      ((3, 2, 1, 0), 1.0)]
    # elastic processes keep their two (or one) roles
    o4 = oracle.Oracle(_problem([0.1, 0.2], [_proc(0, 1, 0, 1, 0), _proc(1, 1, 1, 1, 0)]))
    assert [(r["s"], r["sym"]) for r in o4.roles] == [((0, 1, 0, 1), 1.0), ((1, 0, 1, 0), 1.0), ((1, 1, 1, 1), 0.5)]
    # a + b -> b + a is refused (ambiguous t/u labelling): it has to be written a + b -> a + b
    with pytest.raises(ValueError):
        oracle.Oracle(_problem([0.1, 0.2], [_proc(0, 1, 1, 0, 0)]))


def test_p16_inelastic_kinematics_on_shell_and_threshold():
    masses = [0.2, 0.35, 0.9, 1.4]                      # threshold (m3+m4)^2 = 5.29 > (m1+m2)^2
    o = oracle.Oracle(_problem(masses, [_proc(2, 3, 0, 1, 0, (1.0,))], n=6))
    # roles: (2,3,0,1), (3,2,1,0), (0,1,2,3), (1,0,3,2): role 2 has light incoming, heavy outgoing particles
    assert o.roles[2]["s"] == (0, 1, 2, 3)
    n_ok = n_below = 0
    for ip1 in (0, 100, 215):
        for n in range(60):
            tr = o.trace(None, 2, 0, ip1, n, 3, fcb=lambda s_, p: 1.0, box_cut=False)
            E = lambda p, m: math.sqrt(p @ p + m * m)
            E1, E2 = E(tr["p1"], masses[0]), E(tr["p2"], masses[1])
            s = (E1 + E2) ** 2 - np.sum((tr["p1"] + tr["p2"]) ** 2)
            if s <= (masses[2] + masses[3]) ** 2:
                assert tr["status"] == 2 and tr["w"] == 0.0
                n_below += 1
                continue
            assert tr["status"] == 0
            E3, E4 = E(tr["p3"], masses[2]), E(tr["p4"], masses[3])
            assert E3 + E4 == pytest.approx(E1 + E2, rel=1e-13)
            assert np.allclose(tr["p3"] + tr["p4"], tr["p1"] + tr["p2"], atol=1e-13)
            assert tr["E3"] == pytest.approx(E3, rel=1e-13)
            lam = (s - (masses[2] + masses[3]) ** 2) * (s - (masses[2] - masses[3]) ** 2)
            assert tr["pf"] == pytest.approx(math.sqrt(lam) / (2 * math.sqrt(s)), rel=1e-13)
            n_ok += 1
    assert n_ok > 30 and n_below > 10


def test_p16_detailed_balance_for_inelastic_roles():
    """Fermi-Dirac quarks and Bose-Einstein gluons at one temperature, mu = 0: gain = loss sample by sample."""
    T = 0.4
    masses, stats, gs = [0.3, 0.3, 0.5], [-1, -1, 1], [6.0, 6.0, 16.0]
    hbar = 1.0
    prob = _problem(masses, [_proc(0, 1, 2, 2, K["QQB_GG"], (2.0, 0.5))], n=6, lo=-2.0, hi=2.0, stats=stats, gs=gs, hbar=hbar)
    o = oracle.Oracle(prob)
    kap = [(2 * math.pi * hbar) ** 3 / g for g in gs]
    rows = [[1.0 / kap[i], T, 0.0, masses[i], float(stats[i]), 0, 0, 0] for i in range(3)]     # f = nbar / kappa
    for role in range(o.n_roles):
        for ip1 in (5, 100, 215):
            G, L, Lin, Q = o.point(None, role, 0, ip1, 4096, 11, fcb=("thermal", rows), box_cut=False)
            assert L > 0 and abs(G - L) < 1e-12 * (G + L), (role, ip1, G, L)


def test_p16_inelastic_role_converges_to_quadrature():
    """CONST kind, four different masses, non-equilibrium analytic f: the Monte Carlo estimate of (R) against the
    deterministic quadrature (oracle/quadrature.py), which knows nothing of the oracle's chain."""
    masses = [0.4, 0.7, 0.3, 1.1]
    o = oracle.Oracle(_problem(masses, [_proc(0, 1, 2, 3, 0, (2.0,))], n=4, lo=-2.0, hi=2.0))
    T = [0.5, 0.7, 0.6, 0.9]
    shift = [np.array([0.2, 0, 0]), np.array([0, -0.3, 0]), np.array([0, 0, 0.1]), np.zeros(3)]

    def f_species(i):
        return lambda p: 0.7 * np.exp(-np.sqrt(np.sum((p - shift[i]) ** 2, axis=-1) + masses[i] ** 2) / T[i])
    fs_by_species = [f_species(i) for i in range(4)]
    cb = lambda s_, p: float(fs_by_species[s_](np.array(p)))
    for role in (0, 2, 3):
        sl = o.roles[role]["s"]
        ip1 = (1 * 4 + 2) * 4 + 3
        tr = o.trace(None, role, 0, ip1, 0, 1, fcb=cb, box_cut=False)
        Cq, gq, lq = collision_quadrature(tr["p1"], [masses[i] for i in sl], [fs_by_species[i] for i in sl], [0.0] * 4,
                                          0, (2.0,), o.roles[role]["sym"], ([-2.0] * 3, [2.0] * 3), n_p2=10, n_cos=12,
                                          n_phi=12, panels=2)
        vals = np.array([o.point(None, role, 0, ip1, 1 << 15, 500 + i, fcb=cb, box_cut=False) for i in range(8)])
        G, L = vals[:, 0].mean(), vals[:, 1].mean()
        seG, seL = vals[:, 0].std(ddof=1) / math.sqrt(8), vals[:, 1].std(ddof=1) / math.sqrt(8)
        assert abs(G - gq) < 4 * seG + 2e-3 * gq, (role, G, gq, seG)
        assert abs(L - lq) < 4 * seL + 2e-3 * lq, (role, L, lq, seL)


# ------------------------------------------------------------------------------------------ P17
def _species_rates(n, kind, par, gs, N, seed):
    # heavy species at a low temperature: f ~ exp(-m/T - p^2/(2 m T)) is smooth at p = 0 (the midpoint rule over the
    # p1 grid converges fast) and both the quarks and the gluons they make are negligible at the box walls
    # (exp(-(E - m)/T) = 2e-4 at |p| = 3)
    T = 0.25
    masses = [1.0, 1.0, 0.8]
    lo, hi = -3.0, 3.0
    prob = _problem(masses, [_proc(0, 1, 2, 2, kind, par)], n=n, lo=lo, hi=hi, gs=gs)
    o = oracle.Oracle(prob)
    rows = [[1.0, T, 0.0, masses[0], 0.0, 0, 0, 0], [0.8, T, 0.0, masses[1], 0.0, 0, 0, 0],
            [0.1, T, 0.0, masses[2], 0.0, 0, 0, 0]]
    C, d = o.collision(None, N, seed, detail=True, fcb=("thermal", rows), box_cut=False)
    dp3 = ((hi - lo) / n) ** 3
    c = lo + (np.arange(n) + 0.5) * (hi - lo) / n
    PX, PY, PZ = np.meshgrid(c, c, c, indexing="ij")
    p2 = (PX ** 2 + PY ** 2 + PZ ** 2).reshape(-1)
    rate, erate, err = [], [], []
    for s_ in range(3):
        Cs = C[o.sp_off[s_]:o.sp_off[s_] + n ** 3]
        rate.append(Cs.sum() * dp3)
        erate.append((Cs * np.sqrt(p2 + masses[s_] ** 2)).sum() * dp3)
    for r in range(o.n_roles):          # Monte Carlo standard error of the summed rates from the per-cell sums of squares
        sl = slice(o.role_off[r], o.role_off[r] + n ** 3)
        var = np.maximum(d["Q"][sl] - (d["G"][sl] - d["L"][sl]) ** 2 / N, 0.0)
        err.append(math.sqrt(var.sum()) * dp3)
    return rate, erate, max(err)


@pytest.mark.parametrize("kind,par,gs", [(0, (1.0,), [1.0, 1.0, 1.0]), (K["QQB_GG"], (1.0, 0.5), [6.0, 6.0, 16.0])])
def test_p17_number_and_energy_bookkeeping_across_species(kind, par, gs):
    """q qbar <-> g g out of chemical equilibrium (too few gluons): every reaction removes one q, one qbar and
    makes two gluons, so dn_g/dt = -2 dn_q/dt = -2 dn_qbar/dt, and the energy the quarks lose the gluons gain.
    Analytic f (no box cut).  The p1 sums are midpoint rules on the grid and the p2 integrals Monte Carlo over the
    box, so the balance holds up to the Monte Carlo error plus a small quadrature error.  A wrong symmetry factor or
    DOF factor would be a factor-2 (or 256/36) violation."""
    rate, erate, err = _species_rates(10, kind, par, gs, 4096, 31)
    assert rate[0] < 0 and rate[1] < 0 and rate[2] > 0
    scale = abs(rate[2])
    assert err < 1e-2 * scale
    tol = 4 * err + 3e-3 * scale
    assert abs(rate[0] - rate[1]) < tol, (rate, err)
    assert abs(rate[2] + 2 * rate[0]) < tol, (rate, err)
    assert abs(erate[0] + erate[1] + erate[2]) < 3 * tol * 1.5, (erate, err)


def test_p17_table3_kinds_are_summed_over_all_degrees_of_freedom():
    """Loss rate of an elastic Table III role with classical statistics scales as 1 / (g1 g2) (reading R21)."""
    L = []
    for gs in ([1.0, 1.0], [6.0, 16.0]):
        o = oracle.Oracle(_problem([0.2, 0.3], [_proc(0, 1, 0, 1, K["QG"], (1.5, 0.4))], n=6, gs=gs))
        L.append(o.point(None, 0, 0, 100, 4096, 5, fcb=lambda s_, p: 1.0, box_cut=False)[1])
    assert L[1] == pytest.approx(L[0] / 96.0, rel=1e-13)
    # kinds 0..3 are not rescaled for elastic roles
    L = []
    for gs in ([1.0, 1.0], [6.0, 16.0]):
        o = oracle.Oracle(_problem([0.2, 0.3], [_proc(0, 1, 0, 1, 2, (1.5, 0.4))], n=6, gs=gs))
        L.append(o.point(None, 0, 0, 100, 4096, 5, fcb=lambda s_, p: 1.0, box_cut=False)[1])
    assert L[1] == L[0]
