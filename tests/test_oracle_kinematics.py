"""P2: per-sample kinematic invariants of the oracle's chain (O2-O9), the sampling distributions
(p2 uniform in the box, CM direction uniform on the sphere) and the nearest-cell gather (O10)."""
import math
from fractions import Fraction

import mpmath

mpmath.mp.dps = 40
import numpy as np
import pytest

import oracle

M1, M2 = 0.4, 3.0


def two_species(kind, par, n0=(6, 7, 5), n1=(5, 6, 8)):
    return dict(nx=2,
                species=[dict(mass=M1, charge=0, stat=0, g=1.0), dict(mass=M2, charge=0, stat=0, g=1.0)],
                grids=[dict(n=list(n0), pmin=[-2.0, -1.5, -2.5], pmax=[2.5, 2.0, 2.0]),
                       dict(n=list(n1), pmin=[-6.0, -5.0, -4.0], pmax=[5.0, 6.0, 7.0])],
                processes=[dict(a=0, b=1, c=0, d=1, kind=kind, par=list(par), sym=-1.0)], hbar=1.0)


def mdot(a, b):
    return a[0] * b[0] - a[1:] @ b[1:]


@pytest.mark.parametrize("kind,par", [(0, [1.7]), (1, [1.3, 0.4]), (2, [1.5, 0.7])])
@pytest.mark.parametrize("role", [0, 1])
def test_invariants_every_sample(kind, par, role):
    prob = two_species(kind, par)
    o = oracle.Oracle(prob)
    f = np.random.default_rng(3).random(o.f_elems) + 0.1
    masses = [prob["species"][s]["mass"] for s in o.roles[role]["s"]]
    m1, m2, m3, m4 = masses
    n_ok = 0
    for ip1 in (0, 57, o.np[o.roles[role]["s"][0]] - 1):
        for n in range(60):
            tr = o.trace(f, role, 1, ip1, n, 99)
            if tr["status"] != 0:
                continue
            n_ok += 1
            p1, p2, p3, p4 = tr["p1"], tr["p2"], tr["p3"], tr["p4"]
            E1 = math.sqrt(p1 @ p1 + m1 * m1); E2 = math.sqrt(p2 @ p2 + m2 * m2)
            E3 = math.sqrt(p3 @ p3 + m3 * m3); E4 = math.sqrt(p4 @ p4 + m4 * m4)
            assert tr["E1"] == pytest.approx(E1, rel=1e-14) and tr["E2"] == pytest.approx(E2, rel=1e-14)
            assert tr["E3"] == pytest.approx(E3, rel=1e-12)            # boost formula vs mass shell
            assert E3 + E4 == pytest.approx(E1 + E2, rel=1e-12)        # delta(E), Eq. 17
            assert np.allclose(p3 + p4, p1 + p2, rtol=0, atol=1e-13)   # delta^3
            P1, P2, P3, P4 = (np.array([E, *p]) for E, p in ((E1, p1), (E2, p2), (E3, p3), (E4, p4)))
            s = mdot(P1 + P2, P1 + P2)
            assert tr["s"] == pytest.approx(s, rel=1e-12)
            assert mdot(P3 + P4, P3 + P4) == pytest.approx(s, rel=1e-11)
            t = mdot(P1 - P3, P1 - P3); u = mdot(P1 - P4, P1 - P4)
            assert s + t + u == pytest.approx(m1 ** 2 + m2 ** 2 + m3 ** 2 + m4 ** 2, abs=1e-11 * s)
            pf = math.sqrt((s - (m3 + m4) ** 2) * (s - (m3 - m4) ** 2)) / (2 * math.sqrt(s))
            assert tr["pf"] == pytest.approx(pf, rel=1e-12)
            if kind != 0:
                assert tr["t"] == pytest.approx(t, abs=1e-11 * s)
            M2v = {0: par[0], 1: par[0] / (t - par[-1] ** 2) ** 2 if kind else 0,
                   2: par[0] ** 4 * s * s / (t - par[-1] ** 2) ** 2 if kind else 0}[kind]
            assert tr["w"] == pytest.approx(M2v * pf / (E2 * math.sqrt(s)), rel=1e-9)
    assert n_ok > 150


def test_sampling_distributions():
    prob = two_species(0, [1.0])
    o = oracle.Oracle(prob)
    f = np.ones(o.f_elems)
    g2 = prob["grids"][1]
    lo, hi = np.array(g2["pmin"]), np.array(g2["pmax"])
    nh, p2s = [], []
    for n in range(3000):
        tr = o.trace(f, 0, 0, 100, n, 5)
        assert tr["status"] == 0
        p1, p2, p3 = tr["p1"], tr["p2"], tr["p3"]
        p2s.append(p2)
        # nearest cell of p2 from the test's own arithmetic
        jd = np.floor((p2 - lo) / ((hi - lo) / np.array(g2["n"]))).astype(int)
        assert tr["j2"] == (jd[0] * g2["n"][1] + jd[1]) * g2["n"][2] + jd[2]
        # inverse boost of p3 to the CM frame (textbook form) -> direction
        E1 = math.sqrt(p1 @ p1 + M1 * M1); E2 = math.sqrt(p2 @ p2 + M2 * M2); E3 = math.sqrt(p3 @ p3 + M1 * M1)
        P = p1 + p2; Et = E1 + E2; rs = math.sqrt(Et * Et - P @ P)
        beta = P / Et; gam = Et / rs
        p3s = p3 + beta * gam * (gam / (gam + 1) * (beta @ p3) - E3)
        assert math.sqrt(p3s @ p3s) == pytest.approx(tr["pf"], rel=1e-10)
        nh.append(p3s / tr["pf"])
    nh, p2s = np.array(nh), np.array(p2s)
    N = len(nh)
    assert np.all(np.abs(nh.mean(0)) < 4 * math.sqrt(1 / 3 / N))               # <n> = 0
    cov = nh.T @ nh / N
    assert np.all(np.abs(cov - np.eye(3) / 3) < 4 * math.sqrt(4 / 45 / N) + 1e-3)   # <n_i n_j> = delta/3
    assert abs((nh[:, 2] ** 4).mean() - 0.2) < 0.02                              # <nz^4> = 1/5
    assert np.all(np.abs(p2s.mean(0) - (lo + hi) / 2) < 4 * (hi - lo) / math.sqrt(12 * N))
    assert np.all(np.abs(p2s.var(0) / ((hi - lo) ** 2 / 12) - 1) < 0.1)
    assert np.all(p2s >= lo) and np.all(p2s < hi)


def test_gather_matches_numpy_nearest_cell():
    """O10 against a numpy nearest-cell lookup through the analytic-f callback: same samples, so
    the two runs must agree to rounding.  Non-cubic grids and asymmetric boxes expose any
    transposed stride or swapped axis."""
    prob = two_species(1, [1.0, 0.5])
    o = oracle.Oracle(prob)
    rng = np.random.default_rng(11)
    f = rng.random(o.f_elems) + 0.05
    ix = 1

    def lookup(species, p):
        g = prob["grids"][species]
        lo, hi, n = np.array(g["pmin"]), np.array(g["pmax"]), np.array(g["n"])
        j = np.floor((np.array(p) - lo) * (n / (hi - lo))).astype(int)
        if np.any(j < 0) or np.any(j >= n):
            return 0.0
        return float(f[o.sp_off[species] + ix * o.np[species] + (j[0] * n[1] + j[1]) * n[2] + j[2]])

    for role in (0, 1):
        for ip1 in (3, 101):
            a = o.point(f, role, ix, ip1, 1500, 2024)
            b = o.point(None, role, ix, ip1, 1500, 2024, fcb=lookup, box_cut=True)
            assert np.allclose(a, b, rtol=1e-12, atol=0)
            assert a[0] > 0 and a[1] > a[2] > 0     # some, but not all, losses leave the box


def test_threshold_and_degenerate_samples_contribute_zero():
    # massless species: p2 parallel to p1 is measure-zero, so every sample is valid ...
    prob = dict(nx=1, species=[dict(mass=0.0, charge=0, stat=0, g=1.0)],
                grids=[dict(n=[4, 4, 4], pmin=[-1.0] * 3, pmax=[1.0] * 3)],
                processes=[dict(a=0, b=0, c=0, d=0, kind=0, par=[1.0], sym=-1.0)], hbar=1.0)
    o = oracle.Oracle(prob)
    f = np.ones(o.f_elems)
    st = [o.trace(f, 0, 0, 21, n, 1)["status"] for n in range(200)]
    assert st.count(0) == 200
    # ... and the estimate stays finite
    assert np.all(np.isfinite(o.collision(f, 64, 1)))


def test_direction_against_library_trigonometry():
    """O6: the polynomial, libm-free direction equals
    (sin(theta) cos(phi), sin(theta) sin(phi), cos(theta)) with mpmath's cos/sin (40 digits), for
    cos(theta) = (x3|1) 2^-31 - 1 (odd lattice: never 0 or +-1) and phi = (k + 1/2) 2 pi / 2^24, k from the low bytes of x0..x2
    (float chain), phi = ((k >> 2) + 1/2) 2 pi / 2^22 (double chain v3: the lattice keeps the top 22 bits of k):
    to 4e-16 in double and 3e-7 in float; exactly unit length to rounding; every octant, both ends
    of every octant and the symmetric partner (k -> 2^24 - 1 - k mirrors phi -> -phi exactly)."""
    rng = np.random.default_rng(7)
    ks = [0, 1, 2 ** 21 - 1, 2 ** 21, 2 ** 22 - 1, 2 ** 22, 3 * 2 ** 21, 2 ** 23 - 1, 2 ** 23, 2 ** 24 - 1]
    ks += [int(v) for v in rng.integers(0, 2 ** 24, 400)]
    for k in ks:
        for x3 in [0, 1, 2 ** 31, 2 ** 32 - 1] + [int(v) for v in rng.integers(0, 2 ** 32, 3)]:
            hi = [int(v) << 8 for v in rng.integers(0, 2 ** 24, 3)]          # p2 bits: must not matter
            words = [hi[0] | (k >> 16), hi[1] | ((k >> 8) & 255), hi[2] | (k & 255), x3]
            for use_float, tol in ((False, 4e-16), (True, 3e-7)):
                # 40 digits: no rounding of the angle
                phi = (mpmath.mpf(k) + 0.5) * 2 * mpmath.pi / 2 ** 24 if use_float else (mpmath.mpf(k >> 2) + 0.5) * 2 * mpmath.pi / 2 ** 22
                cphi, sphi = float(mpmath.cos(phi)), float(mpmath.sin(phi))
                ct = ((x3 >> 8) | 1) * 2.0 ** -23 - 1.0 if use_float else (x3 | 1) * 2.0 ** -31 - 1.0
                assert 0.0 < abs(ct) < 1.0
                st = math.sqrt(float(1 - Fraction(ct) ** 2))              # 1 - ct^2 exactly, one rounding
                want = np.array([st * cphi, st * sphi, ct])
                got = oracle.direction(words, use_float)
                assert np.all(np.abs(got - want) <= tol), (k, x3, use_float, got, want)
                assert abs(got @ got - 1.0) <= 4 * tol
                mirror = 2 ** 24 - 1 - k
                wm = [hi[0] | (mirror >> 16), hi[1] | ((mirror >> 8) & 255), hi[2] | (mirror & 255), x3]
                gm = oracle.direction(wm, use_float)
                assert gm[0] == got[0] and gm[1] == -got[1] and gm[2] == got[2]


def test_direction_polynomial_path_against_its_by_eye_twin():
    """O6 once more, in the oracle's own language: direction() (polynomials, octant fold, the 9 + 10-bit angle split of the
    double chain) against direction_by_eye() (the definition of a unit vector with cosl / sinl of the same lattice angle,
    oracle/rbg_oracle.cpp) at the tolerance of the mpmath pin above, 4e-16 in double and 3e-7 in float: every octant
    boundary, both neighbours of each, the ends of the 2^10 blocks of the angle split, and random words."""
    rng = np.random.default_rng(11)
    ks = set()
    for o in range(9):
        for d in (-2, -1, 0, 1, 2):
            ks.add(min(max(o * 2 ** 21 + d, 0), 2 ** 24 - 1))
    for hi in (0, 1, 255, 256, 511):                       # the split a = alpha(hi) + beta(lo): first / last lo of a block
        for lo in (0, 1, 1022, 1023):
            ks.add(((hi << 10) | lo) << 2)
    ks = sorted(ks) + [int(v) for v in rng.integers(0, 2 ** 24, 3000)]
    worst = {False: 0.0, True: 0.0}
    for k in ks:
        for x3 in [0, 1, 2 ** 31 - 1, 2 ** 31, 2 ** 32 - 1, int(rng.integers(0, 2 ** 32))]:
            words = [k >> 16, (k >> 8) & 255, k & 255, x3]
            for use_float, tol in ((False, 4e-16), (True, 3e-7)):
                got, want = oracle.direction(words, use_float), oracle.direction_by_eye(words, use_float)
                err = float(np.max(np.abs(got - want)))
                worst[use_float] = max(worst[use_float], err)
                assert err <= tol, (k, x3, use_float, got, want)
                assert got[2] == want[2]                     # cos(theta) is exact on both paths
    assert worst[False] > 0.0 and worst[True] > 1e-9         # the two paths really are different arithmetic

