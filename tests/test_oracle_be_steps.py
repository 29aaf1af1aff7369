"""P18-P20: pins of oracle/be_steps.py (NEXT-4: moments Eq. 5-9, 15; UPFD drift Eq. 30; UPFD Vlasov Eq. 34).

P18  moments against the closed forms of a (boosted) Maxwell-Juttner gas: N^mu = n0 u^mu,
     T^{mu nu} = (e + P) u^mu u^nu - P g^{mu nu} with n0 = 4 pi m^2 T K2(m/T), P = n0 T, e = n0 (m K1/K2 + 3 T)
     (textbook relativistic ideal gas); rho, J of Eq. 15 from the charges.
P19  drift: Eq. 30 as printed on a hand-sized 1-D example, positivity for any dt, constants and particle number
     preserved under periodic boundaries, first-order convergence to the exact translation by 3 v dt, wall ghosts.
P20  Vlasov: F = Q(E + v x B) against numpy.cross, Eq. 34 as printed on a hand-sized example, positivity, number
     conservation for a uniform E, sense of rotation in a magnetic field.
"""
import math

import numpy as np
import pytest
from scipy import special

from oracle import be_steps as bs


def _problem(masses, charges, n, lo, hi):
    return dict(nx=1, species=[dict(mass=m, charge=q, stat=0, g=1.0) for m, q in zip(masses, charges)],
                grids=[dict(n=list(n), pmin=list(lo), pmax=list(hi)) for _ in masses], processes=[], hbar=1.0)


# ------------------------------------------------------------------------------------------ P18
def test_p18_boosted_maxwell_juttner_moments():
    m, T, beta = 1.0, 0.4, 0.35
    nh = np.array([0.6, -0.48, 0.64])                     # unit vector: every component of T^{ik} is non-zero
    gam = 1.0 / math.sqrt(1 - beta * beta)
    n = (60, 60, 60)
    prob = _problem([m, m], [-1.0, 2.0], n, [-12.0] * 3, [12.0] * 3)
    P, E, V = bs.cell_tables(prob["grids"][0], m)
    f1 = np.exp(-(gam * E - gam * beta * (P @ nh)) / T)
    f = np.concatenate([f1, 0.5 * f1])
    M, tot, em = bs.moments(prob, f)
    z = m / T
    n0 = 4 * math.pi * m * m * T * special.kn(2, z)
    Pr = n0 * T
    e = n0 * (m * special.kn(1, z) / special.kn(2, z) + 3 * T)
    u = gam * np.concatenate([[1.0], beta * nh])
    g = np.diag([1.0, -1.0, -1.0, -1.0])
    Tmn = (e + Pr) * np.outer(u, u) - Pr * g
    want = [n0 * u[0], n0 * u[1], n0 * u[2], n0 * u[3], Tmn[0, 0], Tmn[0, 1], Tmn[0, 2], Tmn[0, 3],
            Tmn[1, 1], Tmn[1, 2], Tmn[1, 3], Tmn[2, 2], Tmn[2, 3], Tmn[3, 3]]
    assert M.shape == (2, 1, 14) and len(bs.MOMENT_NAMES) == 14
    for k, w in enumerate(want):
        assert M[0, 0, k] == pytest.approx(w, rel=2e-6), bs.MOMENT_NAMES[k]
        assert M[1, 0, k] == pytest.approx(0.5 * w, rel=2e-6)
        assert tot[0, k] == pytest.approx(1.5 * w, rel=2e-6)
    # Eq. 15 with charges -1 and +2: rho = -n_1 + 2 n_2 = 0, J likewise
    assert np.all(np.abs(em[0]) < 1e-12 * n0)
    prob["species"][1]["charge"] = 1.0
    _, _, em = bs.moments(prob, f)
    assert em[0, 0] == pytest.approx(-0.5 * n0 * u[0], rel=2e-6) and em[0, 3] == pytest.approx(-0.5 * n0 * u[3], rel=2e-6)


def test_p18_moments_are_per_spatial_cell_and_massless_origin_is_finite():
    prob = _problem([0.0], [1.0], (5, 5, 5), [-1.0] * 3, [1.0] * 3)      # odd grid: a cell centre at p = 0, E = 0
    prob["nx"] = 3
    rng = np.random.default_rng(3)
    f = rng.random(3 * 125)
    M, tot, em = bs.moments(prob, f)
    assert np.all(np.isfinite(M))
    dp3 = 0.4 ** 3
    assert M[0, :, 0] == pytest.approx(f.reshape(3, 125).sum(1) * dp3, rel=1e-14)
    # trace identity for massless particles: T00 = T11 + T22 + T33
    assert M[0, :, 4] == pytest.approx(M[0, :, 8] + M[0, :, 11] + M[0, :, 13], rel=1e-12)


# ------------------------------------------------------------------------------------------ P19
def _drift_1d_problem():
    # massless, momentum cells p_x = -0.5, +0.5 (v_x = -1, +1), p_y = p_z = 0
    return _problem([0.0], [0.0], (2, 1, 1), [-1.0, -1.0, -1.0], [1.0, 1.0, 1.0])


def test_p19_eq30_as_printed_on_a_three_cell_line():
    prob = _drift_1d_problem()
    f = np.array([[1.0, 2.0], [4.0, 8.0], [16.0, 32.0]])          # [ix, ip]
    dt, dx = 0.1, 0.5
    out = bs.drift_upfd(prob, f.reshape(-1), (3, 1, 1), dt, (dx, 1.0, 1.0)).reshape(3, 2)
    pre = 3 * dx / (3 * 1.0 * dt + dx)                             # Eq. 30, |v_x| = 1
    for i in range(3):
        right_mover = pre * (f[i, 1] / 3 + dt / dx * f[(i - 1) % 3, 1])       # v_x > 0: f(x - dx)
        left_mover = pre * (f[i, 0] / 3 + dt / dx * f[(i + 1) % 3, 0])        # v_x < 0: f(x + dx)
        assert out[i, 1] == pytest.approx(right_mover, rel=1e-15)
        assert out[i, 0] == pytest.approx(left_mover, rel=1e-15)
    # walls: absorbing (zeta = 0) -> ghost 0; reflecting (zeta = 1) -> ghost = the wall cell's mirrored momentum
    out0 = bs.drift_upfd(prob, f.reshape(-1), (3, 1, 1), dt, (dx, 1.0, 1.0), bc=(0, 1, 1), zeta=0.0).reshape(3, 2)
    out1 = bs.drift_upfd(prob, f.reshape(-1), (3, 1, 1), dt, (dx, 1.0, 1.0), bc=(0, 1, 1), zeta=0.7).reshape(3, 2)
    assert out0[0, 1] == pytest.approx(pre * (f[0, 1] / 3), rel=1e-15)
    assert out1[0, 1] == pytest.approx(pre * (f[0, 1] / 3 + dt / dx * 0.7 * f[0, 0]), rel=1e-15)
    assert out1[2, 0] == pytest.approx(pre * (f[2, 0] / 3 + dt / dx * 0.7 * f[2, 1]), rel=1e-15)
    assert out1[1] == pytest.approx(out[1], rel=1e-15)


def test_p19_positivity_constants_and_conservation():
    prob = _problem([0.3], [0.0], (4, 3, 5), [-2.0] * 3, [2.0] * 3)
    nxyz = (5, 4, 3)
    rng = np.random.default_rng(1)
    npc = 60
    f = rng.random(60 * npc)
    for dt in (1e-3, 0.3, 50.0):                                    # unconditionally positive
        out = bs.drift_upfd(prob, f, nxyz, dt, (0.2, 0.3, 0.25))
        assert np.all(out > 0)
        # periodic: the particle number of every momentum cell is conserved
        assert out.reshape(60, npc).sum(0) == pytest.approx(f.reshape(60, npc).sum(0), rel=1e-13)
    const = np.full(60 * npc, 0.37)
    assert bs.drift_upfd(prob, const, nxyz, 0.2, (0.2, 0.3, 0.25)) == pytest.approx(const, rel=1e-15)
    assert np.array_equal(bs.drift_upfd(prob, f, nxyz, 0.0, (0.2, 0.3, 0.25)), f / 3.0 / (1.0 / 3.0))


def test_p19_first_order_convergence_to_the_exact_translation():
    """Eq. 25 moves the profile with velocity 3 v.  Eq. 29 evaluates the cell's own value at t + dt, so the step is
    consistent with Eq. 25 only as dt |v| / dx -> 0 (its transport speed is 3 v / (1 + 3 dt |v| / dx)); with dt ~ dx^2
    the error is first order in dx."""
    prob = _drift_1d_problem()
    errs = []
    for n in (64, 128, 256):
        x = (np.arange(n) + 0.5) / n
        prof = lambda y: np.exp(-0.5 * ((y % 1.0 - 0.5) / 0.08) ** 2)
        f = np.stack([prof(x), prof(x)], axis=1)
        dx = 1.0 / n
        dt = 0.05 * dx * (64.0 / n)
        steps = int(round(0.05 / (3 * dt)))                         # translate by 0.05
        g = f.reshape(-1)
        for _ in range(steps):
            g = bs.drift_upfd(prob, g, (n, 1, 1), dt, (dx, 1.0, 1.0))
        g = g.reshape(n, 2)
        shift = 3 * dt * steps
        errs.append(max(np.abs(g[:, 1] - prof(x - shift)).max(), np.abs(g[:, 0] - prof(x + shift)).max()))
    assert errs[1] < 0.65 * errs[0] and errs[2] < 0.6 * errs[1], errs


# ------------------------------------------------------------------------------------------ P20
def test_p20_lorentz_force_against_numpy_cross():
    rng = np.random.default_rng(2)
    V = rng.normal(size=(7, 3)); E = rng.normal(size=(4, 3)); B = rng.normal(size=(4, 3))
    F = bs.lorentz_force(-1.6, V, E, B)
    for ix in range(4):
        for ip in range(7):
            assert F[ix, ip] == pytest.approx(-1.6 * (E[ix] + np.cross(V[ip], B[ix])), rel=1e-14, abs=1e-15)


def test_p20_eq34_as_printed_and_conservation():
    prob = _problem([1.0], [2.0], (4, 1, 1), [-2.0, -1.0, -1.0], [2.0, 1.0, 1.0])
    f = np.array([1.0, 3.0, 9.0, 27.0])
    dt, Ex = 0.05, 1.5
    dp = 1.0
    out = bs.vlasov_upfd(prob, f, dt, [[Ex, 0, 0]], [[0, 0, 0]])
    Fx = 2.0 * Ex
    pre = 3 * dp / (3 * Fx * dt + dp)                               # Eq. 34, F_x > 0: neighbour at p_x - dp, periodic
    for i in range(4):
        assert out[i] == pytest.approx(pre * (f[i] / 3 + dt * Fx / dp * f[(i - 1) % 4]), rel=1e-15)
    out_neg = bs.vlasov_upfd(prob, f, dt, [[-Ex, 0, 0]], [[0, 0, 0]])
    for i in range(4):
        assert out_neg[i] == pytest.approx(pre * (f[i] / 3 + dt * Fx / dp * f[(i + 1) % 4]), rel=1e-15)
    assert out.sum() == pytest.approx(f.sum(), rel=1e-14)           # uniform force, periodic: number conserved
    assert np.array_equal(bs.vlasov_upfd(prob, f, dt, [[0, 0, 0]], [[0, 0, 0]]), f / 3.0 / (1.0 / 3.0))
    assert np.all(bs.vlasov_upfd(prob, f, 1e4, [[Ex, 0.3, -2.0]], [[0.4, 0.1, 7.0]]) > 0)


def test_p20_magnetic_field_turns_a_positive_charge_clockwise_about_b():
    """dp/dt = Q v x B: with B along +z a positive charge moving along +x is pushed towards -y."""
    prob = _problem([0.5], [1.0], (12, 12, 4), [-3.0] * 3, [3.0] * 3)
    P, E, V = bs.cell_tables(prob["grids"][0], 0.5)
    f = np.exp(-((P[:, 0] - 1.5) ** 2 + P[:, 1] ** 2 + P[:, 2] ** 2) / 0.3)
    g = f.copy()
    for _ in range(10):
        g = bs.vlasov_upfd(prob, g, 0.01, [[0, 0, 0]], [[0, 0, 1.0]])
    cy0, cy1 = (f * P[:, 1]).sum() / f.sum(), (g * P[:, 1]).sum() / g.sum()
    cx0, cx1 = (f * P[:, 0]).sum() / f.sum(), (g * P[:, 0]).sum() / g.sum()
    assert abs(cy0) < 1e-12 and cy1 < -0.05 and cx1 < cx0
    # expected turning rate: d<p_y>/dt = -3 Q <v_x> B (the factor 3 of Eq. 26)
    vx = (f * V[:, 0]).sum() / f.sum()
    assert cy1 == pytest.approx(-3 * 1.0 * vx * 1.0 * 0.1, rel=0.15)


# ------------------------------------------------------------------------------------------ P22
def test_p22_flux_limited_drift_conserves_stays_positive_and_moves_ramps_exactly():
    """Second-order flux-limited drift (Eq. 31-33).  Flux form: the particle number of every momentum cell is conserved
    under periodic boundaries.  Positive for sum_d 3 dt |v_d| / dx_d <= 1/2.  On a linear ramp phi = 1 and the step is the
    exact translation by 3 v dt."""
    prob = _problem([0.3], [0.0], (4, 3, 5), [-2.0] * 3, [2.0] * 3)
    nxyz = (6, 5, 4)
    rng = np.random.default_rng(1)
    f = rng.random(120 * 60) ** 3                                  # rough, with values near 0
    f[::7] = 0.0
    dx = (0.2, 0.3, 0.25)
    dt = 0.5 / (3 * (1 / 0.2 + 1 / 0.3 + 1 / 0.25))                # |v| < 1
    out = bs.drift_pfl(prob, f, nxyz, dt, dx)
    assert np.all(out >= 0)
    assert out.reshape(120, 60).sum(0) == pytest.approx(f.reshape(120, 60).sum(0), rel=1e-13)
    const = np.full(120 * 60, 0.37)
    assert bs.drift_pfl(prob, const, nxyz, dt, dx) == pytest.approx(const, rel=1e-15)
    # ramp along x away from the periodic seam: exact translation
    p1 = _drift_1d_problem()
    n = 40
    x = (np.arange(n) + 0.5) / n
    ramp = np.stack([2.0 + 3.0 * x, 2.0 + 3.0 * x], axis=1)
    dt1, dx1 = 0.002, 1.0 / n
    got = bs.drift_pfl(p1, ramp.reshape(-1), (n, 1, 1), dt1, (dx1, 1.0, 1.0)).reshape(n, 2)
    assert got[4:-4, 1] == pytest.approx(2.0 + 3.0 * (x[4:-4] - 3 * dt1), rel=1e-13)      # v_x = +1
    assert got[4:-4, 0] == pytest.approx(2.0 + 3.0 * (x[4:-4] + 3 * dt1), rel=1e-13)      # v_x = -1


def test_p22_flux_limited_drift_is_less_diffusive_and_second_order():
    """Against the exact translation of a smooth profile: the error falls faster than first order with the cell size and
    is several times below the first-order scheme's on the same grid ("to suppress the numerical
    diffusion")."""
    prob = _drift_1d_problem()
    e2, e1 = [], []
    for n in (64, 128, 256):
        x = (np.arange(n) + 0.5) / n
        prof = lambda y: 1.0 + np.exp(-0.5 * ((y % 1.0 - 0.5) / 0.08) ** 2)
        f = np.stack([prof(x), prof(x)], axis=1).reshape(-1)
        dx = 1.0 / n
        dt = 0.05 * dx * (64.0 / n)
        steps = int(round(0.05 / (3 * dt)))
        g2, g1 = f, f
        for _ in range(steps):
            g2 = bs.drift_pfl(prob, g2, (n, 1, 1), dt, (dx, 1.0, 1.0))
            g1 = bs.drift_upfd(prob, g1, (n, 1, 1), dt, (dx, 1.0, 1.0))
        shift = 3 * dt * steps
        e2.append(np.abs(g2.reshape(n, 2)[:, 1] - prof(x - shift)).mean())
        e1.append(np.abs(g1.reshape(n, 2)[:, 1] - prof(x - shift)).mean())
    assert e2[1] < e2[0] / 2.6 and e2[2] < e2[1] / 2.6, e2
    assert e2[2] < e1[2] / 4, (e1, e2)


def test_p22_limiter_special_cases():
    th = 1e-10
    # flat upwind pair: the face value is the cell value; empty upwind cell next to a full one: no anti-diffusion
    assert bs._limited_face(np.array([2.0]), np.array([2.0]), np.array([5.0]), th)[0] == 2.0
    assert bs._limited_face(np.array([3.0]), np.array([0.0]), np.array([1.0]), th)[0] == 0.0
    # smooth increasing data: phi = 1 (linear extrapolation from the upwind side)
    assert bs._limited_face(np.array([1.0]), np.array([2.0]), np.array([3.5]), th)[0] == pytest.approx(2.5)
    # local maximum (r < 0): phi = 0, first-order upwind value
    assert bs._limited_face(np.array([1.0]), np.array([2.0]), np.array([1.5]), th)[0] == 2.0
    # steeply decreasing data: the positivity limiter 2 fc/(fl - fc) keeps the face value >= 0
    v = bs._limited_face(np.array([10.0]), np.array([0.1]), np.array([0.0]), th)[0]
    assert 0.0 <= v <= 0.1
