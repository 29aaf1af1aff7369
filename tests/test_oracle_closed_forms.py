"""P3 / P4: the oracle's loss rate against a closed form and against a scipy quadrature
(Eq. 20-22: loss = f1 * Int f2 sigma_tot v_Moller)."""
import math

import numpy as np
import pytest
from scipy import integrate

import oracle
from conftest import read_golden


def _one_species(m, n, lo, hi, kind=0, par=(1.0,), sym=-1.0, hbar=1.0):
    return dict(nx=1, species=[dict(mass=m, charge=0, stat=0, g=1.0)],
                grids=[dict(n=[n] * 3, pmin=[lo] * 3, pmax=[hi] * 3)],
                processes=[dict(a=0, b=0, c=0, d=0, kind=kind, par=list(par), sym=sym)], hbar=hbar)


def _loss_with_error(o, ip1, fcb, seed, batches=16, n=1 << 20):
    """Mean and empirical standard error of the scaled loss over independent Philox keys."""
    Ls = np.array([o.point(None, 0, 0, ip1, n, seed + 1000 * i, fcb=fcb, box_cut=False)[1] for i in range(batches)])
    return Ls.mean(), Ls.std(ddof=1) / math.sqrt(batches)


def test_p3_massless_closed_form():
    """Massless, classical, constant |M|^2, f2 = exp(-|p|/T): rate/f1 = sym |M|^2 T^2 / (8 E1)."""
    T, M2 = 0.5, 2.5
    prob = _one_species(0.0, 24, -6.0, 6.0, par=(M2,))          # sym=-1 -> paper rule 1/2 (a == b)
    o = oracle.Oracle(prob)
    thermal = ("thermal", [[1.0, T, 0.0, 0.0, 0.0, 0, 0, 0]])
    for ip1 in ((13 * 24 + 9) * 24 + 16, (11 * 24 + 12) * 24 + 12):
        tr = o.trace(None, 0, 0, ip1, 0, 1, fcb=thermal, box_cut=False)
        exact = 0.5 * M2 * T * T / (8 * tr["E1"]) * tr["f1"]
        L, se = _loss_with_error(o, ip1, thermal, 4242 + ip1)
        assert se < 0.02 * exact
        assert abs(L - exact) < 4 * se + 1e-3 * exact, (L, exact, se)


def test_p3_hbar_squared_prefactor_of_eq16():
    """Eq. 16 carries hbar^2 c |M|^2 / (64 pi^2 ...): with c = 1 the closed form of P3 becomes
    hbar^2 sym |M|^2 T^2 / (8 E1) for classical particles (no nbar).  A dropped or single power of hbar fails."""
    T, M2, hbar = 0.5, 2.5, 0.5
    o = oracle.Oracle(_one_species(0.0, 24, -6.0, 6.0, par=(M2,), hbar=hbar))
    thermal = ("thermal", [[1.0, T, 0.0, 0.0, 0.0, 0, 0, 0]])
    ip1 = (13 * 24 + 9) * 24 + 16
    tr = o.trace(None, 0, 0, ip1, 0, 1, fcb=thermal, box_cut=False)
    exact = hbar * hbar * 0.5 * M2 * T * T / (8 * tr["E1"]) * tr["f1"]
    L, se = _loss_with_error(o, ip1, thermal, 99)
    assert se < 0.02 * exact
    assert abs(L - exact) < 4 * se + 1e-3 * exact, (L, exact, se)


def test_cell_centre_with_zero_energy_is_refused():
    """1/p^0 of Eq. 16: a massless species with a cell centre at p = 0 (odd grid, symmetric box) has no
    finite collision term there (reading R14): refused.  The same grid with a mass, or an even grid, is accepted."""
    with pytest.raises(ValueError):
        oracle.Oracle(_one_species(0.0, 7, -3.0, 3.0))
    with pytest.raises(ValueError):
        oracle.Oracle(_one_species(0.0, 7, -0.7, 0.7))            # centre = fma(3.5, 0.2, -0.7) ~ 1e-17, not exactly 0
    oracle.Oracle(_one_species(0.3, 7, -3.0, 3.0))
    oracle.Oracle(_one_species(0.0, 8, -3.0, 3.0))
    oracle.Oracle(_one_species(0.0, 7, -3.0, 4.0))                # odd but not symmetric: no centre at 0


def _rate_quadrature(p1, m, T):
    """Int d3p2 exp(-E2/T) |p*| / (16 pi E1 E2 sqrt s), spherical coordinates about p1."""
    a1 = math.sqrt(p1 @ p1)
    E1 = math.sqrt(a1 * a1 + m * m)

    def integrand(c, q):
        E2 = math.sqrt(q * q + m * m)
        s = 2 * m * m + 2 * (E1 * E2 - a1 * q * c)
        pst = math.sqrt(max(s * (s - 4 * m * m), 0.0)) / (2 * math.sqrt(s))
        return 2 * math.pi * q * q * math.exp(-E2 / T) * pst / (16 * math.pi * E1 * E2 * math.sqrt(s))
    val, err = integrate.dblquad(integrand, 0.0, 40.0 * T, -1.0, 1.0, epsabs=1e-12, epsrel=1e-10)
    return val


def test_p4_golden_value_reproduced_by_scipy():
    gold = float(read_golden("closed_forms.txt")["p4_rate_over_f1"])
    assert _rate_quadrature(np.array([0.3, -0.7, 1.1]), 1.0, 1.0) == pytest.approx(gold, rel=2e-6)


def test_p4_massive_loss_rate_matches_scipy():
    m, T = 1.0, 0.8
    prob = _one_species(m, 120, -12.0, 12.0, sym=1.0)
    o = oracle.Oracle(prob)
    thermal = ("thermal", [[1.0, T, 0.0, m, 0.0, 0, 0, 0]])
    ip1 = (61 * 120 + 56) * 120 + 65
    tr = o.trace(None, 0, 0, ip1, 0, 1, fcb=thermal, box_cut=False)
    assert np.allclose(tr["p1"], [0.3, -0.7, 1.1], atol=1e-12)
    ref = _rate_quadrature(tr["p1"], m, T) * tr["f1"]
    L, se = _loss_with_error(o, ip1, thermal, 777)
    assert se < 0.02 * ref
    assert abs(L - ref) < 4 * se + 1e-3 * ref, (L, ref, se)


def _sigma_rate_quadrature(p1, m1, m2, T, dsigma):
    """Eq. 20-21: loss rate / f1 = Int d3p2 f2 sigma_tot I / (E1 E2) with the invariant flux
    I = sqrt((p1.p2)^2 - m1^2 m2^2) and sigma_tot = 4 pi dsigma/dOmega for an isotropic cross section."""
    a1 = math.sqrt(p1 @ p1)
    E1 = math.sqrt(a1 * a1 + m1 * m1)

    def integrand(c, q):
        E2 = math.sqrt(q * q + m2 * m2)
        k12 = E1 * E2 - a1 * q * c                          # four-product p1.p2
        flux = math.sqrt(max(k12 * k12 - (m1 * m2) ** 2, 0.0))
        return 2 * math.pi * q * q * math.exp(-E2 / T) * 4 * math.pi * dsigma * flux / (E1 * E2)
    val, err = integrate.dblquad(integrand, 0.0, 40.0 * T, -1.0, 1.0, epsabs=1e-12, epsrel=1e-10)
    return val


def test_iso_dsigma_kind_loss_rate_is_sigma_times_flux():
    """Kind 3, |M|^2 = 64 pi^2 s dsigma/dOmega: the loss rate is f1 Int f2 sigma_tot v_Moller with
    sigma_tot = 4 pi dsigma/dOmega (Eq. 20-22), for unequal masses."""
    m1, m2, T, dsig = 0.3, 0.7, 0.6, 2.5
    prob = dict(nx=1, species=[dict(mass=m1, charge=0, stat=0, g=1.0), dict(mass=m2, charge=0, stat=0, g=1.0)],
                grids=[dict(n=[60] * 3, pmin=[-6.0] * 3, pmax=[6.0] * 3), dict(n=[60] * 3, pmin=[-9.0] * 3, pmax=[9.0] * 3)],
                processes=[dict(a=0, b=1, c=0, d=1, kind=3, par=[dsig], sym=-1.0)], hbar=1.0)
    o = oracle.Oracle(prob)
    thermal = ("thermal", [[1.0, T, 0.0, m1, 0.0, 0, 0, 0], [1.0, T, 0.0, m2, 0.0, 0, 0, 0]])
    ip1 = (33 * 60 + 26) * 60 + 35
    tr = o.trace(None, 0, 0, ip1, 0, 1, fcb=thermal, box_cut=False)
    ref = _sigma_rate_quadrature(tr["p1"], m1, m2, T, dsig) * tr["f1"]
    L, se = _loss_with_error(o, ip1, thermal, 999)
    assert se < 0.02 * ref
    assert abs(L - ref) < 4 * se + 1e-3 * ref, (L, ref, se)
    # per sample: the weight is the CONST-kind weight times 64 pi^2 s dsigma
    prob0 = dict(prob, processes=[dict(a=0, b=1, c=0, d=1, kind=0, par=[1.0], sym=-1.0)])
    o0 = oracle.Oracle(prob0)
    for n in range(20):
        a = o.trace(None, 0, 0, ip1, n, 5, fcb=thermal, box_cut=False)
        b = o0.trace(None, 0, 0, ip1, n, 5, fcb=thermal, box_cut=False)
        assert a["w"] == pytest.approx(b["w"] * 64 * math.pi ** 2 * a["s"] * dsig, rel=1e-14)
        assert np.array_equal(a["p3"], b["p3"])
