"""The paper's own 5-dimensional form of the collision integral, Eq. 35-37 (PAPER.md:342-356,
appendix Eq. 49-61) -- TEST INFRASTRUCTURE (pin P6).

  C_{ab->cd}(p) = Int d3k3 dk1x dk1y  |M|^2 / (64 pi^2 k1^0 k2^0 k3^0 p^0)  Sum_{+-} 1/|J(k1z^+-)|
                  [ f_k1 f_k2 F_k3 F_p - F_k1 F_k2 f_k3 f_p ],      k2 = k3 + p - k1,
  J(k1z) = k1z/k1^0 - (-k1z + k3z + pz)/k2^0                                   (Eq. 36 / 59)

hbar = c = 1.  The printed C1, C2, H of Eq. 62 are garbled and truncated, so the
roots of k1^0 + k2^0 - k3^0 - p^0 = 0 are re-derived (reading R1 of DESIGN.md): with Q = k3 + p,
E_T = k3^0 + p^0, a = k1x^2 + k1y^2 + m_a^2, b = (Qx-k1x)^2 + (Qy-k1y)^2 + m_b^2,
D = E_T^2 + a - b - Qz^2:

  k1z^+- = [ D Qz +- E_T sqrt(D^2 - 4 a (E_T^2 - Qz^2)) ] / [ 2 (E_T^2 - Qz^2) ]

which matches the legible parts C2 = 2(E_T - Qz)(E_T + Qz), C1 = Qz D, H = E_T^2 [...].
Squaring introduced spurious roots: a root is kept only if it satisfies the unsquared equation.

Plain Monte Carlo: k3 uniform in its momentum box, (k1x,k1y) uniform in the square of side E_T
centred on Q_perp/2 (the solution ellipsoid has foci 0 and Q and major axis <= E_T).
Labels: grid particle d(p) == particle 1 of the hot path, c(k3) == 2, (a(k1), b(k2)) == (3,4).
"""
from __future__ import annotations

import numpy as np

from .quadrature import m2_value


def eq37_mc(p, masses, fs, theta_kappa, kind, par, sym, box3, n, rng, chunk=1 << 20):
    """masses = (m_d, m_c, m_a, m_b) in hot-path order (1,2,3,4); fs/theta_kappa likewise.
    Returns ((gain, se), (loss, se)): the two terms of the bracket estimated separately."""
    p = np.asarray(p, float)
    md, mc, ma, mb = masses
    lo, hi = np.asarray(box3[0], float), np.asarray(box3[1], float)
    V3 = np.prod(hi - lo)
    p0 = np.sqrt(p @ p + md * md)
    fp = float(fs[0](p[None, :])[0])
    Fp = 1 + theta_kappa[0] * fp
    tot = np.zeros(2)
    tot2 = np.zeros(2)
    done = 0
    while done < n:
        m = min(chunk, n - done)
        k3 = lo + (hi - lo) * rng.random((m, 3))
        k30 = np.sqrt((k3 * k3).sum(1) + mc * mc)
        Q = k3 + p[None, :]
        ET = k30 + p0
        k1x = Q[:, 0] / 2 + ET * (rng.random(m) - 0.5)
        k1y = Q[:, 1] / 2 + ET * (rng.random(m) - 0.5)
        area = ET ** 2
        a = k1x ** 2 + k1y ** 2 + ma * ma
        b = (Q[:, 0] - k1x) ** 2 + (Q[:, 1] - k1y) ** 2 + mb * mb
        D = ET ** 2 + a - b - Q[:, 2] ** 2
        den = 2 * (ET ** 2 - Q[:, 2] ** 2)
        H = D ** 2 - 4 * a * (ET ** 2 - Q[:, 2] ** 2)
        val = np.zeros((2, m))
        okH = H > 0
        sq = ET * np.sqrt(np.where(okH, H, 0.0))
        for sign in (+1.0, -1.0):
            k1z = (D * Q[:, 2] + sign * sq) / den
            k1 = np.stack([k1x, k1y, k1z], 1)
            k2 = Q - k1
            k10 = np.sqrt((k1 * k1).sum(1) + ma * ma)
            k20 = np.sqrt((k2 * k2).sum(1) + mb * mb)
            good = okH & (np.abs(k10 + k20 - ET) < 1e-9 * ET)         # unsquared equation holds
            J = k1z / k10 - (-k1z + k3[:, 2] + p[2]) / k20
            s = ET ** 2 - (Q * Q).sum(1)
            # t = (p - k1)^2: momentum transfer between the grid particle and particle 3
            t = md * md + ma * ma - 2 * (p0 * k10 - (k1 * p[None, :]).sum(1))
            M2 = m2_value(kind, par, s, t)
            f1, f2, f3 = fs[2](k1), fs[3](k2), fs[1](k3)
            F1, F2, F3 = 1 + theta_kappa[2] * f1, 1 + theta_kappa[3] * f2, 1 + theta_kappa[1] * f3
            with np.errstate(divide="ignore", invalid="ignore"):
                kern = M2 / (64 * np.pi ** 2 * k10 * k20 * k30 * p0) / np.abs(J)
            for i, br in enumerate((f1 * f2 * F3 * Fp, F1 * F2 * f3 * fp)):   # gain, loss brackets of Eq. 37
                term = kern * br
                val[i] += np.where(good & np.isfinite(term), term, 0.0)
        val *= sym * V3 * area
        tot += val.sum(1)
        tot2 += (val * val).sum(1)
        done += m
    mean = tot / n
    se = np.sqrt(np.maximum(tot2 / n - mean * mean, 0.0) / n)
    return (mean[0], se[0]), (mean[1], se[1])
