"""Deterministic brute-force quadrature of the reduced collision integral (R) -- TEST INFRASTRUCTURE.

Independent of rbg_oracle.cpp (numpy, textbook Lorentz boost with explicit gamma and beta,
t from four-vector products), used to pin the Monte Carlo oracle (pin P9).

(R), from Eq. 16 after the two-body phase-space integral:

  C_role(p1) = sym * Int_box d3p2 Int dOmega*  |M|^2 |p*| / (64 pi^2 E1 E2 sqrt(s)) [f3 f4 F1 F2 - f1 f2 F3 F4]

p2: tensor Gauss-Legendre over the species-2 momentum box; cos(theta*): Gauss-Legendre;
phi*: periodic trapezoid.  f is analytic (callables), F = 1 + theta*kappa*f (Eq. 18).
"""
from __future__ import annotations

import numpy as np


def m2_value(kind, par, s, t):
    if kind == 0:
        return np.full_like(s, par[0])
    if kind == 1:
        return par[0] / (t - par[1] ** 2) ** 2
    if kind == 2:
        return par[0] ** 4 * s ** 2 / (t - par[1] ** 2) ** 2
    raise ValueError(kind)


def collision_quadrature(p1, masses, fs, theta_kappa, kind, par, sym, box2, n_p2=12, n_cos=16, n_phi=16,
                         boxes_cut=None, panels=1, chunk=4096):
    """masses = (m1,m2,m3,m4); fs = 4 callables f_i(p[...,3]) -> array; theta_kappa = 4 floats;
    box2 = (pmin[3], pmax[3]) of the sampled partner.  boxes_cut: optional 4 (pmin,pmax) boxes; f_i is
    set to zero outside box i (the 'zero outside the box' rule).  p2 uses a composite rule: `panels`
    equal panels per axis with n_p2 Gauss-Legendre nodes each.  Returns (C, gain, loss)."""
    p1 = np.asarray(p1, float)
    m1, m2, m3, m4 = masses
    xg, wg = np.polynomial.legendre.leggauss(n_p2)
    axes, wts = [], []
    for d in range(3):
        edges = np.linspace(box2[0][d], box2[1][d], panels + 1)
        axes.append(np.concatenate([0.5 * (b - a) * xg + 0.5 * (b + a) for a, b in zip(edges[:-1], edges[1:])]))
        wts.append(np.concatenate([0.5 * (b - a) * wg for a, b in zip(edges[:-1], edges[1:])]))
    P2 = np.stack(np.meshgrid(*axes, indexing="ij"), -1).reshape(-1, 3)
    W2 = (wts[0][:, None, None] * wts[1][None, :, None] * wts[2][None, None, :]).reshape(-1)
    cg, cw = np.polynomial.legendre.leggauss(n_cos)
    phi = 2 * np.pi * (np.arange(n_phi) + 0.5) / n_phi
    pw = np.full(n_phi, 2 * np.pi / n_phi)
    ct = cg[:, None] + 0 * phi[None, :]
    st = np.sqrt(1 - ct ** 2)
    nh = np.stack([st * np.cos(phi)[None, :], st * np.sin(phi)[None, :], ct], -1).reshape(-1, 3)   # (A,3)
    WA = (cw[:, None] * pw[None, :]).reshape(-1)

    E1 = np.sqrt(p1 @ p1 + m1 * m1)

    def fval(i, p):
        v = fs[i](p)
        if boxes_cut is not None:
            lo, hi = np.asarray(boxes_cut[i][0]), np.asarray(boxes_cut[i][1])
            inside = np.all((p >= lo) & (p < hi), axis=-1)
            v = np.where(inside, v, 0.0)
        return v

    f1 = float(fval(0, p1[None, :])[0])
    F1 = 1 + theta_kappa[0] * f1
    gain = loss = 0.0
    P2_all, W2_all = P2, W2
    for c0 in range(0, P2_all.shape[0], chunk):
        P2, W2 = P2_all[c0:c0 + chunk], W2_all[c0:c0 + chunk]
        E2 = np.sqrt((P2 * P2).sum(1) + m2 * m2)                  # (B,)
        Pt = p1[None, :] + P2                                     # (B,3)
        Et = E1 + E2
        s = Et ** 2 - (Pt * Pt).sum(1)
        ok = s > (m3 + m4) ** 2
        s = np.where(ok, s, (m3 + m4) ** 2 + 1.0)
        rs = np.sqrt(s)
        pf = np.sqrt((s - (m3 + m4) ** 2) * (s - (m3 - m4) ** 2)) / (2 * rs)
        E3s = np.sqrt(pf ** 2 + m3 * m3)
        beta = Pt / Et[:, None]                                   # (B,3)
        gamma = Et / rs
        # boost p3* = pf * nh to the lab: p = p* + gamma beta (gamma/(gamma+1) beta.p* + E*)
        p3s = pf[:, None, None] * nh[None, :, :]                  # (B,A,3)
        bp = (beta[:, None, :] * p3s).sum(-1)                     # (B,A)
        coef = gamma[:, None] * (gamma[:, None] / (gamma[:, None] + 1) * bp + E3s[:, None])
        p3 = p3s + coef[..., None] * beta[:, None, :]
        p4 = Pt[:, None, :] - p3
        E3 = np.sqrt((p3 * p3).sum(-1) + m3 * m3)
        # t = (p1 - p3)^2 = m1^2 + m3^2 - 2 (E1 E3 - p1.p3)
        t = m1 * m1 + m3 * m3 - 2 * (E1 * E3 - (p3 * p1[None, None, :]).sum(-1))
        M2 = m2_value(kind, par, np.broadcast_to(s[:, None], t.shape), t)
        f2 = fval(1, P2)[:, None]
        f3 = fval(2, p3)
        f4 = fval(3, p4)
        F2 = 1 + theta_kappa[1] * f2
        F3 = 1 + theta_kappa[2] * f3
        F4 = 1 + theta_kappa[3] * f4
        kern = M2 * (pf / (64 * np.pi ** 2 * E1 * E2 * rs))[:, None] * ok[:, None]
        wt = W2[:, None] * WA[None, :]
        gain += sym * np.sum(wt * kern * f3 * f4 * F1 * F2)
        loss += sym * np.sum(wt * kern * f1 * f2 * F3 * F4)
    return gain - loss, gain, loss
