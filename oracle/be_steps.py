"""CPU oracle for the steps either side of the collision term -- TEST INFRASTRUCTURE.

Plain numpy, fp64, no blocking or fusion: each function is the paper's formula written out.  Shares no code with
the CUDA path and never imports it.

* moments()      n_a, j_a (Eq. 5-6), T^{mu nu}_a (Eq. 9), their sums over
                 species (Eq. 7) and the charge and current densities rho, J (Eq. 15).
* drift_upfd()   the first-order unconditionally-positivity-preserving upwind step of the drift term
                 (Eq. 25, 28-30), all three directions at once (reading R23).
* drift_pfl()    the second-order positivity-preserving flux-limited step of the drift term (Eq. 31-33,
                 PAPER.md:300-319), periodic (reading R26).
* vlasov_upfd()  the same scheme for the Vlasov term (Eq. 26, 34), F = Q (E + v x B)
                 (PAPER.md:162), periodic in momentum.

Conventions: hbar = c = 1; f layout [species][ix][ipx][ipy][ipz] with ix = (i_x ny + i_y) nz + i_z
(PAPER.md:402, :469); momentum integrals are midpoint sums over the cell centres, Int d3p -> Sum dp^3.
"""
from __future__ import annotations

import numpy as np

MOMENT_NAMES = ("n", "jx", "jy", "jz", "T00", "T01", "T02", "T03", "T11", "T12", "T13", "T22", "T23", "T33")


def cell_tables(grid, mass):
    """Cell-centre momenta p (np,3), energies E_p = sqrt(|p|^2 + m^2) and velocities v = p/E (Eq. 6)."""
    ax = []
    for d in range(3):
        n, lo, hi = grid["n"][d], grid["pmin"][d], grid["pmax"][d]
        ax.append(lo + (np.arange(n) + 0.5) * ((hi - lo) / n))
    P = np.stack(np.meshgrid(*ax, indexing="ij"), axis=-1).reshape(-1, 3)
    E = np.sqrt((P * P).sum(1) + mass * mass)
    with np.errstate(invalid="ignore", divide="ignore"):
        V = np.where(E[:, None] > 0, P / E[:, None], 0.0)          # a massless particle at p = 0 carries nothing
    return P, E, V


def _blocks(problem, f):
    nx = int(np.prod(problem["nx"])) if not np.isscalar(problem["nx"]) else int(problem["nx"])
    out, off = [], 0
    for g in problem["grids"]:
        npc = int(np.prod(g["n"]))
        out.append(f[off:off + nx * npc].reshape(nx, npc))
        off += nx * npc
    assert off == f.size
    return nx, out


def moments(problem, f):
    """Returns (M, total, em): M[s, ix, 14] per species in MOMENT_NAMES order, total[ix, 14] = Sum_a M_a (Eq. 7, 9)
    and em[ix, 4] = (rho, Jx, Jy, Jz) = Sum_a Q_a (n_a, j_a) (Eq. 15).
      n = Sum f dp3,  j^k = Sum v^k f dp3,  T^{00} = Sum E f dp3,  T^{0k} = Sum p^k f dp3,  T^{ik} = Sum p^i v^k f dp3
    (Eq. 9 with c = 1: d3p/p0 p^mu p^nu = d3p p^mu v^nu, v^0 = 1)."""
    nx, blocks = _blocks(problem, np.asarray(f, dtype=np.float64))
    ns = len(blocks)
    M = np.zeros((ns, nx, 14))
    em = np.zeros((nx, 4))
    for s, (g, sp, fb) in enumerate(zip(problem["grids"], problem["species"], blocks)):
        P, E, V = cell_tables(g, sp["mass"])
        dp3 = np.prod([(g["pmax"][d] - g["pmin"][d]) / g["n"][d] for d in range(3)])
        W = [np.ones_like(E), V[:, 0], V[:, 1], V[:, 2], E, P[:, 0], P[:, 1], P[:, 2]]
        for i, k in ((0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)):
            W.append(P[:, i] * V[:, k])
        for m, w in enumerate(W):
            M[s, :, m] = (fb * w[None, :]).sum(axis=1) * dp3
        em += sp.get("charge", 0.0) * M[s, :, 0:4]
    return M, M.sum(axis=0), em


def _shift_spatial(fb, nxyz, d, step, bc, zeta, mirror):
    """fb[ix, ip] -> value of the neighbour at spatial index i_d + step (step = +-1).  bc: 1 periodic; 0 wall with
    reflection probability zeta: the ghost value is zeta * f(boundary cell, momentum mirrored in d)."""
    a = fb.reshape(*nxyz, -1)
    out = np.roll(a, -step, axis=d)
    if bc != 1:
        ghost = zeta * a[..., mirror]
        idx = [slice(None)] * 4
        idx[d] = -1 if step > 0 else 0
        out = out.copy()
        out[tuple(idx)] = ghost[tuple(idx)]
    return out.reshape(fb.shape)


def _mirror_index(grid, d):
    n = grid["n"]
    I = np.arange(int(np.prod(n))).reshape(n)
    return np.flip(I, axis=d).reshape(-1)


def drift_upfd(problem, f, nxyz, dt, dx, bc=(1, 1, 1), zeta=0.0):
    """One UPFD step of Eq. 25, (1/3) df/dt + v . grad_x f = 0.  Replacing, in every direction d, the upwind
    difference by Eq. 29 (the updated value at the cell itself) gives

        f(t+dt, x) = [ f/3 + dt Sum_d |v_d| f(t, x - sign(v_d) dx_d e_d) / dx_d ] / [ 1/3 + dt Sum_d |v_d| / dx_d ],

    which is Eq. 30 when only v_x is non-zero ("The same formula can be obtained in the y and z directions",
    PAPER.md:298)."""
    f = np.asarray(f, dtype=np.float64)
    nx, blocks = _blocks(dict(problem, nx=int(np.prod(nxyz))), f)
    outs = []
    for g, sp, fb in zip(problem["grids"], problem["species"], blocks):
        _, _, V = cell_tables(g, sp["mass"])
        num = fb / 3.0
        den = np.full(V.shape[0], 1.0 / 3.0)
        for d in range(3):
            c = dt * np.abs(V[:, d]) / dx[d]
            mir = _mirror_index(g, d)
            up_pos = _shift_spatial(fb, nxyz, d, -1, bc[d], zeta, mir)      # v_d > 0: neighbour at x - dx
            up_neg = _shift_spatial(fb, nxyz, d, +1, bc[d], zeta, mir)      # v_d < 0: neighbour at x + dx
            up = np.where(V[None, :, d] > 0, up_pos, up_neg)
            num = num + c[None, :] * up
            den = den + c
        outs.append((num / den[None, :]).reshape(-1))
    return np.concatenate(outs)


def lorentz_force(charge, V, E, B):
    """F = Q (E + v x B) for every (spatial cell, momentum cell): E, B are [nx, 3], V is [np, 3]."""
    vxB = np.stack([V[None, :, 1] * B[:, None, 2] - V[None, :, 2] * B[:, None, 1],
                    V[None, :, 2] * B[:, None, 0] - V[None, :, 0] * B[:, None, 2],
                    V[None, :, 0] * B[:, None, 1] - V[None, :, 1] * B[:, None, 0]], axis=-1)
    return charge * (E[:, None, :] + vxB)


def vlasov_upfd(problem, f, dt, E, B):
    """One UPFD step of Eq. 26, (1/3) df/dt + F . grad_p f = 0 (Eq. 34, all three directions as in drift_upfd):

        f(t+dt, p) = [ f/3 + dt Sum_d |F_d| f(t, p - sign(F_d) dp_d e_d) / dp_d ] / [ 1/3 + dt Sum_d |F_d| / dp_d ],

    periodic in every momentum direction."""
    f = np.asarray(f, dtype=np.float64)
    E = np.asarray(E, dtype=np.float64).reshape(-1, 3)
    B = np.asarray(B, dtype=np.float64).reshape(-1, 3)
    nx, blocks = _blocks(dict(problem, nx=E.shape[0]), f)
    outs = []
    for g, sp, fb in zip(problem["grids"], problem["species"], blocks):
        _, _, V = cell_tables(g, sp["mass"])
        F = lorentz_force(sp.get("charge", 0.0), V, E, B)                    # [nx, np, 3]
        a = fb.reshape(nx, *g["n"])
        num = fb / 3.0
        den = np.full(fb.shape, 1.0 / 3.0)
        for d in range(3):
            dp = (g["pmax"][d] - g["pmin"][d]) / g["n"][d]
            c = dt * np.abs(F[:, :, d]) / dp
            up_pos = np.roll(a, +1, axis=1 + d).reshape(fb.shape)            # F_d > 0: neighbour at p - dp
            up_neg = np.roll(a, -1, axis=1 + d).reshape(fb.shape)            # F_d < 0: neighbour at p + dp
            up = np.where(F[:, :, d] > 0, up_pos, up_neg)
            num = num + c * up
            den = den + c
        outs.append((num / den).reshape(-1))
    return np.concatenate(outs)


def _limited_face(fl, fc, fr, theta):
    """Face value of the flux-limited scheme, Eq. 32-33, between the upwind cell c and the downwind
    cell r, with l the cell upwind of c:  fc + 1/2 phi (fc - fl),
        phi = max(0, min(1, (fr - fc)/(fc - fl), 2 / max(theta, (fl - fc)/fc))).
    The velocity does not depend on x, so the v^+- of Eq. 32-33 factor out.  phi multiplies (fc - fl), so where that
    difference vanishes the face value is fc whatever phi is (phi := 0 there); where fc = 0 (and fl > 0) the positivity
    limiter 2/((fl - fc)/fc) is 0 (reading R26)."""
    d = fc - fl
    with np.errstate(divide="ignore", invalid="ignore"):
        r = (fr - fc) / d
        lim = 2.0 / np.maximum(theta, (fl - fc) / fc)
        phi = np.maximum(0.0, np.minimum(1.0, np.minimum(r, lim)))
    phi = np.where((d == 0.0) | (fc == 0.0), 0.0, phi)
    return fc + 0.5 * phi * d


def drift_pfl(problem, f, nxyz, dt, dx, theta=1e-10):
    """One step of the second-order positivity-preserving flux-limited drift scheme, Eq. 31-33,
    periodic in x, y, z:
        f(t+dt) = f - 3 dt Sum_d (F_{i+1/2} - F_{i-1/2}) / dx_d,
    F_{i+1/2} of Eq. 32 with the limiters of Eq. 33 (first printing; the second printing of phi^- is garbled) and
    theta = 1e-10.  With s = sign(v_d): (F_{i+1/2} - F_{i-1/2}) = |v_d| (O - I), O the face value leaving
    cell i (upwind cell i, its upwind neighbour i-s, downwind i+s) and I the face value entering it (upwind cell i-s)."""
    f = np.asarray(f, dtype=np.float64)
    nx, blocks = _blocks(dict(problem, nx=int(np.prod(nxyz))), f)
    outs = []
    for g, sp, fb in zip(problem["grids"], problem["species"], blocks):
        _, _, V = cell_tables(g, sp["mass"])
        a = fb.reshape(*nxyz, -1)
        div = np.zeros_like(a)
        for d in range(3):
            pos = V[:, d] > 0
            sh = lambda k: np.roll(a, k, axis=d)                 # sh(k)[i] = a[i - k]
            # v > 0: upwind is i-1;  v < 0: upwind is i+1
            O = np.where(pos, _limited_face(sh(1), a, sh(-1), theta), _limited_face(sh(-1), a, sh(1), theta))
            I = np.where(pos, _limited_face(sh(2), sh(1), a, theta), _limited_face(sh(-2), sh(-1), a, theta))
            div = div + (np.abs(V[:, d]) / dx[d]) * (O - I)
        outs.append((a - 3.0 * dt * div).reshape(-1))
    return np.concatenate(outs)
