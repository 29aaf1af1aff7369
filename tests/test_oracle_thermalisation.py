"""P12: the paper's collision test (Eq. 46-48, Fig. 9), run with the oracle on a reduced grid.

What the paper fixes (figure only, no printed numbers): with dsigma/dOmega = 20 for b+b, 1 for a+a and 0.01 for
a+b, "the distribution function of species b gradually achieves the Boltzmann distribution, while species a is
still away from the thermal state".  What the mathematics fixes: an elastic classical gas relaxes
to exp(-E/T) (Eq. 11) with T set by the conserved energy per particle,
<E> = 3T + m K1(m/T)/K2(m/T) (textbook relativistic ideal gas)."""
import numpy as np
from scipy import optimize, special

import oracle
import workloads
from workloads.configs import cell_centres


def boltzmann_fit(f, E):
    """Least-squares line through ln f vs E over the populated cells: (T, rms residual of ln f)."""
    m = f > 1e-4 * f.max()
    A = np.vstack([E[m], np.ones(m.sum())]).T
    y = np.log(f[m])
    coef = np.linalg.lstsq(A, y, rcond=None)[0]
    return -1.0 / coef[0], float(np.sqrt(np.mean((y - A @ coef) ** 2)))


def temperature_from_energy_per_particle(e_over_n, m):
    return optimize.brentq(lambda T: 3 * T + m * special.kn(1, m / T) / special.kn(2, m / T) - e_over_n, 0.02, 5.0)


def test_species_b_thermalises_species_a_does_not():
    side, N, steps, dt = 21, 128, 50, 1e-3
    w = workloads.make(6, np_side=side, n_samples=N)
    o = oracle.Oracle(w["problem"])
    P = cell_centres(w["problem"]["grids"][0])
    E = np.sqrt((P * P).sum(1) + 0.3 ** 2)
    npc, dp3 = P.shape[0], (4.0 / side) ** 3
    f = w["f"].copy()
    n0 = [f[s * npc:(s + 1) * npc].sum() * dp3 for s in range(2)]
    e0 = [(f[s * npc:(s + 1) * npc] * E).sum() * dp3 for s in range(2)]
    for k in range(steps):
        f, neg = oracle.update(f, o.collision(f, N, w["seed"] + k), dt)
        assert neg == 0
    fa, fb = f[:npc], f[npc:]
    Ta, rms_a = boltzmann_fit(fa, E)
    Tb, rms_b = boltzmann_fit(fb, E)
    # b is Boltzmann (straight line in ln f vs E up to Monte Carlo noise), a is still far from it
    assert rms_b < 0.12, rms_b
    assert rms_a > 4 * rms_b, (rms_a, rms_b)
    # the temperature of b is the one its conserved energy per particle dictates
    T_pred = temperature_from_energy_per_particle(e0[1] / n0[1], 0.3)
    assert abs(Tb - T_pred) < 0.05 * T_pred, (Tb, T_pred)
    # bookkeeping: the weakly coupled species keeps its particles and energy; b leaks a few per cent through the
    # momentum box (scattering to |p_d| > 2 is lost: zero outside the box) and nothing is created
    assert abs(fa.sum() * dp3 / n0[0] - 1) < 5e-3
    assert abs((fa * E).sum() * dp3 / e0[0] - 1) < 1e-2
    assert 0.93 < fb.sum() * dp3 / n0[1] < 1.01
