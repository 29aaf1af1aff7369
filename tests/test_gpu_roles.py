"""Role expansion of the PRODUCT, checked against hand-written expectations (no oracle in this file): rbg_role_info
reports, for every role rbg_create made from the process list, the species of the four slots, the symmetry factor and
the degrees-of-freedom factors.  Parity with the oracle compares results, so a role list that was wrong in the same way
on both sides would pass it; these expectations come from Eq. 19 and its text (every species receives
every process it takes part in; 1/2 "when all incident particles are of the same type") and from reading R21 (DESIGN.md
section 7) for the degrees of freedom, written out by hand for each case."""
import pytest

pytestmark = pytest.mark.gpu

QQB_GG, Q1QB1_Q2QB2, CONST, COULOMB = 8, 7, 0, 1


def _problem(masses, procs, gs=None):
    gs = gs or [1.0] * len(masses)
    return dict(nx=1, species=[dict(mass=m, charge=0.0, stat=0, g=g) for m, g in zip(masses, gs)],
                grids=[dict(n=[4, 4, 4], pmin=[-3.0] * 3, pmax=[3.0] * 3) for _ in masses], processes=procs, hbar=1.0)


def _proc(a, b, c, d, kind, sym=-1.0):
    return dict(a=a, b=b, c=c, d=d, kind=kind, par=[1.0, 0.0], sym=sym)


def _roles(problem):
    import paper_2308_04869_b200 as rbg
    col = rbg.Collision(problem)
    return [col.role_info(r) for r in range(col.n_roles)], col


def test_role_lists_and_symmetry_factors():
    # q(0) qbar(1) -> g(2) g(2): seen from q, from qbar, and once from g; the g g pair is the incident pair of the q and
    # qbar views (1/2), the q qbar pair that of the g view (1)
    roles, _ = _roles(_problem([0.3, 0.3, 0.5], [_proc(0, 1, 2, 2, QQB_GG)]))
    assert [(r["s"], r["sym"]) for r in roles] == [((0, 1, 2, 2), 0.5), ((1, 0, 2, 2), 0.5), ((2, 2, 0, 1), 1.0)]
    assert [r["process"] for r in roles] == [0, 0, 0]
    # written the other way round: the same three views
    rev, _ = _roles(_problem([0.3, 0.3, 0.5], [_proc(2, 2, 0, 1, QQB_GG)]))
    assert sorted((r["s"], r["sym"]) for r in rev) == sorted((r["s"], r["sym"]) for r in roles)
    # q1 qb1 -> q2 qb2: four different species, four views, no identical pair; slots 3, 4 ordered so that 1 <-> 3 are
    # the t-channel partners of the process as written (a <-> c, b <-> d)
    four, _ = _roles(_problem([0.1, 0.1, 0.2, 0.2], [_proc(0, 1, 2, 3, Q1QB1_Q2QB2)]))
    assert [(r["s"], r["sym"]) for r in four] == [((0, 1, 2, 3), 1.0), ((1, 0, 3, 2), 1.0), ((2, 3, 0, 1), 1.0), ((3, 2, 1, 0), 1.0)]
    # elastic: a + b -> a + b gives one view per species, a + a -> a + a one view with 1/2; process indices follow the list
    el, col = _roles(_problem([0.1, 0.2], [_proc(0, 1, 0, 1, CONST), _proc(1, 1, 1, 1, CONST)]))
    assert [(r["s"], r["sym"], r["process"]) for r in el] == [((0, 1, 0, 1), 1.0, 0), ((1, 0, 1, 0), 1.0, 0), ((1, 1, 1, 1), 0.5, 1)]
    # an explicit sym overrides the rule in every view of that process
    ov, _ = _roles(_problem([0.1, 0.2], [_proc(0, 1, 0, 1, COULOMB, sym=0.25)]))
    assert [r["sym"] for r in ov] == [0.25, 0.25]
    import paper_2308_04869_b200 as rbg
    with pytest.raises(rbg.RbgError):
        col.role_info(3)
    with pytest.raises(rbg.RbgError):
        col.role_info(-1)
    with pytest.raises(rbg.RbgError):                      # a + b -> b + a must be written a + b -> a + b
        rbg.Collision(_problem([0.1, 0.2], [_proc(0, 1, 1, 0, CONST)]))


def test_degrees_of_freedom_factors():
    # Table III kinds are summed over the DOF of all four particles: loss 1+2 -> 3+4 carries 1/(g1 g2), gain 1/(g3 g4).
    # q, qbar with g = 6, gluons with g = 16
    roles, _ = _roles(_problem([0.3, 0.3, 0.5], [_proc(0, 1, 2, 2, QQB_GG)], gs=[6.0, 6.0, 16.0]))
    assert [(r["cl"], r["cg"]) for r in roles] == [(1 / 36.0, 1 / 256.0), (1 / 36.0, 1 / 256.0), (1 / 256.0, 1 / 36.0)]
    # kinds 0..3 give |M|^2 of the process as written averaged over g_a g_b: elastic views have 1 and 1 ...
    el, _ = _roles(_problem([0.1, 0.2], [_proc(0, 1, 0, 1, COULOMB)], gs=[2.0, 3.0]))
    assert [(r["cl"], r["cg"]) for r in el] == [(1.0, 1.0), (1.0, 1.0)]
    # ... and an inelastic a + b -> c + c of such a kind: |M|^2_sum = |M|^2 g_a g_b, so the views from a and b have
    # loss factor 1 and gain factor g_a g_b / g_c^2, the view from c the reverse
    inel, _ = _roles(_problem([0.1, 0.2, 0.05], [_proc(0, 1, 2, 2, CONST)], gs=[2.0, 3.0, 4.0]))
    assert [(r["s"], r["cl"], r["cg"]) for r in inel] == [((0, 1, 2, 2), 1.0, 6.0 / 16.0), ((1, 0, 2, 2), 1.0, 6.0 / 16.0),
                                                          ((2, 2, 0, 1), 6.0 / 16.0, 1.0)]
