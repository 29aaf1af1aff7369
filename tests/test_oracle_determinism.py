"""P11 and housekeeping: thread-count independence, spatial-subset consistency, the float chain,
role expansion (Eq. 19) and the Euler update (Eq. 27)."""
import os
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest

import oracle
import workloads

ROOT = Path(__file__).resolve().parent.parent

_SCRIPT = """
import sys, numpy as np
sys.path.insert(0, %r)
import oracle, workloads
w = workloads.make(2, nx=2, np_side=6, n_samples=64)
o = oracle.Oracle(w['problem'])
np.save(sys.argv[1], o.collision(w['f'], 64, w['seed']))
"""


def test_p11_result_independent_of_thread_count(tmp_path):
    outs = []
    for nt in ("1", "5"):
        out = tmp_path / f"c{nt}.npy"
        env = dict(os.environ, OMP_NUM_THREADS=nt)
        subprocess.run([sys.executable, "-c", _SCRIPT % str(ROOT), str(out)], check=True, env=env)
        outs.append(np.load(out))
    assert np.array_equal(outs[0], outs[1])
    assert np.any(outs[0] != 0)


def test_spatial_subset_gives_the_same_cells():
    w = workloads.make(2, nx=6, np_side=5, n_samples=32)
    o = oracle.Oracle(w["problem"])
    full = o.collision(w["f"], 32, 1)
    sub = o.collision(w["f"], 32, 1, ix_begin=1, ix_end=6, ix_stride=2)
    for s in range(o.n_species):
        a = full[o.sp_off[s]:o.sp_off[s] + 6 * o.np[s]].reshape(6, -1)
        b = sub[o.sp_off[s]:o.sp_off[s] + 6 * o.np[s]].reshape(6, -1)
        assert np.array_equal(a[1::2], b[1::2]) and np.all(b[0::2] == 0)
    # cells differ from one another (the stream is keyed by the spatial index, the input varies with x)
    assert not np.array_equal(a[1], a[3])


def test_roles_and_symmetry_factor():
    w = workloads.make(3, nx=1, np_side=4, n_samples=8)
    o = oracle.Oracle(w["problem"])
    assert o.n_roles == 12
    for r in o.roles:
        a, b, c, d = r["s"]
        assert (c, d) == (a, b)
        assert r["sym"] == (0.5 if a == b else 1.0)
    # a+b and b+a views of one process are consecutive, "a-side" first
    assert [r["s"][:2] for r in o.roles[4:6]] == [(0, 1), (1, 0)]
    with pytest.raises(ValueError):
        # a + b -> b + a must be written a + b -> a + b (inelastic processes are accepted since NEXT-2(ii):
        # Eq. 16 is general, tests/test_oracle_qcd.py)
        bad = dict(w["problem"], processes=[dict(a=0, b=1, c=1, d=0, kind=0, par=[1.0], sym=-1.0)])
        oracle.Oracle(bad)


def test_collision_is_sum_of_roles_and_seed_matters():
    w = workloads.make(2, nx=1, np_side=6, n_samples=64)
    o = oracle.Oracle(w["problem"])
    C, d = o.collision(w["f"], 64, 5, detail=True)
    acc = np.zeros_like(C); mag = np.zeros_like(C)
    for r in range(o.n_roles):
        s1 = o.roles[r]["s"][0]
        sl = slice(o.role_off[r], o.role_off[r] + o.np[s1])
        acc[o.sp_off[s1]:o.sp_off[s1] + o.np[s1]] += (d["G"] - d["L"])[sl]
        mag[o.sp_off[s1]:o.sp_off[s1] + o.np[s1]] += (d["G"] + d["L"])[sl]
    assert np.all(np.abs(C - acc) <= 1e-14 * mag)
    assert not np.array_equal(C, o.collision(w["f"], 64, 6))


def test_float_chain_tracks_the_double_chain():
    """fp32 kinematics (config 5): same streams, so the two chains see nearly the same samples; a few
    samples land in a neighbouring cell, so agreement is statistical, not bitwise."""
    w = workloads.make(1, np_side=8, n_samples=512)
    od = oracle.Oracle(w["problem"]); of = oracle.Oracle(w["problem"], use_float=True)
    Cd, dd = od.collision(w["f"], 512, 3, detail=True)
    Cf, df = of.collision(w["f"], 512, 3, detail=True)
    assert np.allclose(df["L"], dd["L"], rtol=2e-3)
    assert np.abs(df["G"] - dd["G"]).sum() < 0.02 * dd["G"].sum()
    # heavy species: the cancellation-free float chain keeps s - (m1+m2)^2 accurate
    w2 = workloads.make(2, nx=1, np_side=6, n_samples=16)
    o2d = oracle.Oracle(w2["problem"]); o2f = oracle.Oracle(w2["problem"], use_float=True)
    hh = [r for r in range(o2d.n_roles) if o2d.roles[r]["s"] == (1, 1, 1, 1)][0]
    for n in range(16):
        a = o2d.trace(w2["f"], hh, 0, 100, n, 9); b = o2f.trace(w2["f"], hh, 0, 100, n, 9)
        if a["status"] == 0 and b["status"] == 0:
            hd = a["s"] - (2 * 1836.0) ** 2
            assert abs((b["pf"] - a["pf"]) / a["pf"]) < 1e-4, (a["pf"], b["pf"], hd)


def test_euler_update_and_negativity_count():
    f = np.array([1.0, 0.5, 1e-3, 0.0])
    C = np.array([-1.0, 2.0, -2.0, -1e-9])
    out, neg = oracle.update(f, C, 1e-3)
    assert np.allclose(out, f + 1e-3 * C, rtol=1e-15)
    assert neg == 2
