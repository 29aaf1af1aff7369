"""rbg_moments_static -- the one entry point of librbg.so that allocates no device memory -- against the existing path.

Who needs it: a program that cannot let a library call cudaMalloc at the point where it wants the moments of f -- its
own pool already holds all of HBM, or its time-step loop cannot afford cudaMalloc's device-wide synchronisation, or the
application it is loaded into forbids allocations after start-up.  For such a caller the species' 1/E_p table, which
rbg_create would cudaMalloc, sits in a fixed 512 KB `static __device__` array inside the library instead (at most
RBG_MOMENTS_STATIC_MAX_CELLS = 65536 momentum cells), shared by all calls.

What is checked: on several calls in a row, with a different species and momentum grid each time (so every call finds
the previous call's table in the array), the result equals what rbg_create + rbg_moments give for the same input, within
the tolerance tests/test_gpu_be_steps.py uses for moments (1e-12 of the same sums over |f|; where rbg_moments takes the
same unstaged kernel, bit for bit); that free device memory does not move across a call once the first call on the
device has done its set-up; and that a grid beyond the limit is refused, not truncated.

This file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here must not
hide the parity tests.  It passes alone in a fresh process (its first call then is the first CUDA work of the process and
does the per-device set-up) and after the other GPU tests."""
import numpy as np
import pytest

# (n, pmin, pmax, mass, spatial cells).  In this order each call leaves stale entries of a different grid behind:
# 8000 cells, then 343 (most of the array still holds the first table), then 42 875 (longer than anything before it).
CASES = [((20, 20, 20), (-5.0, -5.0, -5.0), (5.0, 5.0, 5.0), 1.0, 5),        # rbg_moments: symmetric-grid staged kernel
         ((7, 7, 7), (-1.0, -2.0, -0.5), (3.0, 2.0, 2.5), 0.05, 3),          # odd, off-centre grid: general staged kernel
         ((35, 35, 35), (-2.0, -2.0, -2.0), (2.0, 2.0, 2.0), 0.3, 2)]        # 343 KB per cell: rbg_moments' unstaged kernel


def _problem(n, pmin, pmax, mass, cells):
    return dict(nx=cells, species=[dict(mass=mass, charge=0.0, stat=0, g=1.0)],
                grids=[dict(n=list(n), pmin=list(pmin), pmax=list(pmax))], processes=[], hbar=1.0)


@pytest.mark.gpu
def test_static_table_moments_match_the_allocating_path_on_calls_in_a_row():
    import torch
    import paper_2308_04869_b200 as rbg
    torch.cuda.set_device(0)
    rng = np.random.default_rng(20230804)
    inputs = []
    for n, pmin, pmax, mass, cells in CASES:
        f = torch.from_numpy(rng.random(cells * int(np.prod(n))) + 0.01).cuda()
        out = torch.full((cells, rbg.binding.N_MOMENTS), float("nan"), dtype=torch.float64, device="cuda")
        inputs.append((dict(n=n, pmin=pmin, pmax=pmax), mass, f, out))
    # the existing path (it allocates: handle tables, result tensors), evaluated first and kept on the host
    refs = []
    for (n, pmin, pmax, mass, cells), (_, _, f, _) in zip(CASES, inputs):
        col = rbg.Collision(_problem(n, pmin, pmax, mass, cells))
        refs.append(col.moments(f)[0][0].cpu().numpy())
        del col
    torch.cuda.synchronize()
    # two rounds over the three problems = six calls in a row on one stream, every one into a table another grid wrote
    for rnd in range(2):
        for i, (grid, mass, f, out) in enumerate(inputs):
            out.fill_(float("nan"))
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info()[0]
            res = rbg.moments_static(grid, mass, f, out=out)
            torch.cuda.synchronize()
            free_after = torch.cuda.mem_get_info()[0]
            assert res.data_ptr() == out.data_ptr()
            if rnd > 0 or i > 0:                     # the very first call may load the module on this device
                assert free_after == free_before, "rbg_moments_static changed the amount of free device memory"
            M, M_ref = out.cpu().numpy(), refs[i]
            assert np.all(np.isfinite(M))
            # f > 0, so M_ref's n and T00 are the sums over |f| the tolerance of test_gpu_be_steps.py is built from
            pabs = max(abs(v) for v in grid["pmin"] + grid["pmax"])
            scale = np.maximum(M_ref[:, 0:1], M_ref[:, 4:5]) * max(1.0, pabs) ** 2
            assert np.all(np.abs(M - M_ref) <= 1e-12 * scale), (rnd, i, np.max(np.abs(M - M_ref) / scale))
            assert np.all(M_ref[:, 0] > 0) and np.any(M_ref[:, 1:4] != 0)
            if i == 2:                               # same kernel, same table bits
                assert np.array_equal(M, M_ref)


@pytest.mark.gpu
def test_static_table_moments_result_does_not_depend_on_what_the_array_held():
    """The same problem evaluated right after a call on a different species gives the same bits as evaluated twice in a
    row: the array carries nothing over from one call to the next."""
    import torch
    import paper_2308_04869_b200 as rbg
    torch.cuda.set_device(0)
    rng = np.random.default_rng(7)
    gA = dict(n=(12, 10, 14), pmin=(-3.0, -3.0, -3.0), pmax=(3.0, 3.0, 3.0))
    gB = dict(n=(40, 40, 40), pmin=(-9.0, -9.0, -9.0), pmax=(9.0, 9.0, 9.0))          # 64 000 cells: nearly the whole array
    fA = torch.from_numpy(rng.random(4 * 12 * 10 * 14)).cuda()
    fB = torch.from_numpy(rng.random(1 * 64000)).cuda()
    a1 = rbg.moments_static(gA, 0.7, fA).clone()
    a2 = rbg.moments_static(gA, 0.7, fA).clone()
    rbg.moments_static(gB, 1836.0, fB)
    a3 = rbg.moments_static(gA, 0.7, fA).clone()
    torch.cuda.synchronize()
    assert torch.equal(a1, a2) and torch.equal(a1, a3)


def test_static_table_moments_refuse_a_grid_beyond_the_built_in_table():
    """Validation comes before any CUDA call, so this runs without a GPU: 41^3 = 68 921 cells > 65 536."""
    import ctypes as C
    import paper_2308_04869_b200 as rbg
    from paper_2308_04869_b200.binding import _MomentumGrid
    lib = rbg.load_library()
    assert rbg.MOMENTS_STATIC_MAX_CELLS == 65536

    def call(n, pmin=(-1.0, -1.0, -1.0), pmax=(1.0, 1.0, 1.0), mass=1.0, cells=1, f=0x1000, M=0x2000):
        g = _MomentumGrid((C.c_int * 3)(*n), (C.c_double * 3)(*pmin), (C.c_double * 3)(*pmax))
        rc = lib.rbg_moments_static(C.byref(g), mass, cells, C.c_void_p(f), C.c_void_p(M), None)
        return rc, (lib.rbg_last_error(None) or b"").decode()

    rc, msg = call((41, 41, 41))
    assert rc == -2 and "68921" in msg and "65536" in msg            # RBG_E_UNSUPPORTED, both numbers named
    rc, msg = call((2048, 2048, 2048))                                # 2^33 cells: no integer overflow on the way to the refusal
    assert rc == -2 and "65536" in msg
    assert call((0, 4, 4))[0] == -1                                   # RBG_E_INVALID_ARG
    assert call((4, 4, 4), pmax=(1.0, -1.0, 1.0))[0] == -1
    assert call((4, 4, 4), mass=-1.0)[0] == -1
    assert call((4, 4, 4), cells=-1)[0] == -1
    assert call((4, 4, 4), f=None)[0] == -1
    assert call((4, 4, 4), cells=0)[0] == 0                           # nothing to do: no launch, no set-up
