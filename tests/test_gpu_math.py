"""The kernels' own fp64 divide / reciprocal / square root (IEEE fast paths without range checks)
against the CUDA library operators, bit for bit."""
import pytest

pytestmark = pytest.mark.gpu


def test_custom_fp64_ops_are_correctly_rounded():
    import paper_2308_04869_b200 as rbg
    for seed in (1, 2, 3):
        assert rbg.selftest_math(200_000_000, seed) == 0
