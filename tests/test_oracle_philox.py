"""P1: the oracle's Philox4x32-10 against published known-answer vectors, and basic stream hygiene."""
import numpy as np

import oracle
from conftest import read_golden


def test_philox_known_answers():
    for name, line in read_golden("philox_kat.txt").items():
        key, ctr, out = [tuple(int(x, 16) for x in part.split()) for part in line.split("|")]
        assert oracle.philox4x32_10(key, ctr) == out, name


def test_philox_python_reimplementation_agrees():
    # independent pure-Python Philox (written from the SC'11 description) on random inputs
    def ref(key, ctr):
        k0, k1 = key
        c = list(ctr)
        for _ in range(10):
            p0 = 0xD2511F53 * c[0]
            p1 = 0xCD9E8D57 * c[2]
            c = [(p1 >> 32) ^ c[1] ^ k0, p1 & 0xFFFFFFFF, (p0 >> 32) ^ c[3] ^ k1, p0 & 0xFFFFFFFF]
            k0 = (k0 + 0x9E3779B9) & 0xFFFFFFFF
            k1 = (k1 + 0xBB67AE85) & 0xFFFFFFFF
        return tuple(c)
    rng = np.random.default_rng(0)
    for _ in range(200):
        key = tuple(int(x) for x in rng.integers(0, 2 ** 32, 2))
        ctr = tuple(int(x) for x in rng.integers(0, 2 ** 32, 4))
        assert oracle.philox4x32_10(key, ctr) == ref(key, ctr)


def test_philox_words_are_uniform():
    xs = np.array([oracle.philox4x32_10((7, 9), (i, 3, 1, 0)) for i in range(4000)], dtype=np.float64) / 2 ** 32
    assert abs(xs.mean() - 0.5) < 4 * np.sqrt(1 / 12 / xs.size)
    assert abs(np.corrcoef(xs[:, 0], xs[:, 1])[0, 1]) < 0.06
