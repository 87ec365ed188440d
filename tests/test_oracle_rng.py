"""Pin T3: the oracle's Philox-4x32-10 against published known-answer vectors, and U()."""
import os

import numpy as np

GOLD = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


def _vectors():
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        w = [int(x, 16) for x in line.split()]
        yield w[0:4], w[4:6], w[6:10]


def test_philox_known_answers(oracle):
    n = 0
    for ctr, key, out in _vectors():
        got = oracle.philox(ctr, key)
        assert [int(x) for x in got] == out
        n += 1
    assert n == 3


def test_philox_counter_and_key_sensitivity(oracle):
    base = oracle.philox([1, 2, 3, 4], [5, 6])
    for pos in range(4):
        c = [1, 2, 3, 4]
        c[pos] += 1
        assert not np.array_equal(oracle.philox(c, [5, 6]), base)
    assert not np.array_equal(oracle.philox([1, 2, 3, 4], [5, 7]), base)
    assert not np.array_equal(oracle.philox([1, 2, 3, 4], [6, 6]), base)


def test_uniform53_range_and_layout(oracle):
    assert oracle.uniform53(0, 0) == 0.0
    assert oracle.uniform53(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 2.0 ** -53
    # w1 supplies the top 27 bits, w2 the low 26 ((w1>>5)*2^26 + (w2>>6))
    assert oracle.uniform53(1 << 5, 0) == 2.0 ** -27
    assert oracle.uniform53(0, 1 << 6) == 2.0 ** -53
    assert oracle.uniform53(31, 63) == 0.0
    assert oracle.uniform53(0x80000000, 0) == 0.5
