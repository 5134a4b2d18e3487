"""Pins of the oracle's random-number layer."""
import os

import numpy as np

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


def test_philox_known_answers():
    n = 0
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(x, 16) for x in line.split()]
        assert oracle.philox(w[0:4], w[4:6]) == w[6:10]
        n += 1
    assert n == 3


def test_philox_is_a_bijection_on_a_counter_sample():
    # distinct counters -> distinct blocks (Philox is a keyed permutation of the counter space)
    outs = {tuple(oracle.philox([i, 0, 7, j], [1, 2])) for i in range(64) for j in range(64)}
    assert len(outs) == 64 * 64


def test_philox_words_are_uniform():
    words = np.array([oracle.philox([i, 0, 0, 0], [123, 0]) for i in range(20000)], dtype=np.uint64)
    u = (words.astype(np.float64) + 0.5) / 2.0**32
    assert abs(u.mean() - 0.5) < 4 * (1 / 12) ** 0.5 / u.size**0.5
    # each bit is set half of the time
    for b in (0, 7, 8, 31):
        frac = ((words >> np.uint64(b)) & np.uint64(1)).mean()
        assert abs(frac - 0.5) < 4 * 0.5 / words.size**0.5


def test_uniform_mapping_is_open_interval_and_fp32_exact():
    assert oracle.uniform(0) == 0.5 / 2**23
    assert oracle.uniform(0xFFFFFFFF) == 1.0 - 0.5 / 2**23
    assert oracle.uniform(0x000001FF) == oracle.uniform(0)      # low 9 bits unused
    for w in (0, 1 << 9, 0x12345678, 0xFFFFFE00, 0xFFFFFFFF):
        u = oracle.uniform(w)
        assert 0.0 < u < 1.0
        assert float(np.float32(u)) == u                        # survives single precision
