"""Pins for the oracle's RNG layer (R3, R4; PAPER.md line 124 names the Saru hash this replaces)."""
import os

import numpy as np

from oracle import hpmc_oracle as ho

GOLD = os.path.join(os.path.dirname(__file__), "golden", "philox_kat.txt")


def test_philox_known_answers():
    rows = [l.split() for l in open(GOLD) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = ho.philox4x32_10(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def test_philox_counter_and_key_sensitivity():
    base = ho.philox4x32_10([1, 2, 3, 4], [5, 6])
    for w in range(4):
        c = [1, 2, 3, 4]; c[w] ^= 1
        assert not np.array_equal(ho.philox4x32_10(c, [5, 6]), base)
    assert not np.array_equal(ho.philox4x32_10([1, 2, 3, 4], [5, 7]), base)
    assert not np.array_equal(ho.philox4x32_10([1, 2, 3, 4], [4, 6]), base)


def test_u01_usym_exact_and_ranges():
    # R4: 24-bit integers scaled by powers of two are exact in fp32
    assert ho.u01(0) == 0.0 and ho.u01(0xFFFFFFFF) == 1.0 - 2.0 ** -24
    assert ho.usym(0) == -1.0 and ho.usym(0xFFFFFFFF) == 1.0 - 2.0 ** -23
    assert ho.usym(0x80000000) == 0.0 and ho.u01(0x80000000) == 0.5
    for r in (0x12345678, 0xDEADBEEF, 0x000000FF, 0x00000100):
        assert ho.u01(r) == (r >> 8) / 2.0 ** 24
        assert ho.usym(r) == ((r >> 8) - 2 ** 23) / 2.0 ** 23


def test_stream_uniformity_chi2():
    # the paper's own unit test: "trial moves are generated from the proper uniform distribution"
    n = 20000
    words = np.zeros((n, 4), dtype=np.uint64)
    for i in range(n):
        words[i] = ho.philox4x32_10([i, 7, 3, 3 << 24], [1, 0])
    u = (words >> 8).astype(np.float64) / 2.0 ** 24
    for w in range(4):
        hist, _ = np.histogram(u[:, w], bins=64, range=(0, 1))
        chi2 = ((hist - n / 64) ** 2 / (n / 64)).sum()
        assert chi2 < 120.0  # 63 dof: mean 63, sd 11.2; 120 is > 5 sigma
    # lag-1 correlation between words of one block and between consecutive counters
    assert abs(np.corrcoef(u[:, 0], u[:, 1])[0, 1]) < 0.03
    assert abs(np.corrcoef(u[:-1, 2], u[1:, 2])[0, 1]) < 0.03
