"""Pins for the oracle's RNG contract (DESIGN.md section 3 'R'): printed KATs, ranges, closed-form moments."""
import os

import numpy as np
import pytest
from scipy import stats

from oracle import oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden", "philox_kat.txt")


def test_philox_known_answers():
    n = 0
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(x, 16) for x in line.split()]
        assert O.philox(w[0:4], w[4:6]) == w[6:10]
        n += 1
    assert n == 3


def test_philox_matches_numpy_bitgenerator():
    # numpy's Philox is 4x64, not 4x32, so it cannot serve; instead check the bijection property on a counter sweep:
    # distinct counters -> distinct outputs (a dropped round-key bump or swapped lane typically breaks the KATs above;
    # this guards the counter wiring used by the walk: c0 block, c1 step, c2 slot, c3 stream).
    seen = set()
    for c0 in range(3):
        for c1 in range(5):
            for c2 in range(5):
                for c3 in (0, 1 << 24):
                    seen.add(tuple(O.philox([c0, c1, c2, c3], [7, 9])))
    assert len(seen) == 3 * 5 * 5 * 2


def test_u53_range_and_grid():
    assert O.u53(0, 0) == 2.0 ** -53
    assert O.u53(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 2.0 ** -53
    assert 0.0 < O.u53(0, 0) < O.u53(0xFFFFFFFF, 0xFFFFFFFF) < 1.0
    # hi contributes 26 bits, lo 26 bits
    assert O.u53(1 << 6, 0) - O.u53(0, 0) == 2.0 ** -26
    assert O.u53(0, 1 << 6) - O.u53(0, 0) == 2.0 ** -52
    assert O.u53(0x80000000, 0) == 0.5 + 2.0 ** -53


def test_mulhi_index_range():
    for m in (2, 3, 500, 700, 131072):
        assert O.mulhi32(0, m) == 0
        assert O.mulhi32(0xFFFFFFFF, m) == m - 1
        assert O.mulhi32(0x80000000, m) == m // 2


def test_gamma_distribution_and_distinct_donors():
    # gamma = 1 w.p. 1/2 else 2.38/sqrt(2 n_dim) * Gamma(shape 4, scale 0.25)
    n_free, m = 11, 500
    gs, ones, hist = [], 0, np.zeros(m)
    for j in range(6000):
        g, a, b, one = O.gamma_draw(n_free, 12345, j % 7, j, 3, m)
        assert 0 <= a < m and 0 <= b < m and a != b
        hist[a] += 1
        if one:
            ones += 1
            assert g == 1.0
        else:
            gs.append(g / (2.38 / np.sqrt(2 * n_free)))
    assert abs(ones / 6000 - 0.5) < 0.03
    gs = np.array(gs)
    assert abs(gs.mean() - 1.0) < 0.03            # Erlang-4 scale 1/4: mean 1
    assert abs(gs.var() - 0.25) < 0.03            # variance 1/4
    assert stats.kstest(gs, stats.gamma(a=4, scale=0.25).cdf).pvalue > 1e-3
    # donor index roughly uniform (chi^2 over 10 coarse bins)
    coarse = hist.reshape(10, -1).sum(1)
    assert stats.chisquare(coarse).pvalue > 1e-3


def test_draw_live_uniform():
    u = O.draw_live(11, 4000, 99)
    assert u.min() > 0 and u.max() < 1
    for d in range(11):
        assert stats.kstest(u[:, d], "uniform").pvalue > 1e-4
    assert abs(np.corrcoef(u[:, 0], u[:, 1])[0, 1]) < 0.06
