"""Input generators: channel counts the paper prints, grids, rules."""
import os

import numpy as np

from paper_1508_07441_b200 import inputs as I


GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def test_channel_counts_match_paper():
    """tests/golden/paper_channel_counts.txt holds the two channel counts the paper prints (with their citations)."""
    rows = [ln.split() for ln in open(os.path.join(GOLDEN, "paper_channel_counts.txt")) if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 2
    for J2, par, T2, jmax, n in (tuple(int(x) for x in r) for r in rows):
        if J2 == 0:                                  # maximum over all J <= 17/2 and both parities
            counts = [len(I.enumerate_3n_channels(j2, p, T2, jmax)) for j2 in range(1, 19, 2) for p in (+1, -1)]
            assert max(counts) == n
        else:
            assert len(I.enumerate_3n_channels(J2, par, T2, jmax)) == n
    assert len(I.enumerate_3n_channels(1, +1, 1, 3)) == 26


def test_channels_obey_selection_rules():
    for J2, par in ((1, 1), (1, -1), (3, 1), (7, -1)):
        ch = I.enumerate_3n_channels(J2, par, 1, 3)
        assert len({tuple(c) for c in ch.tolist()}) == len(ch)
        for l, s, j, t, lam, I2 in ch.tolist():
            assert (l + s + t) % 2 == 1
            assert abs(l - s) <= j <= l + s and j <= 3
            assert abs(2 * lam - I2) == 1
            assert abs(2 * j - I2) <= J2 <= 2 * j + I2
            assert (-1) ** (l + lam) == par


def test_grids():
    g = I.tan_grid(10, 1.0)
    assert g[0] == 0.0 and len(g) == 11 and np.all(np.diff(g) > 0)
    assert abs(g[-1] - np.tan(np.pi * 10 / 22)) < 1e-14
    s = I.split_grid()
    assert len(s) == 101 and s[20] == 0.5 and s[-1] == 30.0 and np.all(np.diff(s) > 0)
    assert np.allclose(np.diff(s[:21]), 0.025)


def test_rules_are_symmetric_and_exact_for_polynomials():
    for n in (4, 6, 8, 10, 16, 24, 32):
        t, w = I.gauss_legendre(n)
        assert np.all(t == -t[::-1]) and np.all(w == w[::-1])
        assert abs(w.sum() - 2.0) < 1e-14
        assert abs((w * t ** 2).sum() - 2.0 / 3.0) < 1e-14
        assert abs((w * t ** (2 * n - 2)).sum() - 2.0 / (2 * n - 1)) < 1e-13


def test_config_sizes():
    M = [I.config(k).M for k in range(5)]
    assert M == [100, 5000, 180000, 260000, 585000]      # SURVEY.md sec. 8 size table
    assert [I.config(k).nodes_per_cell for k in range(5)] == [128, 576, 1536, 2048, 3200]
