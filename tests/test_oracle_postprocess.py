"""Pins of the oracle's post-processing functions against things other than
themselves: numpy's median / least squares on brute-force windows, exact lines, and the invariants Eq. 2 implies."""
import numpy as np
import pytest

import oracle


@pytest.mark.parametrize("window", [1, 3, 5, 9, 15])
def test_median_matches_numpy_brute_force(window):
    g = np.random.default_rng(window)
    x = g.normal(size=(3, 2, 211)).astype(np.float32)
    n = 200
    y = oracle.median_filter(x, n, window)
    h = window // 2
    for idx in np.ndindex(3, 2):
        for m in range(n):
            lo, hi = max(0, m - h), min(n - 1, m + h)
            assert y[idx][m] == np.float32(np.median(x[idx][lo:hi + 1].astype(np.float64)))
    assert np.array_equal(y[..., n:], x[..., n:])


def test_median_removes_isolated_outliers_and_keeps_monotone_series():
    n = 100
    x = np.arange(n, dtype=np.float32)[None].copy()
    y = oracle.median_filter(x, n, 5)
    assert np.array_equal(y[0, 2:n - 2], x[0, 2:n - 2])              # a monotone series is its own median inside
    x[0, 40] = 1e6                                                  # one isolated spike
    y = oracle.median_filter(x, n, 5)
    assert y.max() < 1e3 and np.array_equal(y[0, :38], oracle.median_filter(np.arange(n, dtype=np.float32)[None].copy(), n, 5)[0, :38])
    step = np.r_[np.zeros(50), np.ones(50)].astype(np.float32)[None].copy()
    assert np.array_equal(oracle.median_filter(step, n, 7), step)    # an edge is preserved exactly


def test_detrend_matches_numpy_least_squares():
    g = np.random.default_rng(3)
    n = 5000
    t = np.arange(n)
    x = (3.0 + 2e-3 * t + g.normal(size=(4, n)) * 1.5).astype(np.float32)
    x = np.ascontiguousarray(np.pad(x, ((0, 0), (0, 7))))
    y, p = oracle.detrend(x, n)
    for s in range(4):
        slope, icpt = np.polyfit(t.astype(np.float64), x[s, :n].astype(np.float64), 1)
        r = x[s, :n].astype(np.float64) - (slope * t + icpt)
        assert p[s, 1] == pytest.approx(slope, rel=1e-9)
        assert p[s, 0] == pytest.approx(icpt + slope * (n - 1) / 2.0, rel=1e-9)
        assert p[s, 2] == pytest.approx(np.sqrt(np.mean(r * r)), rel=1e-9)
        assert np.allclose(y[s, :n], r / p[s, 2], rtol=0, atol=2e-6)
        assert abs(float(y[s, :n].mean())) < 1e-6 and float(y[s, :n].std()) == pytest.approx(1.0, abs=1e-6)


def test_detrend_exact_line_and_constant_give_zeros():
    n = 64
    t = np.arange(n, dtype=np.float32)
    x = np.stack([2.0 + 0.5 * t, np.full(n, 7.0, dtype=np.float32)]).astype(np.float32)
    y, p = oracle.detrend(x, n)
    assert p[0, 1] == pytest.approx(0.5) and p[1, 1] == 0.0 and p[1, 2] == 0.0
    # an exact line leaves a zero residual: both series become zeros (reading E-ii)
    assert p[0, 2] < 1e-6 and np.all(y[0] == 0.0) and np.all(y[1] == 0.0)
