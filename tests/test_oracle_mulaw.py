"""Pins of the oracle's mu-law quantiser (Eq. 5) against closed forms, not against itself."""
import numpy as np

import oracle


def test_end_points_midpoint_and_monotone():
    mu = 255.0
    xmax = 1000.0
    mid = xmax * (np.sqrt(1.0 + mu) - 1.0) / mu                 # log(1 + mu x/X) = log(1 + mu)/2  <=>  y/X = 1/2
    x = np.array([0.0, xmax, mid, 1e-30, -5.0], dtype=np.float32)
    c, xm = oracle.mulaw_u8(x, mu)
    assert xm == 1000.0
    assert c.tolist()[:2] == [0, 255] and c[2] in (127, 128) and c[3] == 0 and c[4] == 0
    g = np.sort(np.random.default_rng(0).uniform(0, 1000, 10000).astype(np.float32))
    cg, _ = oracle.mulaw_u8(np.append(g, np.float32(1000.0)), mu)
    assert np.all(np.diff(cg.astype(int)) >= 0) and cg[-1] == 255 and len(np.unique(cg)) > 200


def test_matches_numpy_formula_and_linear_limit():
    g = np.random.default_rng(1)
    x = np.abs(g.normal(size=50000)).astype(np.float32) * 30          # half-normal, like a power series
    for mu in (1e-6, 10.0, 255.0):
        c, xm = oracle.mulaw_u8(x, mu)
        v = 255.0 * np.log1p(mu * x.astype(np.float64) / float(x.max())) / np.log1p(mu)
        ref = np.floor(v + 0.5).astype(np.uint8)
        near = np.abs(v - np.floor(v) - 0.5) < 1e-9
        assert xm == float(x.max()) and np.array_equal(c[~near], ref[~near])
        if mu < 1e-3:                                                  # mu -> 0: the quantiser becomes linear
            lin = np.floor(255.0 * x.astype(np.float64) / float(x.max()) + 0.5)
            assert np.max(np.abs(c.astype(int) - lin)) <= 1 and np.mean(c == lin) > 0.999


def test_all_zero_series():
    c, xm = oracle.mulaw_u8(np.zeros(16, dtype=np.float32), 255.0)
    assert xm == 0.0 and not c.any()
