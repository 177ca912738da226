"""Pins for oracle.delay_table (reading A; Eq. 1 at PAPER.md:93)."""
import json
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
from workloads import CONFIGS

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "delay_pins.json")))


def _table(cfg):
    return oracle.delay_table(cfg.nchans, cfg.f_top, cfg.foff, cfg.tsamp, cfg.dm_low, cfg.dm_step, cfg.ndms)


@pytest.mark.parametrize("k,key", [(1, "cfg1"), (2, "cfg2"), (5, "cfg5")])
def test_golden_values(k, key):
    d = _table(CONFIGS[k])
    g = GOLD[key]
    assert int(d.max()) == g["max_delay"] == int(d[-1, -1])
    assert int(d.sum(dtype=np.int64)) == g["table_sum"]
    for row, cols in g["rows"].items():
        for c, v in cols.items():
            assert int(d[int(row), int(c)]) == v, (row, c)


def _exact_delay(cfg, d, c):
    """Eq. 1 in exact rational arithmetic, round half up (independent of fp64 evaluation order)."""
    F = Fraction
    dm = F(cfg.dm_low).limit_denominator(10**6) + d * F(cfg.dm_step).limit_denominator(10**6)
    f_top = F(cfg.f_top)
    f = f_top + c * F(cfg.foff)            # foff values are dyadic or 20/4096: exact as binary doubles
    x = F(4148808, 1000) * dm * (1 / (f * f) - 1 / (f_top * f_top)) / F(512, 10**7)
    return (x + F(1, 2)).__floor__(), x


@pytest.mark.parametrize("k", [1, 2, 5])
def test_exact_rational_spot_checks(k):
    cfg = CONFIGS[k]
    d = _table(cfg)
    rng = np.random.default_rng(k)
    pts = [(cfg.ndms - 1, cfg.nchans - 1), (1, cfg.nchans - 1), (cfg.ndms - 1, 1)]
    pts += [(int(rng.integers(cfg.ndms)), int(rng.integers(cfg.nchans))) for _ in range(300)]
    for (dd, c) in pts:
        want, x = _exact_delay(cfg, dd, c)
        assert int(d[dd, c]) == want
        # no entry sits close enough to a half-integer for fp64 evaluation order to matter (A2)
        assert abs((x % 1) - Fraction(1, 2)) > Fraction(1, 10**9)


def test_paper_printed_constant():
    """Eq. 1 prints 4.15e6 ms (3 s.f.) with f in MHz: delays must agree to that precision."""
    cfg = CONFIGS[2]
    d = _table(cfg).astype(np.float64)
    f = cfg.f_top + np.arange(cfg.nchans) * cfg.foff
    dm = cfg.dm_low + np.arange(cfg.ndms) * cfg.dm_step
    dt_ms = 4.15e6 * (f[None, :] ** -2 - cfg.f_top ** -2) * dm[:, None]          # PAPER.md:93 as printed
    samples = dt_ms * 1e-3 / cfg.tsamp
    assert np.all(np.abs(d - samples) <= 0.5 + 5e-4 * samples + 1e-9)


@pytest.mark.parametrize("k", [1, 2, 5])
def test_structure(k):
    cfg = CONFIGS[k]
    d = _table(cfg).astype(np.int64)
    assert np.all(d[0] == 0) and np.all(d[:, 0] == 0)              # DM 0 / reference channel
    assert np.all(np.diff(d, axis=0) >= 0) and np.all(np.diff(d, axis=1) >= 0)   # later at lower f, higher DM
    assert np.all(np.diff(d, axis=0) <= 5)                         # adjacent-DM difference in [0,5] (P1)
    assert np.all(np.diff(d[:, -1]) >= 4)                          # rows distinct (P3 premise)
    # doubling DM doubles the un-rounded delay: |delay(2d) - 2 delay(d)| <= 1.5
    half = (cfg.ndms - 1) // 2
    assert np.all(np.abs(d[2 * np.arange(half + 1)] - 2 * d[: half + 1]) <= 1)


def test_textbook_band_delay():
    """Lorimer & Kramer textbook form: dt = 4.148808 ms * DM * (f_lo^-2 - f_hi^-2), f in GHz."""
    cfg = CONFIGS[1]
    d = _table(cfg)
    f_lo = (cfg.f_top + 63 * cfg.foff) / 1e3
    dt_ms = 4.148808 * 2.0 * (f_lo ** -2 - (cfg.f_top / 1e3) ** -2)
    assert int(d[20, 63]) == round(dt_ms * 1e-3 / cfg.tsamp) == 94
