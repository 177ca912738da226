"""Pins for oracle.dedisperse (reading C; brute-force definition at)."""
import json
import os

import numpy as np
import pytest

import oracle
from workloads import CONFIGS, generate

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "impulse_pin.json")))
CFG1 = CONFIGS[1]


def table(cfg):
    return oracle.delay_table(cfg.nchans, cfg.f_top, cfg.foff, cfg.tsamp, cfg.dm_low, cfg.dm_step, cfg.ndms)


def numpy_gather_sum(x, delay):
    """Three-line brute force: fancy-index gather then sum over channels (ascending c)."""
    nb, nc, ns = x.shape
    nso = ns - int(delay.max())
    idx = delay[:, :, None] + np.arange(nso)[None, None, :]                     # [d][c][t]
    return np.stack([x[b][np.arange(nc)[None, :, None], idx].astype(np.float64).sum(axis=1) for b in range(nb)])


def test_P2_dm0_row_is_channel_sum():
    x = generate(CFG1)
    d = table(CFG1)
    out, _ = oracle.dedisperse(x, d)
    nso = out.shape[2]
    want = np.zeros(nso)
    for c in range(CFG1.nchans):
        want += x[0, c, :nso].astype(np.float64)
    assert np.array_equal(out[0, 0], want)
    xu = (np.abs(x) * 20).astype(np.uint8)
    outu, _ = oracle.dedisperse(xu, d)
    assert np.array_equal(outu[0, 0], xu[0, :, :nso].astype(np.uint32).sum(axis=0))


@pytest.mark.parametrize("dtype", [np.float32, np.uint8])
def test_P3_impulse_recovery_worked_example(dtype):
    d = table(CFG1)
    k, t0 = GOLD["k"], GOLD["t0"]
    x = np.zeros((1, CFG1.nchans, CFG1.nsamps), dtype=dtype)
    x[0, np.arange(CFG1.nchans), t0 + d[k]] = 1
    for variant in ("naive", "rows"):
        out, _ = oracle.dedisperse(x, d, variant=variant)
        assert out[0, k, t0] == GOLD["peak"] == CFG1.nchans
        o = out[0].copy()
        o[k, t0] = 0
        assert o.max() == GOLD["next_largest"]
        assert np.all(out[0].sum(axis=1) == GOLD["row_sum"])


def test_P3_impulse_recovery_other_dm():
    d = table(CFG1)
    for k, t0 in [(31, 17), (7, 3000), (1, 0)]:
        x = np.zeros((1, CFG1.nchans, CFG1.nsamps), dtype=np.float32)
        x[0, np.arange(CFG1.nchans), t0 + d[k]] = 1
        out, _ = oracle.dedisperse(x, d)
        assert out[0, k, t0] == CFG1.nchans
        assert (out[0] == CFG1.nchans).sum() == 1


def test_P4_linearity_shift_constant():
    d = table(CFG1)
    rng = np.random.default_rng(5)
    x = rng.integers(0, 50, size=(1, CFG1.nchans, CFG1.nsamps)).astype(np.uint8)
    y = rng.integers(0, 50, size=x.shape).astype(np.uint8)
    ox, _ = oracle.dedisperse(x, d)
    oy, _ = oracle.dedisperse(y, d)
    oz, _ = oracle.dedisperse((2 * x + 3 * y).astype(np.uint8), d)
    assert np.array_equal(oz, 2 * ox + 3 * oy)                                    # exact
    xf, yf = x.astype(np.float32) * 0.37, y.astype(np.float32) * -1.3
    a, _ = oracle.dedisperse(xf, d)
    b, _ = oracle.dedisperse(yf, d)
    c, ab = oracle.dedisperse((xf + yf).astype(np.float32), d)
    assert np.all(np.abs(c - (a + b)) <= 1e-6 * ab + 1e-9)
    # shifting the input by s shifts every series by s
    s = 37
    xs = np.zeros_like(xf)
    xs[:, :, s:] = xf[:, :, :-s]
    os_, _ = oracle.dedisperse(xs, d)
    assert np.array_equal(os_[:, :, s:], a[:, :, :-s])
    # constant input kappa -> nchans*kappa
    oc, _ = oracle.dedisperse(np.full_like(xf, 0.5), d)
    assert np.all(oc == 0.5 * CFG1.nchans)


@pytest.mark.parametrize("dtype", [np.float32, np.uint8])
def test_P5_brute_force_tiny(dtype):
    rng = np.random.default_rng(11)
    nb, nc, ns, nd = 2, 8, 64, 5
    d = oracle.delay_table(nc, 418.0, -2.5, 51.2e-6, 0.0, 0.15, nd)
    assert 0 < d.max() < ns // 2
    x = (rng.normal(size=(nb, nc, ns)) * 30 + 60).clip(0, 255).astype(dtype)
    want = numpy_gather_sum(x, d)
    # per-sample python loop (the definition, literally)
    nso = ns - int(d.max())
    loop = np.zeros((nb, nd, nso))
    for b in range(nb):
        for dd in range(nd):
            for t in range(nso):
                s = 0.0
                for c in range(nc):
                    s += float(x[b, c, t + d[dd, c]])
                loop[b, dd, t] = s
    for variant in ("naive", "rows"):
        out, ab = oracle.dedisperse(x, d, variant=variant)
        assert out.shape == (nb, nd, nso)
        assert np.array_equal(out.astype(np.float64), loop)
        assert np.array_equal(out.astype(np.float64), want)
        if dtype == np.float32:
            assert np.array_equal(ab, numpy_gather_sum(np.abs(x), d))
    sel, _ = oracle.dedisperse_rows(x, d, np.array([7, 0, 9]))
    assert np.array_equal(sel.astype(np.float64), loop.reshape(nb * nd, nso)[[7, 0, 9]])


def test_rows_equals_naive_cfg1():
    x = generate(CFG1)
    d = table(CFG1)
    a, aa = oracle.dedisperse(x, d, variant="naive")
    b, bb = oracle.dedisperse(x, d, variant="rows")
    assert np.array_equal(a, b) and np.array_equal(aa, bb)
    assert np.array_equal(a, numpy_gather_sum(x, d))


def test_cfg1_injected_pulse_peak():
    """P7 (chain part): cfg 1's pulse (3/channel, width 4, DM index 20, t0 = 1000) gives ~192 at the peak."""
    x = generate(CFG1)
    out, _ = oracle.dedisperse(x, table(CFG1))
    b, dd, t = np.unravel_index(out.argmax(), out.shape)
    assert dd == 20 and 1000 <= t <= 1003
    assert abs(out[0, 20, 1000:1004].mean() - 192.0) < 4 * 8 / 2
