"""Pins for oracle.detect (reading D)."""
import numpy as np
import pytest

import oracle
from workloads import CONFIGS, generate


@pytest.mark.parametrize("dtype", [np.float32, np.float64, np.uint32])
def test_events_equal_brute_force_filter(dtype):
    g = np.random.default_rng(1)
    nb, nd, stride, n = 2, 5, 700, 650
    s = g.normal(size=(nb, nd, stride)) * 30 + 500
    s[0, 3, 100] += 400
    s[1, 1, 649] += 300
    s[1, 1, 660] += 9000          # beyond n: must be ignored
    s = s.astype(dtype)
    ev, cnt, stats = oracle.detect(s, n, 3.0)
    v = s[:, :, :n].astype(np.float64)
    mean = v.sum(axis=2) / n
    rms = np.sqrt(np.maximum((v * v).sum(axis=2) / n - mean * mean, 0))
    assert np.allclose(stats[..., 0], mean, rtol=1e-12) and np.allclose(stats[..., 1], rms, rtol=1e-9)
    snr = (v - stats[..., 0:1]) / stats[..., 1:2]
    b, d, t = np.nonzero(snr > 3.0)
    assert cnt == len(b) == len(ev) > 2
    assert np.array_equal(ev["beam"], b) and np.array_equal(ev["dm_idx"], d) and np.array_equal(ev["t"], t)
    assert np.array_equal(ev["snr"], snr[b, d, t].astype(np.float32))
    assert (0, 3, 100) in set(zip(b, d, t)) and (1, 1, 649) in set(zip(b, d, t))
    assert not np.any((ev["t"] >= n))


def test_population_rms_and_strict_greater():
    # series 0,0,0,4 : mean 1, population var = (16/4) - 1 = 3, rms sqrt(3); snr(4) = 3/sqrt(3) = sqrt(3)
    s = np.array([[[0, 0, 0, 4]]], dtype=np.uint32)
    ev, cnt, st = oracle.detect(s, 4, 1.0)
    assert cnt == 1 and ev["t"][0] == 3 and ev["snr"][0] == np.float32(np.sqrt(3.0))
    assert st[0, 0, 0] == 1.0 and st[0, 0, 1] == np.sqrt(3.0)
    # strict '>' (D-iii): series 0,0,2,2: mean 1 rms 1 snr = 1 exactly -> not an event at thr 1
    s = np.array([[[0, 0, 2, 2]]], dtype=np.uint32)
    assert oracle.detect(s, 4, 1.0)[1] == 0
    assert oracle.detect(s, 4, 0.999)[1] == 2


def test_constant_series_no_events():
    s = np.full((1, 2, 100), 5, dtype=np.uint32)
    assert oracle.detect(s, 100, 0.0)[1] == 0          # rms == 0 -> no events


def test_overflow_counts_past_capacity():
    g = np.random.default_rng(3)
    s = g.normal(size=(1, 4, 1000)).astype(np.float32)
    ev_all, cnt, _ = oracle.detect(s, 1000, 1.0)
    ev, cnt2, _ = oracle.detect(s, 1000, 1.0, max_events=10)
    assert cnt2 == cnt > 10 and len(ev) == 10 and len(ev_all) == cnt


def test_noise_false_alarm_rate():
    from math import erfc, sqrt
    g = np.random.default_rng(4)
    s = g.normal(size=(4, 64, 8192)).astype(np.float32) * 8
    thr = 3.5
    ev, cnt, st = oracle.detect(s, 8192, thr)
    exp = 0.5 * erfc(thr / sqrt(2)) * s.size
    assert 0.8 * exp < cnt < 1.2 * exp
    assert np.all(np.abs(st[..., 0]) < 0.5) and np.all(np.abs(st[..., 1] - 8) < 0.3)


def test_cfg1_chain_strongest_event():
    """P7: cfg 1's injected pulse is the strongest event, at dm_idx 20, t in [1000,1003], SNR ~ 19."""
    cfg = CONFIGS[1]
    x = generate(cfg)
    d = oracle.delay_table(cfg.nchans, cfg.f_top, cfg.foff, cfg.tsamp, cfg.dm_low, cfg.dm_step, cfg.ndms)
    out, _ = oracle.dedisperse(x, d)
    ev, cnt, st = oracle.detect(out, out.shape[2], 6.0)
    top = ev[np.argmax(ev["snr"])]
    assert top["dm_idx"] == 20 and 1000 <= top["t"] <= 1003
    assert 15 < top["snr"] < 23
    assert 9.0 < st[0, 20, 1] < 11.5          # rms ~ 10.1: sqrt(64)=8 inflated by the pulse
    # every event belongs to the pulse's bow-tie in (DM, t): no noise events at 6 sigma in 126k samples
    assert np.all(np.abs(ev["t"] - 1001.5) < 60)
