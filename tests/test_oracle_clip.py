"""Pins for oracle.rfi_clip (reading B).  The threshold CHOICE (per-buffer
mean + k*sigma) has no worked numbers in the paper: pinned by invariants only (P6)."""
import math

import numpy as np
import pytest

import oracle


def noise(nb=1, nc=16, ns=4096, seed=0, dtype=np.float32):
    g = np.random.default_rng(seed)
    x = g.normal(size=(nb, nc, ns))
    if dtype == np.uint8:
        return np.clip(np.rint(64 + 10 * x), 0, 255).astype(np.uint8)
    return x.astype(np.float32)


@pytest.mark.parametrize("dtype", [np.float32, np.uint8])
def test_constant_input_no_flags(dtype):
    x = np.full((2, 8, 1024), 7, dtype=dtype)
    r = oracle.rfi_clip(x, 64, 5.0, 5.0)
    assert r["chan_mask"].sum() == 0 and r["spec_mask"].sum() == 0
    assert np.all(x == 7)


@pytest.mark.parametrize("dtype", [np.float32, np.uint8])
def test_single_chunk_and_dilation(dtype):
    W = 64
    x = noise(dtype=dtype, seed=1)
    x0 = x.copy()
    c, j = 5, 20
    x[0, c, j * W:(j + 1) * W] += dtype(100) if dtype == np.uint8 else np.float32(50.0)
    xin = x.copy()
    r = oracle.rfi_clip(x, W, 6.0, 1e9, debug=True)
    want = np.zeros_like(r["chan_mask"])
    want[0, c, j - 1:j + 2] = 1                         # the chunk and its immediate neighbours in time (B-ii)
    assert np.array_equal(r["chan_mask"], want)
    assert r["spec_mask"].sum() == 0
    repl = r["repl"][0, c]
    assert np.all(x[0, c, (j - 1) * W:(j + 2) * W] == dtype(repl))          # replaced by the channel value (B-iii)
    keep = np.ones(x.shape, bool)
    keep[0, c, (j - 1) * W:(j + 2) * W] = False
    assert np.array_equal(x[keep], xin[keep])           # everything else untouched
    # repl is the pre-clip channel mean (u8: rounded half up)
    m = xin[0, c].astype(np.float64).mean()
    if dtype == np.uint8:
        assert repl == math.floor(m + 0.5)
    else:
        assert repl == np.float32(r["chan_mean"][0, c])
        assert abs(r["chan_mean"][0, c] - m) < 1e-9
    assert abs(r["chan_sig"][0, c] - xin[0, c].astype(np.float64).std()) < 1e-9
    del x0


def test_edge_chunks_dilate_inside_only():
    W = 32
    x = noise(seed=2)
    x[0, 3, :W] += 40.0
    x[0, 9, -W:] += 40.0
    r = oracle.rfi_clip(x, W, 6.0, 1e9)
    m = r["chan_mask"][0]
    assert m[3].nonzero()[0].tolist() == [0, 1]
    n = m.shape[1]
    assert m[9].nonzero()[0].tolist() == [n - 2, n - 1]
    assert m.sum() == 4


@pytest.mark.parametrize("dtype", [np.float32, np.uint8])
def test_single_spectrum_spike(dtype):
    x = noise(nc=64, dtype=dtype, seed=3)
    xin = x.copy()
    t = 777
    x[0, :, t] += dtype(60)
    r = oracle.rfi_clip(x, 64, 1e9, 5.0, debug=True)
    assert r["chan_mask"].sum() == 0
    assert r["spec_mask"][0].nonzero()[0].tolist() == [t]
    assert np.array_equal(x[0, :, t].astype(np.float64), r["repl"][0])      # spectrum := per-channel value
    keep = np.ones(x.shape, bool)
    keep[0, :, t] = False
    assert np.array_equal(x[keep], xin[keep])
    # debug spectrum sums are the sums of the data B3 saw
    xs = xin.copy()
    xs[0, :, t] += dtype(60)
    assert np.allclose(r["spec_sum"][0], xs[0].astype(np.float64).sum(axis=0))


def test_order_channel_stage_before_spectrum_stage():
    """B-iv: the spectrum stage sees the data as modified by the channel stage."""
    W = 64
    x = noise(nc=8, seed=4)
    # one very strong narrowband chunk: alone it would also push its spectra over the spectrum threshold
    x[0, 2, 10 * W:11 * W] += 400.0
    a = x.copy()
    ra = oracle.rfi_clip(a, W, 5.0, 5.0)
    assert ra["chan_mask"][0, 2, 9:12].all()
    assert ra["spec_mask"][0, 10 * W:11 * W].sum() == 0        # already removed by the channel stage
    b = x.copy()
    rb = oracle.rfi_clip(b, W, 1e9, 5.0)                       # channel stage disabled
    assert rb["spec_mask"][0, 10 * W:11 * W].all()


def test_one_sided():
    """B-v: only excess power is flagged; zeroed packet-loss gaps are not."""
    W = 64
    x = noise(seed=5) + np.float32(10.0)
    x[0, 4, 5 * W:6 * W] = 0.0
    x[0, :, 2000] = 0.0
    r = oracle.rfi_clip(x, W, 5.0, 5.0)
    assert r["chan_mask"].sum() == 0 and r["spec_mask"].sum() == 0


@pytest.mark.parametrize("dtype", [np.float32, np.uint8])
def test_post_clip_never_exceeds_threshold(dtype):
    """P6(ii) / north_star: clipped samples must never exceed the threshold."""
    W = 64
    g = np.random.default_rng(6)
    x = noise(nb=2, nc=32, ns=8192, dtype=dtype, seed=6)
    for _ in range(12):
        b, c, j = g.integers(2), g.integers(32), g.integers(8192 // W)
        x[b, c, j * W:(j + 1) * W] = np.clip(x[b, c, j * W:(j + 1) * W].astype(np.float64) + 40, 0, 255).astype(dtype)
    for _ in range(5):
        b, t = g.integers(2), g.integers(8192)
        x[b, :, t] = np.clip(x[b, :, t].astype(np.float64) + 60, 0, 255).astype(dtype)
    r = oracle.rfi_clip(x, W, 5.0, 5.0, debug=True)
    assert r["chan_mask"].sum() >= 12 and r["spec_mask"].sum() >= 5
    csum = x.astype(np.float64).reshape(2, 32, -1, W).sum(axis=3)
    # after B3 every chunk sum is <= its threshold, every spectrum sum <= its threshold
    assert np.all(csum <= r["chan_thr"][:, :, None])
    ssum = x.astype(np.float64).sum(axis=1)
    assert np.all(ssum <= r["spec_thr"][:, 0:1])
    # flagged units hold the replacement value
    cm = np.repeat(r["chan_mask"], W, axis=2).astype(bool)
    sm = np.broadcast_to(r["spec_mask"][:, None, :].astype(bool), x.shape)
    repl = np.broadcast_to(r["repl"][:, :, None], x.shape)
    assert np.all(x[cm | sm].astype(np.float64) == repl[cm | sm])


def test_gaussian_flag_rates():
    """P6(v): noise -> raw chunk flag rate Q(k), dilated ~3Q(k); spectrum flag rate Q(k)."""
    from math import erfc, sqrt
    k = 2.5
    q = 0.5 * erfc(k / sqrt(2))
    x = noise(nb=1, nc=64, ns=65536, seed=7)
    r = oracle.rfi_clip(x.copy(), 16, k, 1e9)
    rate = r["chan_mask"].mean()
    assert 2.3 * q < rate < 3.2 * q
    x = noise(nb=1, nc=64, ns=65536, seed=8)
    r = oracle.rfi_clip(x, 16, 1e9, k)
    assert 0.7 * q < r["spec_mask"].mean() < 1.3 * q


def test_bad_window():
    with pytest.raises(ValueError):
        oracle.rfi_clip(noise(ns=1000), 64, 5, 5)


def test_u8_threshold_arithmetic_by_hand():
    """A 2-channel, 8-sample case worked by hand from the rules B1-B3."""
    x = np.array([[[10, 10, 10, 10, 10, 10, 50, 50],
                   [20, 20, 20, 20, 20, 20, 20, 20]]], dtype=np.uint8)
    # channel 0: S=160, N=8 -> mean 20, Q=6*100+2*2500=5600 -> var 700-400=300, sig=17.32
    # W=2: thr = 2*20 + k*17.32*sqrt(2); chunk sums 20,20,20,100. k=2 -> thr=88.99 -> chunk 3 flagged, 2 by dilation
    r = oracle.rfi_clip(x, 2, 2.0, 1e9, debug=True)
    assert r["chan_mask"][0].tolist() == [[0, 0, 1, 1], [0, 0, 0, 0]]
    assert abs(r["chan_thr"][0, 0] - (40 + 2 * math.sqrt(300) * math.sqrt(2))) < 1e-12
    assert x[0, 0].tolist() == [10, 10, 10, 10, 20, 20, 20, 20]     # repl = (160+4)//8 = 20
    assert r["repl"][0].tolist() == [20.0, 20.0]


def test_channel_threshold_tie_is_not_a_flag_strict_greater():
    """Reading B-v / PAPER.md:79 "exceeds": a chunk sum EQUAL to the threshold is not flagged.  Worked by hand:
    x = 0,0,0,0,4,4,4,4: mean 2, Q/N = 8, var 4, sig 2; W = 4: thr = 4*2 + k*2*sqrt(4) = 8 + 4k; chunk sums 0, 16."""
    def run(k):
        x = np.array([[[0, 0, 0, 0, 4, 4, 4, 4]]], dtype=np.uint8)
        r = oracle.rfi_clip(x, 4, k, 1e9, debug=True)
        return r, x
    r, x = run(2.0)                                            # thr = 16 = the second chunk's sum
    assert r["chan_thr"][0, 0] == 16.0 and not r["chan_mask"].any() and x[0, 0].tolist() == [0, 0, 0, 0, 4, 4, 4, 4]
    r, x = run(1.9999)                                         # just below: flagged, its neighbour by dilation, both replaced by 2
    assert r["chan_mask"][0, 0].tolist() == [1, 1] and x[0, 0].tolist() == [2] * 8


def test_spectrum_threshold_by_hand_and_its_tie():
    """B3 worked by hand: two channels 0,2 -> spectrum sums s = 0, 4: mean_s 2, M2/N = 8, var 4, sig 2;
    thr = 2 + 2 k_spec.  k_spec = 1 -> thr = 4 = s_1: not flagged (strict); k_spec = 0.999 -> flagged and replaced by
    repl_c = (2 + 1) // 2 = 1."""
    def run(k):
        x = np.array([[[0, 2], [0, 2]]], dtype=np.uint8)
        r = oracle.rfi_clip(x, 1, 1e9, k, debug=True)
        return r, x
    r, x = run(1.0)
    assert r["spec_thr"][0].tolist() == [4.0, 2.0, 2.0]
    assert not r["spec_mask"].any() and x[0].tolist() == [[0, 2], [0, 2]]
    r, x = run(0.999)
    assert r["spec_mask"][0].tolist() == [0, 1] and x[0].tolist() == [[0, 1], [0, 1]]
    assert abs(r["spec_thr"][0, 0] - 3.998) < 1e-12
