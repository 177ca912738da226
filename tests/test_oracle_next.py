"""Pins of the oracle functions for the SURVEY 8(f) rows (oracle/mdsm_oracle_next.c): each check is something other
than the oracle's own formula -- numpy.polyfit, scikit-learn's DBSCAN, closed forms, hand-worked cases, invariants."""
import math

import numpy as np
import pytest

import oracle


# ------------------------------------------------------------------ bandpass stage
@pytest.mark.parametrize("order", [0, 1, 3, 6, 8])
def test_polyfit_matches_numpy_polyfit(order):
    g = np.random.default_rng(order)
    n = 200
    y = g.normal(size=n) + np.linspace(0, 3, n) ** 2
    u = 2.0 * np.arange(n) / (n - 1) - 1.0
    ref = np.polyfit(u, y, order)[::-1]                      # library routine (SVD least squares), ascending powers
    got = oracle.polyfit_u(y, order)
    assert np.allclose(got, ref, rtol=1e-8, atol=1e-9)


def _poly_bandpass(nchans):
    u = 2.0 * np.arange(nchans) / (nchans - 1) - 1.0
    return 1.0 + 0.5 * u - 0.25 * u * u                       # exactly representable when nchans - 1 is a power of two


def test_polynomial_bandpass_is_recovered_exactly_and_nothing_is_flagged():
    nc, ns = 17, 256
    bp = _poly_bandpass(nc)
    x = np.repeat(bp[None, :, None], ns, axis=2).astype(np.float32)
    assert np.array_equal(x[0, :, 0].astype(np.float64), bp)  # the fp32 data carries the polynomial exactly
    r = oracle.bandpass_clip(x, 16, 2, 5.0, 5.0, 5.0, subtract=False)
    assert np.allclose(r["fit"][0], bp, atol=1e-12) and r["rmse"][0] < 1e-12
    assert r["nmasked"][0] == 0 and not r["chan_mask"].any() and not r["spec_mask"].any()
    assert abs(r["mean_bp"][0] - bp.mean()) < 1e-12 and abs(r["std_bp"][0] - bp.std()) < 1e-12


def test_rfi_channels_are_masked_and_interpolated_before_the_fit():
    nc, ns = 33, 128
    bp = _poly_bandpass(nc)
    dirty = bp.copy()
    dirty[7] += 4.0
    dirty[20] += 8.0
    dirty[21] += 8.0                                          # two adjacent RFI channels: nearest clean neighbours are 19, 22
    x = np.repeat(dirty[None, :, None], ns, axis=2).astype(np.float32)
    r = oracle.bandpass_clip(x, 16, 2, 5.0, 1e9, 1e9, subtract=False)
    assert r["nmasked"][0] == 3
    assert r["bpi"][0, 7] == 0.5 * (bp[6] + bp[8])
    assert r["bpi"][0, 20] == 0.5 * (bp[19] + bp[22]) and r["bpi"][0, 21] == 0.5 * (bp[19] + bp[22])
    clean = np.delete(np.arange(nc), [7, 20, 21])
    assert np.array_equal(r["bpi"][0, clean], bp[clean])
    # the interpolated values are not on the parabola, but they move the fit by far less than the RFI would have
    assert np.abs(r["fit"][0] - bp).max() < 0.02
    r2 = oracle.bandpass_clip(np.repeat(dirty[None, :, None], ns, axis=2).astype(np.float32), 16, 2, 1e9, 1e9, 1e9, subtract=False)
    assert r2["nmasked"][0] == 0 and np.abs(r2["fit"][0] - bp).max() > 0.5


def test_band_edge_channel_takes_its_only_clean_neighbour():
    nc, ns = 9, 64
    bp = np.full(nc, 2.0)
    bp[0] = 9.0
    x = np.repeat(bp[None, :, None], ns, axis=2).astype(np.float32)
    r = oracle.bandpass_clip(x, 8, 0, 3.0, 1e9, 1e9, subtract=False)
    assert r["nmasked"][0] == 1 and r["bpi"][0, 0] == 2.0 and np.allclose(r["fit"][0], 2.0, atol=1e-14)


def test_mask_limit_is_k_times_1_4826_mad_pinned_from_both_sides():
    """Reading H-ii: a channel is masked when bp - median > k_mask * 1.4826 * MAD.  bp = 1..9: median 5, deviations
    4,3,2,1,0,1,2,3,4, MAD 2, so the limit is 2.9652 * k_mask.  Channel 8 (bp = 9, 4 above the median) sits exactly on the
    limit at k_mask = 4 / 2.9652 = 1.34898...: k = 1.3489 masks it (limit 3.99976), k = 1.3491 does not (4.00035), which
    pins the constant to 1.4826 +- 0.0001; k = 1.3 masks channel 8 only, where a limit of k * MAD (no 1.4826: 2.6) would
    also take channel 7 (3 above), and k * 1.4826 * std (std = 2.582: 4.98) would take none."""
    bp = np.arange(1.0, 10.0)
    x = np.repeat(bp[None, :, None], 64, axis=2).astype(np.float32)
    for k_mask, masked in ((1.3489, [8]), (1.3491, []), (1.3, [8]), (1.0, [7, 8]), (0.68, [7, 8]), (0.67, [6, 7, 8])):
        r = oracle.bandpass_clip(x.copy(), 8, 0, k_mask, 1e9, 1e9, subtract=False)
        got = np.flatnonzero(r["bpi"][0] != bp).tolist()
        assert r["nmasked"][0] == len(masked) and got == masked, (k_mask, got)


def test_constant_input_order0_no_flags_strict_comparison():
    x = np.full((2, 8, 256), 3.0, dtype=np.float32)
    r = oracle.bandpass_clip(x, 32, 0, 5.0, 0.0, 0.0, subtract=False)     # k = 0: thresholds sit exactly on the data
    assert not r["chan_mask"].any() and not r["spec_mask"].any() and np.all(x == 3.0)
    assert np.all(r["rmse"] == 0) and np.all(r["std_bp"] == 0) and np.all(r["fit"] == 3.0)


def test_hand_worked_channel_and_spectrum_flags_replacement_and_subtraction():
    nc, ns, W = 17, 512, 32
    bp = _poly_bandpass(nc)
    x = np.repeat(bp[None, :, None], ns, axis=2).astype(np.float32)
    x[0, 4, 5 * W:6 * W] += 1.0                              # one chunk of channel 4 raised: chunks 4, 5, 6 must be flagged
    x[0, :, 300] += 2.0                                      # one broadband spike at t = 300
    x0 = x.copy()
    # in numbers: bp[4] rises by 1/16, every bp[c] by 2/512; the order-2 fit absorbs the constant and misses the 1/16 by
    # rmse ~ 0.014, so k_chan = 10 puts the channel threshold ~0.14 above the fit: only the raised chunk (1.0 above)
    # exceeds it.  std_bp ~ 0.2 (the parabola), so k_spec = 0.5 puts the spectrum threshold ~0.1 above mean_bp: only
    # t = 300 (2.0 above) exceeds it.
    r = oracle.bandpass_clip(x, W, 2, 5.0, 10.0, 0.5, subtract=True)
    assert 0.005 < r["rmse"][0] < 0.03 and 0.1 < r["std_bp"][0] < 0.4 and r["nmasked"][0] == 0
    cm = r["chan_mask"][0]
    expect = np.zeros_like(cm)
    expect[4, 4:7] = 1
    assert np.array_equal(cm, expect)
    assert np.flatnonzero(r["spec_mask"][0]).tolist() == [300]
    fit32 = r["fit"][0].astype(np.float32)
    # flagged samples were replaced by the fitted bandpass value and are exactly 0 after the subtraction
    assert np.all(x[0, 4, 4 * W:7 * W] == 0.0) and np.all(x[0, :, 300] == 0.0)
    keep = np.ones((nc, ns), dtype=bool)
    keep[4, 4 * W:7 * W] = False
    keep[:, 300] = False
    assert np.array_equal(x[0][keep], (x0[0] - fit32[:, None])[keep])


def test_bad_arguments():
    x = np.zeros((1, 4, 64), dtype=np.float32)
    with pytest.raises(ValueError):
        oracle.bandpass_clip(x, 48, 1, 5, 5, 5, False)        # window does not divide nsamps (reading B-viii)
    with pytest.raises(ValueError):
        oracle.bandpass_clip(x, 16, 4, 5, 5, 5, False)        # order >= nchans


# ------------------------------------------------------------------ clustering
def _blobs(seed, nblob=6, per=40, nnoise=60):
    g = np.random.default_rng(seed)
    pts = []
    for _ in range(nblob):
        c = g.uniform([0, 0, 6], [4000, 60, 30])
        pts.append(c + g.normal(size=(per, 3)) * [6.0, 1.5, 1.0])
    pts.append(g.uniform([0, 0, 6], [4000, 60, 30], size=(nnoise, 3)))
    pts = np.concatenate(pts)
    g.shuffle(pts)
    return pts


def _same_partition(a, b):
    pairs = set(zip(a.tolist(), b.tolist()))
    return len(pairs) == len(set(a.tolist())) == len(set(b.tolist()))


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_dbscan_matches_scikit_learn_on_core_points_and_noise(seed):
    sk = pytest.importorskip("sklearn.cluster")
    pts = _blobs(seed)
    eps = np.array([8.0, 2.0, 1.5])
    min_pts = 5
    lab, ncl = oracle.dbscan(pts, eps, min_pts)
    ref = sk.DBSCAN(eps=1.0, min_samples=min_pts, metric="chebyshev").fit(pts / eps)     # box = unit Chebyshev ball
    core = np.zeros(len(pts), dtype=bool)
    core[ref.core_sample_indices_] = True
    assert np.array_equal(lab == -1, ref.labels_ == -1)
    assert ncl == ref.labels_.max() + 1
    assert _same_partition(lab[core], ref.labels_[core])


def test_dbscan_hand_worked_chain_and_noise():
    t = np.array([0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 50, 100, 101, 102], dtype=np.float64)
    pts = np.stack([t, np.zeros_like(t), np.zeros_like(t)], axis=1)
    lab, ncl = oracle.dbscan(pts, [1.5, 1.0, 1.0], 3)
    assert ncl == 2 and lab.tolist() == [0] * 10 + [-1] + [1, 1, 1]
    labf, nclf, nq = oracle.fdbscan(pts, [1.5, 1.0, 1.0], 3)
    assert nclf == 2 and labf.tolist() == lab.tolist()


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_fdbscan_clusters_refine_dbscan_clusters_with_fewer_queries(seed):
    pts = _blobs(seed, nblob=8, per=60, nnoise=100)
    eps = np.array([8.0, 2.0, 1.5])
    lab, _ = oracle.dbscan(pts, eps, 5)
    labf, nclf, nq = oracle.fdbscan(pts, eps, 5)
    assert nq < len(pts)                                       # the point of FDBSCAN
    # every FDBSCAN cluster lies inside ONE DBSCAN cluster (it only ever follows density-reachability) ...
    for c in range(nclf):
        inside = set(lab[labf == c].tolist())
        assert len(inside) == 1 and -1 not in inside
    # ... and DBSCAN's noise stays noise
    assert np.all(labf[lab == -1] == -1)
    # "some points might be lost ... however the probability of this happening is very low"
    assert np.mean(labf[lab >= 0] >= 0) > 0.95


def test_fdbscan_equals_dbscan_on_compact_separated_blobs():
    g = np.random.default_rng(9)
    centres = np.array([[100, 10, 10], [500, 30, 12], [900, 50, 20]], dtype=np.float64)
    pts = np.concatenate([c + g.uniform(-0.4, 0.4, size=(30, 3)) * [8.0, 2.0, 1.5] for c in centres])   # each inside one box
    lab, ncl = oracle.dbscan(pts, [8.0, 2.0, 1.5], 4)
    labf, nclf, nq = oracle.fdbscan(pts, [8.0, 2.0, 1.5], 4)
    assert ncl == nclf == 3 and np.array_equal(lab, labf)


def _pins():
    import os
    import runpy
    return runpy.run_path(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "fdbscan_pins.py"))


@pytest.mark.parametrize("name", ["split", "lost", "other"])
def test_fdbscan_hand_worked_sets_labels_and_query_counts(name):
    """PAPER.md:126, reading K-ii.  Expected labels and query counts are written out by hand in tests/golden/fdbscan_pins.py
    (walk-through above each set), not produced by the oracle.  Each set fails for one plausible one-line misreading, and this
    was checked by applying the mutation to oracle/mdsm_oracle_next.c (orc_fdbscan) and re-running this test:
      split -- `v > bestv` turned into "nearest" (smallest positive v): labels become one cluster;
      lost  -- `v > bestv` -> `v >= bestv` (ties to the higher index): points 3 and 4 join the cluster;
      other -- the `label[r] != cid` filter removed (representatives among all neighbours): point 8 becomes noise.
    The DBSCAN labels of the same sets are pinned by scikit-learn, so "split" exhibits the paper's "clusters might be split
    apart" and "lost" its "some points might be lost" against an independent exact clustering."""
    sk = pytest.importorskip("sklearn.cluster")
    S = _pins()["SETS"][name]
    pts = np.array([(t, d, 10.0) for t, d in S["pts"]], dtype=np.float64)
    eps = np.array([S["eps"], S["eps"], 1.0])
    lab, ncl, nq = oracle.fdbscan(pts, eps, S["min_pts"])
    assert lab.tolist() == S["fdbscan_labels"], S["fails_for"]
    assert ncl == max(S["fdbscan_labels"]) + 1 and nq == S["fdbscan_queries"], S["fails_for"]
    ref = sk.DBSCAN(eps=1.0, min_samples=S["min_pts"], metric="chebyshev").fit(pts / eps)
    assert ref.labels_.tolist() == S["dbscan_labels"]
    assert oracle.dbscan(pts, eps, S["min_pts"])[0].tolist() == S["dbscan_labels"]
    # the same set with the second coordinate in the SNR dimension instead of DM: dimension 2 is treated like the others
    pts3 = np.array([(t, 3.0, d) for t, d in S["pts"]], dtype=np.float64)
    lab3, _, nq3 = oracle.fdbscan(pts3, np.array([S["eps"], 1.0, S["eps"]]), S["min_pts"])
    assert lab3.tolist() == S["fdbscan_labels"] and nq3 == S["fdbscan_queries"]


@pytest.mark.parametrize("dim", [0, 1, 2])
@pytest.mark.parametrize("sign", [1, -1])
def test_fdbscan_chain_along_every_dimension_and_direction(dim, sign):
    """"Two for each dimension, one for each direction": a row of points along one axis is followed to its
    end through the far representative only (4 queries for 7 points; the nearest-representative misreading needs 7, a
    dimension or direction left out breaks the row into several clusters)."""
    C = _pins()["CHAIN"]
    pts = np.zeros((C["n"], 3))
    pts[:, 2] = 10.0
    pts[:, dim] += sign * C["step"] * np.arange(C["n"])
    lab, ncl, nq = oracle.fdbscan(pts, [C["eps"]] * 3, C["min_pts"])
    assert ncl == 1 and lab.tolist() == [0] * C["n"] and nq == C["fdbscan_queries"], C["fails_for"]


# ------------------------------------------------------------------ classifier (Eqs. 3, 4)
def test_eq3_closed_form_values():
    assert oracle.dm_response(0.0) == 1.0
    assert abs(oracle.dm_response(1.0) - 0.5 * math.sqrt(math.pi) * math.erf(1.0)) < 1e-15
    assert abs(oracle.dm_response(1.0) - 0.7468241328) < 1e-9          # sqrt(pi)/2 erf(1), tabulated
    assert abs(oracle.dm_response(100.0) - math.sqrt(math.pi) / 200.0) < 1e-15      # erf -> 1
    assert abs(oracle.dm_response(1e-4) - (1 - 1e-8 / 3)) < 1e-12       # series: 1 - zeta^2/3
    assert oracle.dm_response(-2.0) == oracle.dm_response(2.0)


def test_eq4_printed_constant():
    # BEST-2: 20 MHz at 408 MHz, a 1 ms pulse 1 pc/cm^3 off: 6.91e-3 * 1 * 20 / (1 * 0.408^3) = 2.0348...
    assert abs(oracle.zeta(1.0, 20.0, 1.0, 0.408) - 2.03479) < 1e-4
    assert oracle.zeta(2.0, 20.0, 1.0, 0.408) == 2 * oracle.zeta(1.0, 20.0, 1.0, 0.408)
    assert abs(oracle.zeta(1.0, 20.0, 2.0, 0.408) - 0.5 * oracle.zeta(1.0, 20.0, 1.0, 0.408)) < 1e-15


def _model_cluster(d0, width, snr0, dm_step=0.1, tsamp=51.2e-6, bw=20.0, nu=0.408, thr=0.3, dm_low=0.0):
    t, d, s = [], [], []
    w_ms = width * tsamp * 1e3
    for di in range(d0 - 200, d0 + 201):
        if di < 0:
            continue
        z = 6.91e-3 * ((di - d0) * dm_step) * bw / (w_ms * nu ** 3)
        resp = 1.0 if z == 0 else 0.5 * math.sqrt(math.pi) * math.erf(abs(z)) / abs(z)
        if resp < thr:
            continue
        # at the true DM the pulse fills `width` samples; off it, fewer detections survive: one (the strongest) is enough
        n = width if di == d0 else 1
        for k in range(n):
            t.append(1000 + k); d.append(di); s.append(snr0 * resp * (1.0 if k == 0 else 0.9))
    return np.array(t), np.array(d), np.array(s, dtype=np.float32), w_ms


def test_classifier_accepts_a_cluster_drawn_from_the_model_curve():
    t, d, s, w_ms = _model_cluster(d0=300, width=8, snr0=20.0)
    r = oracle.classify_cluster(t, d, s, 0.0, 0.1, 51.2e-6, 20.0, 0.408, 1, 0.05)
    assert r["cls"] == 0 and r["dm_idx"] == 300 and abs(r["snr"] - 20.0) < 1e-6
    assert abs(r["width_ms"] - w_ms) < 1e-12 and r["rmse"] < 1e-6


def test_classifier_discards_low_dm_and_flat_signatures():
    t, d, s, _ = _model_cluster(d0=5, width=8, snr0=20.0)              # DM 0.5 < 1.0: broadband RFI (step 3)
    r = oracle.classify_cluster(t, d, s, 0.0, 0.1, 51.2e-6, 20.0, 0.408, 1, 0.05)
    assert r["cls"] == 1 and r["dm_idx"] == 5
    dd = np.arange(100, 400)
    tt = np.concatenate([[1000, 1001, 1002], np.full(len(dd) - 1, 1000)])
    dflat = np.concatenate([[250, 250, 250], np.delete(dd, 150)])
    flat = oracle.classify_cluster(tt, dflat, np.full(len(tt), 9.0, dtype=np.float32), 0.0, 0.1, 51.2e-6, 20.0, 0.408, 1, 0.05)
    assert flat["cls"] == 2 and flat["dm_idx"] == 250 and flat["rmse"] > 0.5      # SNR does not fall off with DM: RFI


def test_classifier_hand_worked_three_dm_cluster_with_smoothing():
    # DMs 20.0, 20.1, 20.2; detections: d=200: snr 6; d=201: snr 10, 9, 8 at t = 50, 51, 53; d=202: snr 4
    t = np.array([50, 50, 51, 53, 52]); d = np.array([200, 201, 201, 201, 202]); s = np.array([6, 10, 9, 8, 4], dtype=np.float32)
    r = oracle.classify_cluster(t, d, s, 0.0, 0.1, 1e-3, 20.0, 0.408, 3, 10.0)
    assert r["dm_idx"] == 201 and r["snr"] == 10.0 and abs(r["width_ms"] - 4.0) < 1e-12     # (53 - 50 + 1) * 1 ms
    sm = np.array([(6 + 10) / 2, (6 + 10 + 4) / 3, (10 + 4) / 2])                            # 3-element moving average, clipped
    sig = sm / sm.max()
    z = 6.91e-3 * 0.1 * 20.0 / (4.0 * 0.408 ** 3)
    m = 0.5 * math.sqrt(math.pi) * math.erf(z) / z
    rmse = math.sqrt(((m - sig[0]) ** 2 + (1 - sig[1]) ** 2 + (m - sig[2]) ** 2) / 3)
    assert abs(r["rmse"] - rmse) < 1e-12


# ------------------------------------------------------------------ 4-bit quantiser
def test_mulaw_c4_end_points_sign_and_packing():
    v = np.array([[0, 0], [1000, -1000], [-1, 1], [1000, 0]], dtype=np.int16)
    out, xmax = oracle.mulaw_c4(v, 255.0)
    assert xmax == 1000
    assert out[0] == 0x00
    assert out[1] == (7 | ((-7 & 15) << 4))                    # +Xmax -> +7, -Xmax -> -7 = nibble 0x9
    assert out[3] == 7
    # |v| = 1 of 1000 at mu = 255: 7 * log(1.255)/log(256) = 0.287 -> 0
    assert out[2] == 0


def test_mulaw_c4_code_boundaries_are_the_inverse_law():
    mu, xmax = 255.0, 32767
    v = np.arange(0, xmax + 1, dtype=np.int32)
    volt = np.stack([v, -v], axis=1).astype(np.int16)
    out, xm = oracle.mulaw_c4(volt, mu)
    assert xm == xmax
    re = (out & 15).astype(np.int32)
    im = (out >> 4).astype(np.int32)
    im = np.where(im >= 8, im - 16, im)
    assert np.array_equal(im, -re) and np.all(np.diff(re) >= 0) and re[0] == 0 and re[-1] == 7
    for k in range(1, 8):
        # code >= k  <=>  |v|/Xmax >= ((1 + mu)^((k - 1/2)/7) - 1)/mu   (Eq. 5 inverted)
        edge = xmax * ((1 + mu) ** ((k - 0.5) / 7) - 1) / mu
        first = int(np.argmax(re >= k))
        assert first == math.ceil(edge), (k, first, edge)


# ------------------------------------------------------------------ 16-bit / 4-bit dedispersion input
def test_dedisperse_u16_matches_numpy_gather_sum_and_the_u8_oracle():
    g = np.random.default_rng(3)
    nb, nc, ns, nd = 2, 12, 300, 7
    delay = oracle.delay_table(nc, 418.0, -1.5, 51.2e-6, 0.0, 0.4, nd)
    x = g.integers(0, 65536, size=(nb, nc, ns), dtype=np.uint16)
    out = oracle.dedisperse_u16(x, delay)
    nso = ns - int(delay.max())
    ref = np.zeros((nb, nd, nso), dtype=np.uint64)
    for d in range(nd):
        for c in range(nc):
            ref[:, d, :] += x[:, c, delay[d, c]:delay[d, c] + nso]
    assert np.array_equal(out.astype(np.uint64), ref)
    x8 = g.integers(0, 256, size=(nb, nc, ns), dtype=np.uint8)
    o8, _ = oracle.dedisperse(x8, delay)
    assert np.array_equal(oracle.dedisperse_u16(x8.astype(np.uint16), delay), o8)


def test_unpack_u4_nibble_order():
    x = np.array([[0x21, 0xF0]], dtype=np.uint8)
    assert oracle.unpack_u4(x).tolist() == [[1, 2, 0, 15]]
