"""Host candidate stage of the library (mdsm_cluster_events, mdsm_classify_clusters) against the oracle.
Host-only code: runs without a GPU.  Labels must be IDENTICAL (same visiting order, same tie-breaks), the grid index only
replaces the oracle's O(N^2) neighbourhood scan."""
import numpy as np
import pytest

import oracle
import paper_1307_5700_b200 as m

DM_LOW, DM_STEP, TSAMP = 0.0, 0.1, 51.2e-6
BW, NU = 20.0, 0.408


def _events(seed, nbeams=1, nblob=10, per=80, nnoise=300):
    """Synthetic detection lists: dispersed-pulse-like blobs (narrow in time near the centre DM, SNR falling off with DM
    distance) plus uniformly scattered noise events."""
    g = np.random.default_rng(seed)
    ev = []
    for b in range(nbeams):
        for _ in range(nblob):
            t0, d0, s0 = g.integers(100, 60000), g.integers(20, 600), g.uniform(8, 30)
            dd = g.integers(-25, 26, size=per)
            tt = t0 - 2 * dd + g.integers(-3, 4, size=per)
            ss = 6.0 + (s0 - 6.0) * np.exp(-(dd / 12.0) ** 2) + g.normal(size=per) * 0.3
            for k in range(per):
                ev.append((b, int(np.clip(d0 + dd[k], 0, 639)), int(max(0, tt[k])), np.float32(ss[k])))
        for _ in range(nnoise):
            ev.append((b, int(g.integers(0, 640)), int(g.integers(0, 62000)), np.float32(g.uniform(6, 7))))
    ev = np.array(ev, dtype=[("beam", "<i4"), ("dm_idx", "<i4"), ("t", "<i4"), ("snr", "<f4")])
    g.shuffle(ev)
    return ev.astype(m.EVENT_DTYPE)


def _points(ev):
    return np.stack([ev["t"].astype(np.float64), DM_LOW + ev["dm_idx"].astype(np.float64) * DM_STEP, ev["snr"].astype(np.float64)], axis=1)


@pytest.mark.parametrize("exact", [False, True])
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_clustering_labels_identical_to_the_oracle(seed, exact):
    ev = _events(seed)
    eps = (8.0, 0.5, 4.0)
    lab, ncl, nq = m.mdsm_cluster_events(ev, DM_LOW, DM_STEP, *eps, 5, exact=exact)
    if exact:
        ref, nref = oracle.dbscan(_points(ev), eps, 5)
    else:
        ref, nref, nq_ref = oracle.fdbscan(_points(ev), eps, 5)
        assert nq == nq_ref and nq < len(ev)
    assert ncl == nref and ncl >= 8 and np.array_equal(lab, ref)


def test_beams_are_clustered_separately_and_ids_continue():
    ev = _events(7, nbeams=3, nblob=4, per=60, nnoise=100)
    eps = (8.0, 0.5, 4.0)
    lab, ncl, _ = m.mdsm_cluster_events(ev, DM_LOW, DM_STEP, *eps, 5)
    first = 0
    order = []
    for b in ev["beam"]:
        if b not in order:
            order.append(int(b))
    for b in order:
        sel = ev["beam"] == b
        ref, nref, _ = oracle.fdbscan(_points(ev[sel]), eps, 5)
        expect = np.where(ref >= 0, ref + first, -1)
        assert np.array_equal(lab[sel], expect)
        first += nref
    assert first == ncl


def test_degenerate_inputs_and_errors():
    empty = np.zeros(0, dtype=m.EVENT_DTYPE)
    lab, ncl, nq = m.mdsm_cluster_events(empty, 0.0, 0.1, 8.0, 0.5, 4.0, 5)
    assert lab.size == 0 and ncl == 0 and nq == 0
    one = np.array([(0, 5, 10, 7.0)], dtype=m.EVENT_DTYPE)
    lab, ncl, _ = m.mdsm_cluster_events(one, 0.0, 0.1, 8.0, 0.5, 4.0, 2)
    assert lab.tolist() == [-1] and ncl == 0
    lab, ncl, _ = m.mdsm_cluster_events(one, 0.0, 0.1, 8.0, 0.5, 4.0, 1)           # min_pts = 1: every point is a core point
    assert lab.tolist() == [0] and ncl == 1
    dup = np.array([(0, 5, 10, 7.0)] * 6, dtype=m.EVENT_DTYPE)                     # identical points
    lab, ncl, _ = m.mdsm_cluster_events(dup, 0.0, 0.1, 8.0, 0.5, 4.0, 5)
    assert lab.tolist() == [0] * 6
    with pytest.raises(m.MdsmError):
        m.mdsm_cluster_events(one, 0.0, 0.1, 0.0, 0.5, 4.0, 5)                     # eps_t = 0
    with pytest.raises(m.MdsmError):
        m.mdsm_classify_clusters(one, np.array([3], dtype=np.int32), 1, 0.0, 0.1, TSAMP, BW, NU, 3, 0.1)   # label out of range
    with pytest.raises(m.MdsmError):
        m.mdsm_classify_clusters(one, np.array([0], dtype=np.int32), 1, 0.0, 0.1, TSAMP, BW, NU, 4, 0.1)   # even k_smooth


@pytest.mark.parametrize("k_smooth", [1, 5])
def test_classifier_matches_the_oracle_cluster_by_cluster(k_smooth):
    ev = _events(3, nbeams=2, nblob=8, per=120, nnoise=200)
    # a broadband-RFI-like cluster at DM < 1 and a flat one (SNR independent of DM)
    extra = [(0, d, 30000 + k, np.float32(12.0)) for d in range(0, 8) for k in range(4)]
    extra += [(1, d, 45000, np.float32(9.0)) for d in range(200, 260)]
    ev = np.concatenate([ev, np.array(extra, dtype=m.EVENT_DTYPE)])
    lab, ncl, _ = m.mdsm_cluster_events(ev, DM_LOW, DM_STEP, 8.0, 0.5, 4.0, 5)
    res = m.mdsm_classify_clusters(ev, lab, ncl, DM_LOW, DM_STEP, TSAMP, BW, NU, k_smooth, 0.25)
    classes = set()
    for c in range(ncl):
        sel = lab == c
        r = oracle.classify_cluster(ev["t"][sel], ev["dm_idx"][sel], ev["snr"][sel], DM_LOW, DM_STEP, TSAMP, BW, NU, k_smooth, 0.25)
        assert int(res[c, 0]) == r["cls"] and int(res[c, 1]) == r["dm_idx"] and res[c, 2] == r["snr"]
        assert res[c, 3] == pytest.approx(r["width_ms"], rel=1e-14) and res[c, 4] == pytest.approx(r["rmse"], rel=1e-12, abs=1e-15)
        classes.add(r["cls"])
    assert classes >= {1, 2}                                   # both rejection paths are exercised


# ------------------------------------------------------------------ checks that do not pass through the oracle
def _pins():
    import os
    import runpy
    return runpy.run_path(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "fdbscan_pins.py"))


def _pin_events(S, shift_t=100, shift_d=16):
    """The integer (time, DM) points of a hand-worked set as events: t = time + 100, dm_idx = DM + 16 at dm_step 1."""
    return np.array([(0, d + shift_d, t + shift_t, 10.0) for t, d in S["pts"]], dtype=m.EVENT_DTYPE)


@pytest.mark.parametrize("name", ["split", "lost", "other"])
def test_library_clustering_on_the_hand_worked_sets(name):
    """mdsm_cluster_events against the labels and query counts written out by hand in tests/golden/fdbscan_pins.py (reading
    K-ii of PAPER.md:126) -- the expectation is the paper's sentence worked on paper, not another implementation."""
    S = _pins()["SETS"][name]
    ev = _pin_events(S)
    lab, ncl, nq = m.mdsm_cluster_events(ev, 0.0, 1.0, float(S["eps"]), float(S["eps"]), 1.0, S["min_pts"])
    assert lab.tolist() == S["fdbscan_labels"] and ncl == max(S["fdbscan_labels"]) + 1 and nq == S["fdbscan_queries"], S["fails_for"]
    lab, ncl, nq = m.mdsm_cluster_events(ev, 0.0, 1.0, float(S["eps"]), float(S["eps"]), 1.0, S["min_pts"], exact=True)
    assert lab.tolist() == S["dbscan_labels"] and nq == len(ev)            # exact: every point is queried exactly once


@pytest.mark.parametrize("dim", [0, 1, 2])
@pytest.mark.parametrize("sign", [1, -1])
def test_library_follows_a_chain_along_every_dimension_and_direction(dim, sign):
    C = _pins()["CHAIN"]
    pos = 50 + sign * C["step"] * np.arange(C["n"])
    col = {0: ("t", pos), 1: ("dm_idx", pos), 2: ("snr", pos.astype(np.float32))}[dim]
    ev = np.zeros(C["n"], dtype=m.EVENT_DTYPE)
    ev["t"], ev["dm_idx"], ev["snr"] = 7, 7, 7.0
    ev[col[0]] = col[1]
    lab, ncl, nq = m.mdsm_cluster_events(ev, 0.0, 1.0, float(C["eps"]), float(C["eps"]), float(C["eps"]), C["min_pts"])
    assert ncl == 1 and lab.tolist() == [0] * C["n"] and nq == C["fdbscan_queries"], C["fails_for"]


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_library_clustering_against_scikit_learn(seed):
    """exact = 1 is DBSCAN: same noise set, same number of clusters, same partition of the core points as scikit-learn's
    (border points may go to either adjacent cluster).  exact = 0 (FDBSCAN) only follows density-reachability: each of its
    clusters lies inside ONE scikit-learn cluster, DBSCAN's noise stays noise, and what FDBSCAN loses on top is rare."""
    sk = pytest.importorskip("sklearn.cluster")
    ev = _events(seed)
    eps = np.array([8.0, 0.5, 4.0])
    ref = sk.DBSCAN(eps=1.0, min_samples=5, metric="chebyshev").fit(_points(ev) / eps)
    core = np.zeros(len(ev), dtype=bool)
    core[ref.core_sample_indices_] = True
    lab, ncl, nq = m.mdsm_cluster_events(ev, DM_LOW, DM_STEP, *eps, 5, exact=True)
    assert np.array_equal(lab == -1, ref.labels_ == -1) and ncl == ref.labels_.max() + 1 and nq == len(ev)
    pairs = set(zip(lab[core].tolist(), ref.labels_[core].tolist()))
    assert len(pairs) == ncl
    labf, nclf, nqf = m.mdsm_cluster_events(ev, DM_LOW, DM_STEP, *eps, 5, exact=False)
    assert nqf < len(ev) and nclf >= ncl
    for c in range(nclf):
        # an FDBSCAN cluster may hold border points scikit-learn gave to a neighbouring cluster: look at its core points
        inside = set(ref.labels_[(labf == c) & core].tolist())
        assert len(inside) == 1 and -1 not in inside
    assert np.all(labf[ref.labels_ == -1] == -1)
    assert np.mean(labf[ref.labels_ >= 0] >= 0) > 0.95


def _curve(ddm, w_ms):
    import math
    z = abs(6.91e-3 * ddm * BW / (w_ms * NU ** 3))                        # Eq. 4
    return 1.0 if z == 0 else 0.5 * math.sqrt(math.pi) * math.erf(z) / z   # Eq. 3


def test_library_classifier_on_a_cluster_drawn_from_the_model_curve_and_on_its_rejections():
    """mdsm_classify_clusters against closed forms: detections whose SNR follows Eq. 3 exactly around DM index 300 (pulse of
    8 samples) are a candidate with RMSE ~ 0; the same cluster at DM index 5 (0.5 pc/cm^3 < 1) is broadband RFI; a cluster whose
    SNR does not fall off with DM is rejected by the curve.  One call classifies all three."""
    width, snr0 = 8, 20.0
    w_ms = width * TSAMP * 1e3
    ev, lab = [], []
    for cid, d0 in ((0, 300), (1, 5)):
        for di in range(max(0, d0 - 200), d0 + 201):
            resp = _curve((di - d0) * DM_STEP, w_ms)
            if resp < 0.3:
                continue
            for k in range(width if di == d0 else 1):
                ev.append((0, di, 1000 + k, np.float32(snr0 * resp * (1.0 if k == 0 else 0.9))))
                lab.append(cid)
    for di in range(100, 400):                                                # flat: SNR 9 at every DM, three hits at DM index 250
        for k in range(3 if di == 250 else 1):
            ev.append((0, di, 5000 + k, np.float32(9.0)))
            lab.append(2)
    ev = np.array(ev, dtype=m.EVENT_DTYPE)
    lab = np.array(lab, dtype=np.int32)
    perm = np.random.default_rng(5).permutation(len(ev))                      # event order must not matter
    res = m.mdsm_classify_clusters(ev[perm], lab[perm], 4, DM_LOW, DM_STEP, TSAMP, BW, NU, 1, 0.05)
    assert res[0].tolist()[:2] == [0.0, 300.0] and abs(res[0, 2] - snr0) < 1e-6 and abs(res[0, 3] - w_ms) < 1e-12 and res[0, 4] < 1e-6
    assert res[1].tolist()[:2] == [1.0, 5.0] and res[1, 4] == 0.0
    assert res[2].tolist()[:2] == [2.0, 250.0] and res[2, 2] == 9.0 and abs(res[2, 3] - 3 * TSAMP * 1e3) < 1e-12 and res[2, 4] > 0.5
    assert res[3].tolist() == [-1.0, 0.0, 0.0, 0.0, 0.0]                      # a cluster id without events


def test_library_classifier_hand_worked_three_dm_cluster_with_smoothing():
    """DMs 20.0, 20.1, 20.2; detections: d=200: snr 6; d=201: snr 10, 9, 8 at t = 50, 51, 53; d=202: snr 4; 1 ms samples;
    3-element moving average.  Every number below is worked from PAPER.md:144-156 and Eqs. 3/4 in the test itself."""
    import math
    ev = np.array([(0, 200, 50, 6), (0, 201, 50, 10), (0, 201, 51, 9), (0, 201, 53, 8), (0, 202, 52, 4)], dtype=m.EVENT_DTYPE)
    res = m.mdsm_classify_clusters(ev[::-1].copy(), np.zeros(5, dtype=np.int32), 1, 0.0, 0.1, 1e-3, BW, NU, 3, 10.0)[0]
    assert res[0] == 0.0 and res[1] == 201.0 and res[2] == 10.0 and abs(res[3] - 4.0) < 1e-12          # (53 - 50 + 1) * 1 ms
    sm = np.array([(6 + 10) / 2, (6 + 10 + 4) / 3, (10 + 4) / 2])
    sig = sm / sm.max()
    mm = _curve(0.1, 4.0)
    rmse = math.sqrt(((mm - sig[0]) ** 2 + (1 - sig[1]) ** 2 + (mm - sig[2]) ** 2) / 3)
    assert abs(res[4] - rmse) < 1e-12
    strict = m.mdsm_classify_clusters(ev, np.zeros(5, dtype=np.int32), 1, 0.0, 0.1, 1e-3, BW, NU, 3, rmse - 1e-9)[0]
    assert strict[0] == 2.0                                                   # "exceeds a preset threshold" (step 8)
