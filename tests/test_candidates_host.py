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
