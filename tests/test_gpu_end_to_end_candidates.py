"""The whole path on one small simulated observation: host buffer -> mdsm_pipeline_host (clip, dedisperse, detect on the
GPU) -> host candidate stage (FDBSCAN + DM-SNR classifier).  A dispersed pulse must come out as ONE candidate at its DM;
a broadband (DM 0) burst must be removed by the clip, or, with the clip off, be rejected by the classifier's DM < 1 rule
(PAPER.md:116-156).  The GPU event list is also compared with the oracle chain."""
import numpy as np
import pytest

import oracle

from gpu_util import Plan, compare_events_f32

pytestmark = pytest.mark.gpu

NC, NS, ND = 256, 16384, 200
F_TOP, FOFF, TSAMP = 418.0, -20.0 / 256, 51.2e-6
DM_TRUE, T0, WIDTH = 100, 6000, 4


def _observation():
    g = np.random.default_rng(3)
    x = g.normal(size=(1, NC, NS)).astype(np.float32)
    delays = oracle.delay_table(NC, F_TOP, FOFF, TSAMP, 0.0, 0.1, ND)
    for c in range(NC):
        x[0, c, T0 + delays[DM_TRUE, c]: T0 + delays[DM_TRUE, c] + WIDTH] += 1.5      # a pulse at DM 10.0
    x[0, :, 12000:12002] += 3.0                                                       # a broadband burst (DM 0)
    return x, delays


@pytest.mark.parametrize("clip", [True, False])
def test_pulse_becomes_one_candidate_and_the_broadband_burst_does_not(clip):
    x, delays = _observation()
    window = 64 if clip else 0
    xo = x.copy()
    if clip:
        oracle.rfi_clip(xo, 64, 5.0, 5.0)
    ref, _ = oracle.dedisperse(xo, delays, want_abs=False)
    ev_o, cnt_o, _ = oracle.detect(ref, ref.shape[2], 5.0)
    args = (1, NC, F_TOP, FOFF, TSAMP, NS, 0.0, 0.1, ND)
    with Plan(args) as p:
        m = p.m
        ev = np.zeros(1 << 16, dtype=m.EVENT_DTYPE)
        rc, cnt = m.mdsm_pipeline_host(p.h, x, window, 5.0, 5.0, 5.0, ev, len(ev), 1)
        assert rc == m.MDSM_OK and abs(cnt - cnt_o) <= 2
        ev = ev[:cnt]
        ev = ev[np.lexsort((ev["t"], ev["dm_idx"], ev["beam"]))]
        compare_events_f32(ev, ev_o, 5.0)
        lab, ncl, nq = m.mdsm_cluster_events(ev, 0.0, 0.1, 12.0, 0.35, 1e9, 5)
        res = m.mdsm_classify_clusters(ev, lab, ncl, 0.0, 0.1, TSAMP, 20.0, 0.408, 5, 0.3)
    cands = [c for c in range(ncl) if int(res[c, 0]) == 0]
    assert len(cands) == 1
    c = cands[0]
    sel = lab == c
    assert abs(int(res[c, 1]) - DM_TRUE) <= 4 and res[c, 2] > 7.0                      # peak at the pulse's DM
    assert T0 - 30 <= ev["t"][sel].min() and ev["t"][sel].max() <= T0 + 30 + WIDTH
    assert 0.5 * WIDTH * TSAMP * 1e3 <= res[c, 3] <= 4 * WIDTH * TSAMP * 1e3           # width of the order of the pulse's
    burst = (ev["t"] >= 11990) & (ev["t"] <= 12012)
    if clip:
        assert not burst.any()                                                         # the spectrum clip removed it
    else:
        assert burst.sum() > 20
        rejected = {int(res[l, 0]) for l in set(lab[burst].tolist()) if l >= 0}
        assert rejected == {1}                                                         # clustered, then discarded: DM < 1
