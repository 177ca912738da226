"""GPU-vs-oracle parity of the post-processing calls through the C ABI."""
import numpy as np
import pytest

import oracle
from workloads import CONFIGS, generate

from gpu_util import Plan, compare_events_f32

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    return torch


def _series(nb, nd, ns, seed):
    g = np.random.default_rng(seed)
    t = np.arange(ns)
    s = (g.normal(size=(nb, nd, ns)) * 6 + 50 + 3e-3 * t[None, None, :] * g.uniform(-1, 1, size=(nb, nd, 1))).astype(np.float32)
    s[:, :, ::97] += 80                    # isolated outliers for the median to remove
    s[0, 1, 300:320] += 40                 # a wide pulse that must survive
    s[1, 0, :] = 3.25                      # constant series: zero variance
    return s


@pytest.mark.parametrize("window", [1, 3, 5, 9, 33])
def test_median_filter_bit_exact(window):
    torch = _torch()
    import paper_1307_5700_b200 as m
    nb, nd, ns = 2, 3, 5003
    args = (nb, 8, 418.0, -2.5, 51.2e-6, ns, 0.0, 0.15, nd)
    with Plan(args) as p:
        n = p.nsamps_out
        s = _series(nb, nd, ns, window)
        ref = oracle.median_filter(s, n, window)
        ds = torch.from_numpy(s).cuda()
        df = torch.full_like(ds, -7.0)
        m.mdsm_median_filter(p.h, ds, df, 0, nb, window)
        torch.cuda.synchronize()
        got = df.cpu().numpy()
        assert np.array_equal(got[:, :, :n], ref[:, :, :n])
        assert np.all(got[:, :, n:] == -7.0)
        # beam sub-range and argument errors
        df2 = torch.full_like(ds, -7.0)
        m.mdsm_median_filter(p.h, ds, df2, 1, 1, window)
        torch.cuda.synchronize()
        assert np.all(df2[0].cpu().numpy() == -7.0) and np.array_equal(df2[1, :, :n].cpu().numpy(), ref[1, :, :n])
        for bad in (0, 4, 35):
            with pytest.raises(m.MdsmError):
                m.mdsm_median_filter(p.h, ds, df2, 0, nb, bad)
        with pytest.raises(m.MdsmError):
            m.mdsm_median_filter(p.h, ds, ds, 0, nb, 3)


def test_detrend_parity():
    torch = _torch()
    import paper_1307_5700_b200 as m
    nb, nd, ns = 2, 3, 20011
    args = (nb, 8, 418.0, -2.5, 51.2e-6, ns, 0.0, 0.15, nd)
    with Plan(args) as p:
        n = p.nsamps_out
        s = _series(nb, nd, ns, 4)
        ref, par = oracle.detrend(s, n)
        ds = torch.from_numpy(s).cuda()
        dp = torch.zeros((nb, nd, 3), dtype=torch.float64, device="cuda")
        m.mdsm_detrend(p.h, ds, 0, nb, dp)
        torch.cuda.synchronize()
        got = ds.cpu().numpy()
        gp = dp.cpu().numpy()
        # fp64 sums in tree order instead of sequential order: parameters agree to ~1e-12, samples to float rounding
        assert np.allclose(gp[..., 0], par[..., 0], rtol=1e-10, atol=1e-10)
        assert np.allclose(gp[..., 1], par[..., 1], rtol=1e-8, atol=1e-13)
        assert np.allclose(gp[..., 2], par[..., 2], rtol=1e-10, atol=1e-12)
        assert np.allclose(got[:, :, :n], ref[:, :, :n], rtol=0, atol=2e-6)
        assert np.all(got[1, 0, :n] == 0.0)                       # zero-variance series -> zeros (reading E-ii)
        assert np.array_equal(got[:, :, n:], s[:, :, n:])         # the tail is not touched


def test_chain_with_postprocess_cfg1():
    """cfg 1: dedisperse -> median(5) -> detrend -> detect against the same chain of oracle calls."""
    torch = _torch()
    import paper_1307_5700_b200 as m
    cfg = CONFIGS[1]
    x = generate(cfg)
    d = oracle.delay_table(cfg.nchans, cfg.f_top, cfg.foff, cfg.tsamp, cfg.dm_low, cfg.dm_step, cfg.ndms)
    with Plan(cfg) as p:
        n = p.nsamps_out
        out = p.dedisperse(torch.from_numpy(x).cuda())
        filt = torch.zeros_like(out)
        m.mdsm_median_filter(p.h, out, filt, 0, 1, 5)
        m.mdsm_detrend(p.h, filt, 0, 1, None)
        ev_g, cnt_g = p.detect(filt, cfg.snr_thresh)
        # the oracle continues from the GPU's dedispersed series (its own parity is tested elsewhere)
        so = out.cpu().numpy()
        so[:, :, n:] = 0
        fo = oracle.median_filter(so, n, 5)
        no, _ = oracle.detrend(fo, n)
        ev_o, cnt_o, _ = oracle.detect(np.ascontiguousarray(no), n, cfg.snr_thresh)
        assert compare_events_f32(ev_g, ev_o, cfg.snr_thresh) > 0
        top = ev_g[np.argmax(ev_g["snr"])]
        assert top["dm_idx"] == 20 and 999 <= top["t"] <= 1004   # the 4-sample pulse survives a 5-point median


def test_pipeline_host_with_postprocess_options():
    """mdsm_pipeline_host with plan options post_median_window / post_detrend = the same events as the separate calls."""
    torch = _torch()
    import paper_1307_5700_b200 as m
    cfg = CONFIGS[1]
    x = generate(cfg)
    with Plan(cfg) as p:
        out = p.dedisperse(torch.from_numpy(x).cuda())
        filt = torch.zeros_like(out)
        m.mdsm_median_filter(p.h, out, filt, 0, 1, 5)
        m.mdsm_detrend(p.h, filt, 0, 1, None)
        ev_sep, cnt_sep = p.detect(filt, cfg.snr_thresh)
        m.mdsm_plan_set_option(p.h, "post_median_window", 5)
        m.mdsm_plan_set_option(p.h, "post_detrend", 1)
        hev = np.zeros(4096, dtype=m.EVENT_DTYPE)
        rc, cnt = m.mdsm_pipeline_host(p.h, x, 0, 0.0, 0.0, cfg.snr_thresh, hev, 4096, 1)       # window 0: no clip
        assert rc == m.MDSM_OK and cnt == cnt_sep > 0
        hev = hev[:cnt]
        hev = hev[np.lexsort((hev["t"], hev["dm_idx"], hev["beam"]))]
        assert np.array_equal(hev, ev_sep)
        with pytest.raises(m.MdsmError):
            m.mdsm_plan_set_option(p.h, "post_median_window", 4)
