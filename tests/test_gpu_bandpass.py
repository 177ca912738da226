"""The paper's bandpass-fit RFI stage (mdsm_bandpass_clip) on the GPU against the oracle."""
import numpy as np
import pytest

import oracle
from workloads import power_filterbank

from gpu_util import Plan

pytestmark = pytest.mark.gpu


def _run(nb, nc, ns, window, order, k_mask, k_chan, k_spec, subtract, seed, beam0=0, nbeams_run=None):
    import torch
    x = power_filterbank(nb, nc, ns, seed, window)
    xo = x.copy()
    ref = oracle.bandpass_clip(xo, window, order, k_mask, k_chan, k_spec, subtract)
    args = (nb, nc, 418.0, -20.0 / nc, 51.2e-6, ns, 0.0, 0.1, 4)
    with Plan(args) as p:
        d = torch.from_numpy(x).cuda()
        cm = torch.full((nb, nc, ns // window), 9, dtype=torch.uint8, device="cuda")
        sm = torch.full((nb, ns), 9, dtype=torch.uint8, device="cuda")
        fit = torch.zeros((nb, nc, 2), dtype=torch.float64, device="cuda")
        st = torch.zeros((nb, 4), dtype=torch.float64, device="cuda")
        n_run = nb - beam0 if nbeams_run is None else nbeams_run
        p.m.mdsm_bandpass_clip(p.h, d, beam0, n_run, window, order, k_mask, k_chan, k_spec, subtract, cm, sm, fit, st)
        torch.cuda.synchronize()
        return x, xo, ref, d.cpu().numpy(), cm.cpu().numpy(), sm.cpu().numpy(), fit.cpu().numpy(), st.cpu().numpy()


def _check(x, xo, ref, got, cm, sm, fit, st, window, k_chan, k_spec, beams, subtract, need_flags=True):
    """Guard-band comparison (the form tests/test_gpu_parity_small.py uses for mdsm_rfi_clip).  The GPU reduces the same
    fp64 sums in another order and fits with its own elimination order, so a decision may differ from the oracle's only when
    the unit's statistic is within the band of its threshold:
      chunk of channel c:  |mean - (fit[c] + k_chan rmse)| <= 1e-6 max(1, |k_chan|) rmse + 1e-9 |fit[c]|
      spectrum t:          |mean_c y - (mean_bp + k_spec std_bp)| <= 1e-6 max(1, |k_spec|) std_bp + 2^-22 max|fit|
    (y = the data after the channel stage; the last term is one fp32 ulp of a replacement value).  Outside the bands flags
    must be equal, and every sample whose chunk (with its dilation neighbours) and whose spectrum are outside them must
    equal the oracle's to one fp32 ulp of the fit."""
    nb, nc, ns = x.shape
    nchunk = ns // window
    if need_flags:
        assert ref["chan_mask"].sum() > 0 and ref["spec_mask"].sum() > 0      # the case exercises both stages
    for b in beams:
        assert int(st[b, 3]) == int(ref["nmasked"][b])
        assert np.allclose(fit[b, :, 0], ref["fit"][b], rtol=1e-9, atol=1e-12)
        assert np.array_equal(fit[b, :, 1], ref["bpi"][b]) or np.allclose(fit[b, :, 1], ref["bpi"][b], rtol=1e-13)
        assert np.allclose(st[b, :3], [ref["rmse"][b], ref["mean_bp"][b], ref["std_bp"][b]], rtol=1e-8, atol=1e-12)
        f, rmse = ref["fit"][b], ref["rmse"][b]
        # channel stage
        cmean = x[b].astype(np.float64).reshape(nc, nchunk, window).mean(axis=2)
        thr_c = (f + k_chan * rmse)[:, None]
        band_c = (1e-6 * max(1.0, abs(k_chan)) * rmse + 1e-9 * np.abs(f))[:, None]
        near = np.abs(cmean - thr_c) <= band_c                               # raw decision in doubt
        near_d = near.copy()                                                  # ... and with it its two time neighbours' flags
        near_d[:, 1:] |= near[:, :-1]
        near_d[:, :-1] |= near[:, 1:]
        assert np.array_equal(cm[b][~near_d], ref["chan_mask"][b][~near_d])
        t_doubt = np.repeat(near_d.any(axis=0), window)                       # samples whose spectrum saw a chunk in doubt
        # spectrum stage, on the oracle's channel-stage result rebuilt here from its flags
        y = x[b].astype(np.float64)
        flagged = np.repeat(ref["chan_mask"][b].astype(bool), window, axis=1)
        y = np.where(flagged, f.astype(np.float32).astype(np.float64)[:, None], y)
        m_t = y.mean(axis=0)
        thr_s = ref["mean_bp"][b] + k_spec * ref["std_bp"][b]
        band_s = 1e-6 * max(1.0, abs(k_spec)) * ref["std_bp"][b] + 2.0 ** -22 * np.abs(f).max()
        near_s = np.abs(m_t - thr_s) <= band_s
        sure_t = ~(near_s | t_doubt)
        assert np.array_equal(sm[b][sure_t], ref["spec_mask"][b][sure_t])
        if need_flags:
            assert (~sure_t).mean() < 0.01 and near_d.mean() < 0.01           # the bands stay the exception
        # data
        sure = np.repeat(~near_d, window, axis=1) & sure_t[None, :]
        assert np.allclose(got[b][sure], xo[b][sure], rtol=0, atol=np.abs(f).max() * 2.0 ** -22)


@pytest.mark.parametrize("subtract", [False, True])
@pytest.mark.parametrize("shape", [(2, 256, 8192, 64, 4), (1, 1024, 16384, 64, 6), (2, 100, 4000, 50, 3)])
def test_bandpass_stage_matches_the_oracle(shape, subtract):
    nb, nc, ns, window, order = shape
    k_mask, k_chan, k_spec = 5.0, 150.0 if nc >= 256 else 60.0, 1.5
    r = _run(nb, nc, ns, window, order, k_mask, k_chan, k_spec, subtract, seed=11)
    _check(*r, window, k_chan, k_spec, range(nb), subtract)


def test_bandpass_stage_beam_subrange_leaves_other_beams_alone():
    nb, nc, ns, window = 3, 128, 4096, 64
    x, xo, ref, got, cm, sm, fit, st = _run(nb, nc, ns, window, 3, 5.0, 100.0, 1.5, True, seed=12, beam0=1, nbeams_run=1)
    assert np.array_equal(got[0], x[0]) and np.array_equal(got[2], x[2])
    assert np.all(cm[0] == 9) and np.all(cm[2] == 9) and np.all(sm[0] == 9)
    _check(x, xo, ref, got, cm, sm, fit, st, window, 100.0, 1.5, [1], True)


def test_bandpass_stage_argument_errors():
    import torch
    args = (1, 16, 418.0, -1.0, 51.2e-6, 1024, 0.0, 0.1, 2)
    with Plan(args) as p:
        d = torch.zeros((1, 16, 1024), dtype=torch.float32, device="cuda")
        with pytest.raises(p.m.MdsmError):
            p.m.mdsm_bandpass_clip(p.h, d, 0, 1, 48, 2, 5.0, 5.0, 5.0, False)       # window does not divide nsamps
        with pytest.raises(p.m.MdsmError):
            p.m.mdsm_bandpass_clip(p.h, d, 0, 1, 64, 16, 5.0, 5.0, 5.0, False)      # order >= nchans
        with pytest.raises(p.m.MdsmError):
            p.m.mdsm_bandpass_clip(p.h, d, 0, 2, 64, 2, 5.0, 5.0, 5.0, False)       # beam range


@pytest.mark.parametrize("shape", [(1, 2, 256, 256, 0), (1, 3, 1001, 7, 1), (2, 5, 96, 1, 2), (1, 64, 2048, 2048, 5)])
def test_bandpass_stage_degenerate_shapes(shape):
    """Few channels (order < nchans), one chunk per channel, window 1, rows that are not 16-byte aligned."""
    import torch
    nb, nc, ns, window, order = shape
    g = np.random.default_rng(nc * 1000 + ns)
    x = (g.exponential(size=(nb, nc, ns)) * (5.0 + np.arange(nc))[None, :, None]).astype(np.float32)
    x[:, :, ns // 3] += 40.0
    xo = x.copy()
    ref = oracle.bandpass_clip(xo, window, order, 5.0, 30.0, 1.0, True)
    args = (nb, nc, 418.0, -20.0 / nc, 51.2e-6, ns, 0.0, 0.01, 2)
    with Plan(args) as p:
        d = torch.from_numpy(x).cuda()
        cm = torch.zeros((nb, nc, ns // window), dtype=torch.uint8, device="cuda")
        sm = torch.zeros((nb, ns), dtype=torch.uint8, device="cuda")
        fit = torch.zeros((nb, nc, 2), dtype=torch.float64, device="cuda")
        st = torch.zeros((nb, 4), dtype=torch.float64, device="cuda")
        p.m.mdsm_bandpass_clip(p.h, d, 0, nb, window, order, 5.0, 30.0, 1.0, True, cm, sm, fit, st)
        torch.cuda.synchronize()
        _check(x, xo, ref, d.cpu().numpy(), cm.cpu().numpy(), sm.cpu().numpy(), fit.cpu().numpy(), st.cpu().numpy(), window, 30.0, 1.0,
               range(nb), True, need_flags=False)
        assert ref["spec_mask"].sum() > 0
