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


def _check(x, xo, ref, got, cm, sm, fit, st, window, k_chan, k_spec, beams):
    nc = x.shape[1]
    assert ref["chan_mask"].sum() > 0 and ref["spec_mask"].sum() > 0          # the case exercises both stages
    for b in beams:
        assert int(st[b, 3]) == int(ref["nmasked"][b])
        assert np.allclose(fit[b, :, 0], ref["fit"][b], rtol=1e-9, atol=1e-12)
        assert np.array_equal(fit[b, :, 1], ref["bpi"][b]) or np.allclose(fit[b, :, 1], ref["bpi"][b], rtol=1e-13)
        assert np.allclose(st[b, :3], [ref["rmse"][b], ref["mean_bp"][b], ref["std_bp"][b]], rtol=1e-8)
        # channel flags: identical outside a guard band around the threshold (the sums are fp64 in another order)
        cmean = x[b].astype(np.float64).reshape(nc, -1, window).mean(axis=2)
        z = (cmean - ref["fit"][b][:, None]) / ref["rmse"][b]
        raw_sure = np.abs(z - k_chan) > 1e-6 * max(1.0, abs(k_chan))
        sure = raw_sure.copy()
        sure[:, 1:] &= raw_sure[:, :-1]
        sure[:, :-1] &= raw_sure[:, 1:]
        assert np.array_equal(cm[b][sure], ref["chan_mask"][b][sure])
        if np.array_equal(cm[b], ref["chan_mask"][b]):
            # spectrum flags on the modified data
            same = sm[b] == ref["spec_mask"][b]
            assert same.mean() > 0.9999
            if same.all():
                scale = np.abs(ref["fit"][b]).max()
                assert np.allclose(got[b], xo[b], rtol=0, atol=scale * 2.0 ** -22)


@pytest.mark.parametrize("subtract", [False, True])
@pytest.mark.parametrize("shape", [(2, 256, 8192, 64, 4), (1, 1024, 16384, 64, 6), (2, 100, 4000, 50, 3)])
def test_bandpass_stage_matches_the_oracle(shape, subtract):
    nb, nc, ns, window, order = shape
    k_mask, k_chan, k_spec = 5.0, 150.0 if nc >= 256 else 60.0, 1.5
    r = _run(nb, nc, ns, window, order, k_mask, k_chan, k_spec, subtract, seed=11)
    _check(*r, window, k_chan, k_spec, range(nb))


def test_bandpass_stage_beam_subrange_leaves_other_beams_alone():
    nb, nc, ns, window = 3, 128, 4096, 64
    x, xo, ref, got, cm, sm, fit, st = _run(nb, nc, ns, window, 3, 5.0, 100.0, 1.5, True, seed=12, beam0=1, nbeams_run=1)
    assert np.array_equal(got[0], x[0]) and np.array_equal(got[2], x[2])
    assert np.all(cm[0] == 9) and np.all(cm[2] == 9) and np.all(sm[0] == 9)
    _check(x, xo, ref, got, cm, sm, fit, st, window, 100.0, 1.5, [1])


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
        f = fit.cpu().numpy()
        assert np.allclose(f[:, :, 0], ref["fit"], rtol=1e-8, atol=1e-10)
        assert np.array_equal(st.cpu().numpy()[:, 3].astype(int), ref["nmasked"])
        same_c = np.array_equal(cm.cpu().numpy(), ref["chan_mask"])
        same_s = np.array_equal(sm.cpu().numpy(), ref["spec_mask"])
        assert (cm.cpu().numpy() != ref["chan_mask"]).mean() < 1e-3 and (sm.cpu().numpy() != ref["spec_mask"]).mean() < 1e-3
        if same_c and same_s:
            assert np.allclose(d.cpu().numpy(), xo, rtol=0, atol=np.abs(ref["fit"]).max() * 2.0 ** -22)
