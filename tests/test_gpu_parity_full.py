"""GPU-vs-oracle parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(all beams in one call per stage, default kernel selection, the same plan options).

cfg 2, 3, 4: every output element of every beam is compared with the oracle (beam by beam, so the
fp64 reference of one beam is all that is resident); clip masks, the clipped input and the event
lists are compared too (bit-exact for u8, guard-banded for f32: readings B-ix, D-vi of DESIGN.md).
cfg 5 (34 GB in, 17 GB out): every one of the 2048 series of beam 0 is compared element by element, plus a seeded
sample of (beam, DM) series of two other beams (`oracle.dedisperse_rows` computes series one by one), plus the clip of
one whole beam; detection is checked on the compared series.  Two more plans put the element offsets of the
checked beam beyond 2^32 (4096 channels, fp32 and uint8).
"""
import numpy as np
import pytest

import oracle
from workloads import CONFIGS, generate, generate_beam

from gpu_util import Plan, compare_events_f32

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    return torch


def _f32_check(got, ref, ab, what):
    err = np.abs(got.astype(np.float64) - ref)
    tol = 1e-5 * ab + 1e-6                                   # north_star tolerance
    bad = err > tol
    assert not bad.any(), f"{what}: {int(bad.sum())} of {bad.size} outside tolerance (worst err/tol {np.max(err / tol):.3g})"
    return float(np.max(err / tol))


def _clip_f32_check(x_pre, x_gpu, cm, sm, r, W, k, what):
    """Reading B-ix: masks may differ from the oracle only for units whose z-score is within 1e-4 of k."""
    nc, ns = x_pre.shape
    csum = x_pre.astype(np.float64).reshape(nc, ns // W, W).sum(axis=2)
    z = (csum - W * r["chan_mean"][0][:, None]) / (np.maximum(r["chan_sig"][0], 1e-300)[:, None] * np.sqrt(W))
    near = np.abs(z - k) <= 1e-4
    nd = near.copy()
    nd[:, 1:] |= near[:, :-1]
    nd[:, :-1] |= near[:, 1:]
    assert np.array_equal(cm[~nd], r["chan_mask"][0][~nd]), what
    if near.any():
        return False                                          # downstream data may legitimately differ
    zs = (r["spec_sum"][0] - r["spec_thr"][0, 1]) / max(r["spec_thr"][0, 2], 1e-300)
    near_s = np.abs(zs - k) <= 1e-4
    assert np.array_equal(sm[~near_s], r["spec_mask"][0][~near_s]), what
    return not near_s.any()


def _chain_full(k):
    torch = _torch()
    cfg = CONFIGS[k]
    x = generate(cfg)
    is_u8 = cfg.dtype == "u8"
    delays = oracle.delay_table(cfg.nchans, cfg.f_top, cfg.foff, cfg.tsamp, cfg.dm_low, cfg.dm_step, cfg.ndms)
    with Plan(cfg) as p:
        nso = p.nsamps_out
        assert np.array_equal(p.delays(), delays)
        dx = torch.from_numpy(x).cuda()
        cm, sm = p.clip(dx, cfg.window, cfg.k_chan, cfg.k_spec)
        out = p.dedisperse(dx)                                # all beams, one launch: the bench configuration
        ev_g, cnt_g = p.detect(out, cfg.snr_thresh, max_events=1 << 22)
        x_gpu = dx.cpu().numpy()
        del dx
        n_ev_o = 0
        worst = 0.0
        for b in range(cfg.nbeams):
            xo = x[b:b + 1].copy()
            r = oracle.rfi_clip(xo, cfg.window, cfg.k_chan, cfg.k_spec, debug=not is_u8)
            if is_u8:
                assert np.array_equal(cm[b], r["chan_mask"][0]) and np.array_equal(sm[b], r["spec_mask"][0]), f"beam {b} masks"
                assert np.array_equal(x_gpu[b], xo[0]), f"beam {b} clipped input"
            else:
                same = _clip_f32_check(x[b], x_gpu[b], cm[b], sm[b], r, cfg.window, cfg.k_chan, f"beam {b} masks")
                if same:
                    assert np.array_equal(x_gpu[b], xo[0]), f"beam {b} clipped input"
                else:                                         # a unit sat in the guard band: continue from the GPU's data
                    xo = x_gpu[b:b + 1].copy()
            ref, ab = oracle.dedisperse(xo, delays)
            got = out[b, :, :nso].cpu().numpy()
            if is_u8:
                assert np.array_equal(got.view(np.uint32), ref[0]), f"beam {b} dedispersed output"
            else:
                worst = max(worst, _f32_check(got, ref[0], ab[0], f"beam {b}"))
            ev_o, cnt_o, _ = oracle.detect(ref, nso, cfg.snr_thresh)
            ev_o["beam"] = b
            ev_b = ev_g[ev_g["beam"] == b]
            if is_u8:
                assert np.array_equal(ev_b, ev_o), f"beam {b} events"
            else:
                compare_events_f32(ev_b, ev_o, cfg.snr_thresh)
            n_ev_o += cnt_o
            del ref, ab, got
        assert n_ev_o > 0 and abs(cnt_g - n_ev_o) <= (0 if is_u8 else 8)
        tail = out[:, :, nso:]
        assert bool((tail == -7).all()), "samples t >= nsamps_out must not be written"
    return worst


def test_cfg2_full_chain_every_element():
    _chain_full(2)


def test_cfg3_full_chain_every_element():
    _chain_full(3)


def test_cfg4_full_chain_bit_exact():
    _chain_full(4)


def test_cfg5_sampled_series():
    torch = _torch()
    cfg = CONFIGS[5]
    delays = oracle.delay_table(cfg.nchans, cfg.f_top, cfg.foff, cfg.tsamp, cfg.dm_low, cfg.dm_step, cfg.ndms)
    g = np.random.default_rng(55)
    check_beams = [0, 9, cfg.nbeams - 1]
    host = {}
    with Plan(cfg) as p:
        nso = p.nsamps_out
        assert p.max_delay == 9778 and nso == 121294
        assert np.array_equal(p.delays(), delays)
        dx = torch.empty((cfg.nbeams, cfg.nchans, cfg.nsamps), dtype=torch.float32, device="cuda")
        for b in range(cfg.nbeams):
            xb = generate_beam(cfg, b)
            dx[b].copy_(torch.from_numpy(xb))
            if b in check_beams:
                host[b] = xb
        torch.cuda.synchronize()
        cm, sm = p.clip(dx, cfg.window, cfg.k_chan, cfg.k_spec)
        out = p.dedisperse(dx)
        ev_g, cnt_g = p.detect(out, cfg.snr_thresh, max_events=1 << 22)
        assert cnt_g == len(ev_g)
        # 26 GB of pre-summed rows per beam: the reservation holds fewer beams than the plan, so the beams are walked through
        # the slots in stream order and every checked beam but the first re-uses a slot
        slots = p.info(p.m.MDSM_F32)["scratch_slots"]
        assert 1 <= slots < cfg.nbeams and (cfg.nbeams - 1) >= slots, slots
        # the injected pulses (20 per beam, amplitude >= 0.5 per channel over 4096 channels) must be found
        assert all((ev_g["beam"] == b).sum() > 0 for b in range(cfg.nbeams))
        for b in check_beams:
            xo = host[b][None].copy()
            if b == check_beams[0]:                           # the clip of one whole beam against the oracle
                r = oracle.rfi_clip(xo, cfg.window, cfg.k_chan, cfg.k_spec, debug=True)
                same = _clip_f32_check(host[b], None, cm[b], sm[b], r, cfg.window, cfg.k_chan, f"beam {b} masks")
                xg = dx[b].cpu().numpy()
                if same:
                    assert np.array_equal(xg, xo[0])
                xo = xg[None]
            else:
                xo = dx[b].cpu().numpy()[None]                # clipped data as the GPU left it
            if b == check_beams[-1]:                          # one whole beam: all 2048 series, element by element -- the LAST
                ds = np.arange(cfg.ndms)                      # beam, which goes through a scratch slot other beams used before it
            else:
                ds = np.unique(np.concatenate([[0, 1, cfg.ndms - 1, cfg.ndms - 2], g.integers(0, cfg.ndms, size=8)]))
            ref, ab = oracle.dedisperse_rows(xo, delays, ds.astype(np.int64))
            got = out[b, torch.from_numpy(ds).cuda(), :nso].cpu().numpy()
            _f32_check(got, ref, ab, f"beam {b} series")
            # detection on the sampled series: per-series statistics make each series independent
            ev_o, cnt_o, _ = oracle.detect(np.ascontiguousarray(ref[None]), nso, cfg.snr_thresh)
            ev_o = ev_o.copy()
            ev_o["dm_idx"] = ds[ev_o["dm_idx"]]
            ev_o["beam"] = b
            sel = ev_g[(ev_g["beam"] == b) & np.isin(ev_g["dm_idx"], ds)]
            compare_events_f32(sel, ev_o, cfg.snr_thresh)
        tail = out[:, :, nso:]
        assert bool((tail == -7).all())


@pytest.mark.parametrize("dtype", ["f32", "u8"])
def test_4096_channels_with_element_offsets_beyond_2_to_32(dtype):
    """A 4096-channel plan whose last beam starts past 2^32 elements of the input (and, for the pre-summed rows, of the
    scratch): all series of the LAST beam against the oracle.  The other beams are device-generated filler."""
    torch = _torch()
    import paper_1307_5700_b200 as m
    nbeams, nchans, nsamps, ndms = (3, 4096, 532480, 24) if dtype == "f32" else (4, 4096, 360448, 24)
    args = (nbeams, nchans, 418.0, -20.0 / nchans, 51.2e-6, nsamps, 150.0, 0.1, ndms)
    assert (nbeams - 1) * nchans * nsamps > 2 ** 32
    delays = oracle.delay_table(nchans, 418.0, -20.0 / nchans, 51.2e-6, 150.0, 0.1, ndms)
    g = np.random.default_rng(77)
    last = nbeams - 1
    with Plan(args) as p:
        nso = p.nsamps_out
        if dtype == "f32":
            dx = torch.empty((nbeams, nchans, nsamps), dtype=torch.float32, device="cuda")
            dx.normal_(generator=torch.Generator(device="cuda").manual_seed(5))
            xb = np.empty((nchans, nsamps), dtype=np.float32)
            g.standard_normal(out=xb, dtype=np.float32)
        else:
            dx = torch.randint(0, 256, (nbeams, nchans, nsamps), dtype=torch.uint8, device="cuda",
                               generator=torch.Generator(device="cuda").manual_seed(5))
            xb = g.integers(0, 256, size=(nchans, nsamps), dtype=np.uint8)
        dx[last].copy_(torch.from_numpy(xb))
        out = p.dedisperse(dx, kernel=2)
        info = p.info(m.MDSM_F32 if dtype == "f32" else m.MDSM_U8)
        assert info["kernel"] == "rows"
        ds = np.arange(ndms, dtype=np.int64)
        ref, ab = oracle.dedisperse_rows(xb[None], delays, ds)
        got = out[last, :, :nso].cpu().numpy()
        if dtype == "f32":
            _f32_check(got, ref, ab, "last beam")
        else:
            assert np.array_equal(got.view(np.uint32), ref)
        assert bool((out[:, :, nso:] == -7).all())
