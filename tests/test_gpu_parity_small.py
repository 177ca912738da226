"""GPU-vs-oracle parity through the C ABI at sizes the oracle finishes in seconds (several tiles + ragged tails)."""
import numpy as np
import pytest

import oracle
from workloads import CONFIGS, generate

from gpu_util import Plan, assert_f32_parity, compare_events_f32, out_to_numpy

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    return torch


def _rand_input(shape, dtype, seed):
    g = np.random.default_rng(seed)
    if dtype == np.uint8:
        return np.clip(np.rint(64 + 10 * g.normal(size=shape)), 0, 255).astype(np.uint8)
    return (g.normal(size=shape) * (1 + g.uniform(size=(shape[0], shape[1], 1)))).astype(np.float32)


# (nbeams, nchans, f_top, foff, tsamp, nsamps, dm_low, dm_step, ndms)
SHAPES = {
    "cfg1": CONFIGS[1].plan_args(),
    "ragged": (3, 37, 418.0, -0.5, 51.2e-6, 5003, 0.0, 0.13, 13),          # unaligned rows, odd everything
    "multi_tile": (2, 96, 418.0, -0.2, 51.2e-6, 12288, 1.0, 0.1, 75),       # several DM blocks and time tiles
    "one_dm": (1, 16, 418.0, -1.0, 51.2e-6, 2048, 3.0, 0.0, 1),
    "one_chan": (2, 1, 418.0, -1.0, 51.2e-6, 1024, 0.0, 0.5, 9),
    "wide": (1, 512, 418.0, -20.0 / 512, 51.2e-6, 16384, 0.0, 0.1, 200),
    "tail8": (3, 37, 418.0, -0.5, 51.2e-6, 5000, 0.0, 0.13, 13),            # beams of 8k (not 16k) samples: u16 widening tail
    "parts": (2, 300, 418.0, -20.0 / 300, 51.2e-6, 16384, 0.0, 0.1, 100),   # two 256-channel parts on the integer path
}


@pytest.mark.parametrize("name", list(SHAPES))
def test_plan_delay_table_bit_exact(name):
    args = SHAPES[name]
    with Plan(args) as p:
        d = oracle.delay_table(args[1], args[2], args[3], args[4], args[6], args[7], args[8])
        assert np.array_equal(p.delays(), d)
        assert p.max_delay == int(d[-1, -1]) and p.nsamps_out == args[5] - int(d.max())


@pytest.mark.parametrize("k", [2, 5])
def test_plan_delay_table_full_configs(k):
    cfg = CONFIGS[k]
    torch = _torch()
    # plan creation for cfg 5 only needs the tables, not the data
    with Plan(cfg) as p:
        d = oracle.delay_table(cfg.nchans, cfg.f_top, cfg.foff, cfg.tsamp, cfg.dm_low, cfg.dm_step, cfg.ndms)
        assert np.array_equal(p.delays(), d)
    torch.cuda.synchronize()


@pytest.mark.parametrize("kernel", [1, 0])
@pytest.mark.parametrize("dtype", [np.float32, np.uint8])
@pytest.mark.parametrize("name", list(SHAPES))
def test_dedisperse_parity(name, dtype, kernel):
    torch = _torch()
    args = SHAPES[name]
    nb, nc, ns = args[0], args[1], args[5]
    x = generate(CONFIGS[1]) if (name == "cfg1" and dtype == np.float32) else _rand_input((nb, nc, ns), dtype, 42)
    d = oracle.delay_table(args[1], args[2], args[3], args[4], args[6], args[7], args[8])
    ref, ab = oracle.dedisperse(x, d)
    with Plan(args) as p:
        out = p.dedisperse(torch.from_numpy(x).cuda(), kernel=kernel)
        got = out_to_numpy(out, p.nsamps_out)
        if dtype == np.uint8:
            assert np.array_equal(got, ref)
        else:
            assert_f32_parity(got, ref, ab, name)
        # samples t >= nsamps_out are never touched
        tail = out[:, :, p.nsamps_out:].cpu().numpy()
        assert np.all(tail == -7)


@pytest.mark.parametrize("dtype", [np.float32, np.uint8])
def test_dedisperse_beam_subrange(dtype):
    torch = _torch()
    args = SHAPES["multi_tile"][:0] + (4,) + SHAPES["multi_tile"][1:]
    x = _rand_input((4, args[1], args[5]), dtype, 7)
    d = oracle.delay_table(args[1], args[2], args[3], args[4], args[6], args[7], args[8])
    ref, ab = oracle.dedisperse(x, d)
    with Plan(args) as p:
        dx = torch.from_numpy(x).cuda()
        out = p.dedisperse(dx, beam0=1, nb=2)
        got = out_to_numpy(out, p.nsamps_out)
        assert np.all(out[0].cpu().numpy() == -7) and np.all(out[3].cpu().numpy() == -7)
        if dtype == np.uint8:
            assert np.array_equal(got[1:3], ref[1:3])
        else:
            assert_f32_parity(got[1:3], ref[1:3], ab[1:3])


def _clip_case(dtype, seed=3, nb=2, nc=48, ns=8192, W=64):
    g = np.random.default_rng(seed)
    x = _rand_input((nb, nc, ns), dtype, seed)
    for _ in range(10):
        b, c, j = g.integers(nb), g.integers(nc), g.integers(ns // W)
        x[b, c, j * W:(j + 1) * W] = np.clip(x[b, c, j * W:(j + 1) * W].astype(np.float64) + 45, 0, 255).astype(dtype)
    x[0, 5] = np.clip(x[0, 5].astype(np.float64) + 30 * (np.sin(np.arange(ns) / 300.0) > 0.9), 0, 255).astype(dtype)
    for _ in range(6):
        b, t = g.integers(nb), g.integers(ns)
        x[b, :, t] = np.clip(x[b, :, t].astype(np.float64) + 70, 0, 255).astype(dtype)
    return x


@pytest.mark.parametrize("W", [64, 16, 512, 48, 1])
def test_clip_u8_bit_exact(W):
    torch = _torch()
    x = _clip_case(np.uint8, W=64)
    nb, nc, ns = x.shape
    if ns % W:
        ns = (ns // W) * W
        x = np.ascontiguousarray(x[:, :, :ns])
    xo = x.copy()
    r = oracle.rfi_clip(xo, W, 4.0, 4.0)
    with Plan((nb, nc, 418.0, -0.4, 51.2e-6, ns, 0.0, 0.1, 4)) as p:
        dx = torch.from_numpy(x).cuda()
        cm, sm = p.clip(dx, W, 4.0, 4.0)
        assert np.array_equal(cm, r["chan_mask"]) and np.array_equal(sm, r["spec_mask"])
        assert np.array_equal(dx.cpu().numpy(), xo)
        assert r["chan_mask"].sum() > 0 and (W == 1 or r["spec_mask"].sum() > 0)


def test_clip_u8_unaligned_rows():
    torch = _torch()
    x = np.ascontiguousarray(_clip_case(np.uint8)[:, :, :8190])       # 8190 = 2*3*3*5*7*13: not a multiple of 16
    nb, nc, ns = x.shape
    xo = x.copy()
    r = oracle.rfi_clip(xo, 90, 4.0, 4.0)
    with Plan((nb, nc, 418.0, -0.4, 51.2e-6, ns, 0.0, 0.1, 4)) as p:
        dx = torch.from_numpy(x).cuda()
        cm, sm = p.clip(dx, 90, 4.0, 4.0)
        assert np.array_equal(cm, r["chan_mask"]) and np.array_equal(sm, r["spec_mask"])
        assert np.array_equal(dx.cpu().numpy(), xo)


@pytest.mark.parametrize("W", [64, 4, 256, 1024])
def test_clip_f32_guard_band(W):
    """Reading B-ix: decisions may differ from the oracle only where the unit's z-score is within 1e-4 of k."""
    torch = _torch()
    x = _clip_case(np.float32, seed=5)
    nb, nc, ns = x.shape
    k = 4.0
    xo = x.copy()
    r = oracle.rfi_clip(xo, W, k, k, debug=True)
    with Plan((nb, nc, 418.0, -0.4, 51.2e-6, ns, 0.0, 0.1, 4)) as p:
        dx = torch.from_numpy(x).cuda()
        cm, sm = p.clip(dx, W, k, k)
    # raw (undilated) decisions outside the band must match; compare dilated masks where no nearby chunk is in the band
    csum = x.astype(np.float64).reshape(nb, nc, ns // W, W).sum(axis=3)
    z = (csum - W * r["chan_mean"][:, :, None]) / (np.maximum(r["chan_sig"], 1e-300)[:, :, None] * np.sqrt(W))
    near = np.abs(z - k) <= 1e-4
    near_d = near.copy()
    near_d[:, :, 1:] |= near[:, :, :-1]
    near_d[:, :, :-1] |= near[:, :, 1:]
    assert np.array_equal(cm[~near_d], r["chan_mask"][~near_d])
    if not near.any():
        zs = (r["spec_sum"] - r["spec_thr"][:, 1:2]) / np.maximum(r["spec_thr"][:, 2:3], 1e-300)
        near_s = np.abs(zs - k) <= 1e-4
        assert np.array_equal(sm[~near_s], r["spec_mask"][~near_s])
        if not near_s.any():
            got = dx.cpu().numpy()
            assert np.array_equal(got, xo)       # replacement values are (float)mean: allow 1 ulp below
    assert r["chan_mask"].sum() > 0 and r["spec_mask"].sum() > 0


def test_clip_beam_subrange_and_null_masks():
    torch = _torch()
    import paper_1307_5700_b200 as m
    x = _clip_case(np.uint8, nb=3)
    xo = x.copy()
    oracle.rfi_clip(xo[1:2], 64, 4.0, 4.0)
    with Plan((3, x.shape[1], 418.0, -0.4, 51.2e-6, x.shape[2], 0.0, 0.1, 4)) as p:
        dx = torch.from_numpy(x).cuda()
        m.mdsm_rfi_clip(p.h, dx, 1, 1, 64, 4.0, 4.0, None, None)
        torch.cuda.synchronize()
        assert np.array_equal(dx.cpu().numpy(), xo)
        with pytest.raises(m.MdsmError):
            m.mdsm_rfi_clip(p.h, dx, 0, 3, 100, 4.0, 4.0, None, None)          # 8192 % 100 != 0
        with pytest.raises(m.MdsmError):
            m.mdsm_rfi_clip(p.h, dx, 2, 2, 64, 4.0, 4.0, None, None)           # beam range


def test_detect_u32_bit_exact():
    torch = _torch()
    g = np.random.default_rng(9)
    nb, nd, ns = 2, 7, 6000
    args = (nb, 8, 418.0, -2.5, 51.2e-6, ns, 0.0, 0.15, nd)
    with Plan(args) as p:
        n = p.nsamps_out
        s = np.rint(g.normal(size=(nb, nd, ns)) * 40 + 4000).astype(np.uint32)
        s[1, 3, 17] += 900
        s[0, 0, n - 1] += 700
        s[0, 6, n] += 90000          # outside the valid range
        s[1, 5, :] = 1234            # constant series: rms == 0 -> no events
        ev_o, cnt_o, _ = oracle.detect(s, n, 3.0)
        ev_g, cnt_g = p.detect(torch.from_numpy(s.view(np.int32)).cuda(), 3.0)
        assert cnt_g == cnt_o > 10
        assert np.array_equal(ev_g, ev_o)          # includes the float snr, bit for bit
        # overflow: the count keeps counting, stored events are a subset
        ev_s, cnt_s = p.detect(torch.from_numpy(s.view(np.int32)).cuda(), 3.0, max_events=5)
        assert cnt_s == cnt_o and len(ev_s) == 5
        allk = set(zip(ev_o["beam"], ev_o["dm_idx"], ev_o["t"]))
        assert all((a, b, c) in allk for a, b, c in zip(ev_s["beam"], ev_s["dm_idx"], ev_s["t"]))


def test_detect_f32_guard_band():
    torch = _torch()
    g = np.random.default_rng(10)
    nb, nd, ns = 2, 5, 7001
    args = (nb, 8, 418.0, -2.5, 51.2e-6, ns, 0.0, 0.15, nd)
    with Plan(args) as p:
        n = p.nsamps_out
        s = (g.normal(size=(nb, nd, ns)) * 8 + 3).astype(np.float32)
        s[1, 2, 100:104] += 60
        ev_o, cnt_o, _ = oracle.detect(s, n, 3.0)
        ev_g, cnt_g = p.detect(torch.from_numpy(s).cuda(), 3.0)
        assert compare_events_f32(ev_g, ev_o, 3.0) > 10
        assert abs(cnt_g - cnt_o) <= 2


def test_chain_cfg1():
    """Config 1 end to end: clip -> dedisperse -> detect at 6 sigma, device-resident and via host buffers."""
    torch = _torch()
    import paper_1307_5700_b200 as m
    cfg = CONFIGS[1]
    x = generate(cfg)
    xo = x.copy()
    r = oracle.rfi_clip(xo, cfg.window, cfg.k_chan, cfg.k_spec)
    d = oracle.delay_table(cfg.nchans, cfg.f_top, cfg.foff, cfg.tsamp, cfg.dm_low, cfg.dm_step, cfg.ndms)
    ref, ab = oracle.dedisperse(xo, d)
    ev_o, cnt_o, _ = oracle.detect(ref, ref.shape[2], cfg.snr_thresh)
    with Plan(cfg) as p:
        dx = torch.from_numpy(x).cuda()
        cm, sm = p.clip(dx, cfg.window, cfg.k_chan, cfg.k_spec)
        assert np.array_equal(cm, r["chan_mask"]) and np.array_equal(sm, r["spec_mask"])
        out = p.dedisperse(dx)
        assert_f32_parity(out_to_numpy(out, p.nsamps_out), ref, ab)
        ev_g, cnt_g = p.detect(out, cfg.snr_thresh)
        assert compare_events_f32(ev_g, ev_o, cfg.snr_thresh) >= 20
        top = ev_g[np.argmax(ev_g["snr"])]
        assert top["dm_idx"] == 20 and 1000 <= top["t"] <= 1003
        # the same chain from host buffers through mdsm_pipeline_host
        hev = np.zeros(4096, dtype=m.EVENT_DTYPE)
        rc, cnt_h = m.mdsm_pipeline_host(p.h, x, cfg.window, cfg.k_chan, cfg.k_spec, cfg.snr_thresh, hev, 4096, 2)
        assert rc == m.MDSM_OK and cnt_h == cnt_g
        hev = hev[:cnt_h]
        hev = hev[np.lexsort((hev["t"], hev["dm_idx"], hev["beam"]))]
        assert np.array_equal(hev, ev_g)
        assert m.mdsm_plan_launch_count(p.h) >= 14


def test_chain_u8_small_bit_exact():
    torch = _torch()
    import paper_1307_5700_b200 as m
    args = (3, 64, 418.0, -0.3125, 51.2e-6, 8192, 0.0, 0.1, 40)
    x = _clip_case(np.uint8, nb=3, nc=64, ns=8192)
    d = oracle.delay_table(args[1], args[2], args[3], args[4], args[6], args[7], args[8])
    x[1, np.arange(64), 3000 + d[25]] += 60                     # one dispersed pulse
    xo = x.copy()
    r = oracle.rfi_clip(xo, 64, 5.0, 5.0)
    ref, _ = oracle.dedisperse(xo, d)
    ev_o, cnt_o, _ = oracle.detect(ref, ref.shape[2], 5.0)
    assert cnt_o > 0
    with Plan(args) as p:
        hev = np.zeros(1 << 16, dtype=m.EVENT_DTYPE)
        rc, cnt = m.mdsm_pipeline_host(p.h, x, 64, 5.0, 5.0, 5.0, hev, len(hev), 3)
        assert rc == m.MDSM_OK and cnt == cnt_o
        hev = hev[:cnt]
        hev = hev[np.lexsort((hev["t"], hev["dm_idx"], hev["beam"]))]
        assert np.array_equal(hev, ev_o)
        rc, cnt = m.mdsm_pipeline_host(p.h, x, 64, 5.0, 5.0, 5.0, hev, 3, 3)
        assert rc == m.MDSM_EOVERFLOW and cnt == cnt_o


def test_add_peak_microbenchmark_runs():
    import paper_1307_5700_b200 as m
    for kind in (0, 1, 2):
        v = m.mdsm_measure_add_peak(kind)
        assert 1e13 < v < 1e14


@pytest.mark.parametrize("name", ["cfg1", "ragged", "multi_tile", "wide", "parts"])
def test_tmem_operand_variant_matches_the_oracle(name):
    """dedisp_kernel = 3: the same pre-summed rows with the operand windows staged in tensor memory (tcgen05.st /
    tcgen05.ld at run-time column offsets).  Experimental (slower than the shared-memory variant), kept parity-green."""
    torch = _torch()
    args = SHAPES[name]
    nb, nc, ns = args[0], args[1], args[5]
    x = generate(CONFIGS[1]) if name == "cfg1" else _rand_input((nb, nc, ns), np.float32, 43)
    d = oracle.delay_table(args[1], args[2], args[3], args[4], args[6], args[7], args[8])
    ref, ab = oracle.dedisperse(x, d)
    with Plan(args) as p:
        p.set_option("dedisp_kernel", 3)
        info = p.info(p.m.MDSM_F32)
        if info.get("operands") != "tmem":
            pytest.skip(f"no TMEM tables for this plan: {info}")
        out = p.dedisperse(torch.from_numpy(x).cuda(), kernel=3)
        assert_f32_parity(out_to_numpy(out, p.nsamps_out), ref, ab, name)
        assert np.all(out[:, :, p.nsamps_out:].cpu().numpy() == -7)


@pytest.mark.parametrize("ns", [40, 131, 6000, 6003, 70001])
def test_detect_one_launch_and_two_launch_forms_agree_with_the_oracle(ns):
    """mdsm_detect is one launch (chunk maxima + revisits) by default; option detect_two_pass keeps the two-launch form.
    Both must give the oracle's events bit for bit on uint32 series, for aligned and unaligned rows, negative thresholds
    (every sample is a candidate) and series longer than one pass of the CTA."""
    torch = _torch()
    g = np.random.default_rng(ns)
    nb, nd = 2, 5
    args = (nb, 8, 418.0, -2.5, 51.2e-6, ns, 0.0, 0.15, nd)
    with Plan(args) as p:
        n = p.nsamps_out
        s = np.rint(g.normal(size=(nb, nd, ns)) * 40 + 4000).astype(np.uint32)
        s[1, 3, min(17, n - 1)] += 900
        s[0, 0, n - 1] += 700
        s[0, 2, n - 2:n] += 500
        s[1, 4, :] = 77
        d = torch.from_numpy(s.view(np.int32)).cuda()
        for thr in (3.0, -0.5):
            ev_o, cnt_o, _ = oracle.detect(s, n, thr)
            for two_pass in (0, 1):
                p.set_option("detect_two_pass", two_pass)
                l0 = p.m.mdsm_plan_launch_count(p.h)
                ev_g, cnt_g = p.detect(d, thr, max_events=1 << 21)
                assert p.m.mdsm_plan_launch_count(p.h) - l0 == (2 if two_pass else 1)
                assert cnt_g == cnt_o and np.array_equal(ev_g, ev_o)
