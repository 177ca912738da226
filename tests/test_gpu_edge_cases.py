"""Edge and degenerate cases of the CUDA path through the C ABI: the paper's pins applied to the GPU directly, the
capacity limit of the packed 16-bit lanes, empty results, argument errors."""
import numpy as np
import pytest

import oracle
from workloads import CONFIGS

from gpu_util import Plan, out_to_numpy

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    return torch


@pytest.mark.parametrize("kernel", [1, 2])
def test_u8_saturated_input_fills_the_16_bit_lanes_exactly(kernel):
    """All samples 255 over 1024 channels: every 256-channel part drives its u16 lanes to 65280 (the most they can
    hold) and every output must be exactly 1024 * 255."""
    torch = _torch()
    args = (1, 1024, 418.0, -20.0 / 1024, 51.2e-6, 4096, 0.0, 0.1, 48)
    x = np.full((1, 1024, 4096), 255, dtype=np.uint8)
    with Plan(args) as p:
        out = p.dedisperse(torch.from_numpy(x).cuda(), kernel=kernel)
        got = out_to_numpy(out, p.nsamps_out)
        assert got.min() == got.max() == 1024 * 255


@pytest.mark.parametrize("dtype", [np.float32, np.uint8])
def test_impulse_recovery_on_the_gpu(dtype):
    """SURVEY 8(c) P3 on the CUDA path: one unit impulse per channel along the sweep of DM index 20 of cfg 1 gives
    exactly nchans at (20, 1000), nothing larger anywhere, and every row sums to nchans."""
    torch = _torch()
    cfg = CONFIGS[1]
    with Plan(cfg) as p:
        d = p.delays()
        x = np.zeros((1, cfg.nchans, cfg.nsamps), dtype=dtype)
        x[0, np.arange(cfg.nchans), 1000 + d[20]] = 1
        for kernel in (1, 2):
            got = out_to_numpy(p.dedisperse(torch.from_numpy(x).cuda(), kernel=kernel), p.nsamps_out)[0].astype(np.float64)
            assert got[20, 1000] == cfg.nchans
            g2 = got.copy()
            g2[20, 1000] = 0
            assert g2.max() == 16                               # the worked value of SURVEY 8(c) P3
            assert np.all(got.sum(axis=1) == cfg.nchans)


def test_dm0_row_is_the_channel_sum_and_u8_is_linear():
    torch = _torch()
    args = (2, 300, 418.0, -20.0 / 300, 51.2e-6, 8192, 0.0, 0.1, 50)
    g = np.random.default_rng(5)
    a = g.integers(0, 100, size=(2, 300, 8192)).astype(np.uint8)
    b = g.integers(0, 100, size=(2, 300, 8192)).astype(np.uint8)
    with Plan(args) as p:
        n = p.nsamps_out
        oa = out_to_numpy(p.dedisperse(torch.from_numpy(a).cuda()), n).astype(np.int64)
        ob = out_to_numpy(p.dedisperse(torch.from_numpy(b).cuda()), n).astype(np.int64)
        oab = out_to_numpy(p.dedisperse(torch.from_numpy((a + b).astype(np.uint8)).cuda()), n).astype(np.int64)
        assert np.array_equal(oa[:, 0, :], a.astype(np.int64).sum(axis=1)[:, :n])      # P2
        assert np.array_equal(oab, oa + ob)                                            # P4, exact for integers


def test_no_events_constant_input_and_argument_errors():
    torch = _torch()
    import paper_1307_5700_b200 as m
    args = (2, 32, 418.0, -0.5, 51.2e-6, 4096, 0.0, 0.1, 8)
    with Plan(args) as p:
        x = np.full((2, 32, 4096), 7, dtype=np.uint8)
        dx = torch.from_numpy(x).cuda()
        cm, sm = p.clip(dx, 64, 5.0, 5.0)
        assert cm.sum() == 0 and sm.sum() == 0 and np.array_equal(dx.cpu().numpy(), x)   # constant input: no flags
        out = p.dedisperse(dx)
        assert np.all(out_to_numpy(out, p.nsamps_out) == 32 * 7)
        ev, cnt = p.detect(out, 6.0)
        assert cnt == 0 and len(ev) == 0                                                  # rms == 0: no events
        noise = torch.from_numpy(np.random.default_rng(1).normal(size=(2, 8, 4096)).astype(np.float32)).cuda()
        ev, cnt = p.detect(noise, 1e9)
        assert cnt == 0                                                                   # nothing above threshold
        for beam0, nb in ((0, 0), (1, 2), (-1, 1), (2, 1)):
            with pytest.raises(m.MdsmError):
                m.mdsm_dedisperse(p.h, dx, beam0, nb, out)
            with pytest.raises(m.MdsmError):
                m.mdsm_detect(p.h, out, beam0, nb, 6.0, torch.zeros((4, 4), dtype=torch.int32, device="cuda"), 4,
                              torch.zeros(1, dtype=torch.int64, device="cuda"), dtype=m.MDSM_U8)
    for bad in ((1, 8, 418.0, 0.5, 51.2e-6, 1024, 0.0, 0.1, 4),          # foff must be negative
                (1, 8, 418.0, -0.5, 51.2e-6, 16, 0.0, 50.0, 4),          # nsamps <= max_delay
                (0, 8, 418.0, -0.5, 51.2e-6, 1024, 0.0, 0.1, 4)):
        with pytest.raises(m.MdsmError):
            m.mdsm_plan_create(*bad)


def test_coarse_dm_grid_selects_a_narrower_tile_geometry():
    """dm_step = 0.3: three times the delay spread per DM step of the BEST-2 grid.  The automatic geometry choice must
    still find a tiled fp32 kernel (fewer DMs per warp); whatever runs must match the oracle."""
    torch = _torch()
    args = (2, 256, 418.0, -20.0 / 256, 51.2e-6, 16384, 0.0, 0.3, 60)
    g = np.random.default_rng(8)
    d = oracle.delay_table(args[1], args[2], args[3], args[4], args[6], args[7], args[8])
    xf = g.normal(size=(2, 256, 16384)).astype(np.float32)
    xu = g.integers(0, 256, size=(2, 256, 16384)).astype(np.uint8)
    with Plan(args) as p:
        ref, ab = oracle.dedisperse(xf, d)
        got = out_to_numpy(p.dedisperse(torch.from_numpy(xf).cuda(), kernel=2), p.nsamps_out)      # tiled, not direct
        assert np.all(np.abs(got - ref) <= 1e-5 * ab + 1e-6)
        refu, _ = oracle.dedisperse(xu, d)
        gotu = out_to_numpy(p.dedisperse(torch.from_numpy(xu).cuda(), kernel=0), p.nsamps_out)
        assert np.array_equal(gotu, refu)


def test_fp32_same_sign_data_stays_inside_the_tolerance_at_4096_channels():
    """The north_star tolerance 1e-5 * sum|in| + 1e-6 against sequential fp32 accumulation of 4096 same-sign terms
    (the hardest case for a running sum: no cancellation, the partial sum grows to 4096 times a term)."""
    torch = _torch()
    nch = 4096
    args = (1, nch, 418.0, -20.0 / nch, 51.2e-6, 16384, 0.0, 0.1, 96)
    g = np.random.default_rng(2)
    d = oracle.delay_table(args[1], args[2], args[3], args[4], args[6], args[7], args[8])
    for x in ((1000 + g.normal(size=(1, nch, 16384))).astype(np.float32), g.uniform(size=(1, nch, 16384)).astype(np.float32)):
        ref, ab = oracle.dedisperse(x, d)
        with Plan(args) as p:
            got = out_to_numpy(p.dedisperse(torch.from_numpy(x).cuda(), kernel=2), p.nsamps_out)
        ratio = np.abs(got.astype(np.float64) - ref) / (1e-5 * ab + 1e-6)
        assert ratio.max() < 0.7, ratio.max()              # measured 0.42 / 0.44: a factor two of margin


def test_pair_presum_falls_back_when_its_scratch_does_not_fit():
    """With device memory nearly full the fp32 path must go on without the pre-summed copy, not fail."""
    torch = _torch()
    import paper_1307_5700_b200 as m
    args = (1, 256, 418.0, -20.0 / 256, 51.2e-6, 1 << 17, 0.0, 0.1, 64)         # pair scratch ~ 2 x 134 MB
    g = np.random.default_rng(12)
    x = g.normal(size=(1, 256, 1 << 17)).astype(np.float32)
    d = oracle.delay_table(args[1], args[2], args[3], args[4], args[6], args[7], args[8])
    ref, ab = oracle.dedisperse(x, d)
    with Plan(args) as p:
        dx = torch.from_numpy(x).cuda()
        out = torch.full((1, 64, 1 << 17), -7, dtype=torch.float32, device="cuda")
        torch.cuda.synchronize()
        torch.cuda.empty_cache()
        free, _ = torch.cuda.mem_get_info()
        hog = torch.empty((max(free - (96 << 20), 0),), dtype=torch.uint8, device="cuda")   # leave 96 MB
        try:
            l0 = m.mdsm_plan_launch_count(p.h)
            m.mdsm_dedisperse(p.h, dx, 0, 1, out)
            torch.cuda.synchronize()
            assert m.mdsm_plan_launch_count(p.h) - l0 == 1                      # no pre-pass launch: plain tiled kernel
        finally:
            del hog
            torch.cuda.empty_cache()
        got = out_to_numpy(out, p.nsamps_out)
        assert np.all(np.abs(got - ref) <= 1e-5 * ab + 1e-6)
