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


def test_coarse_dm_grid_still_runs_the_rows_kernel():
    """dm_step = 0.3: three times the delay spread per DM step of the BEST-2 grid, so a channel group takes many more
    delay patterns.  The plan's cost model must still find a group size whose tables fit the kernel (kernel=2 errors
    otherwise); whatever it picks must match the oracle."""
    torch = _torch()
    args = (2, 256, 418.0, -20.0 / 256, 51.2e-6, 16384, 0.0, 0.3, 60)
    g = np.random.default_rng(8)
    d = oracle.delay_table(args[1], args[2], args[3], args[4], args[6], args[7], args[8])
    xf = g.normal(size=(2, 256, 16384)).astype(np.float32)
    xu = g.integers(0, 256, size=(2, 256, 16384)).astype(np.uint8)
    with Plan(args) as p:
        assert p.info(0)["kernel"] == "rows" and p.info(1)["kernel"] == "rows"
        ref, ab = oracle.dedisperse(xf, d)
        got = out_to_numpy(p.dedisperse(torch.from_numpy(xf).cuda(), kernel=2), p.nsamps_out)
        assert np.all(np.abs(got - ref) <= 1e-5 * ab + 1e-6)
        refu, _ = oracle.dedisperse(xu, d)
        gotu = out_to_numpy(p.dedisperse(torch.from_numpy(xu).cuda(), kernel=2), p.nsamps_out)
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


def test_dedisperse_refuses_to_run_unreserved_and_reserve_reports_out_of_memory():
    """nothing is allocated per call.  The scratch of the rows kernel comes from mdsm_plan_reserve; without
    it mdsm_dedisperse returns MDSM_EINVAL (it never allocates or falls back silently), and a reservation that does not
    fit returns MDSM_ENOMEM and leaves the plan usable."""
    torch = _torch()
    import paper_1307_5700_b200 as m
    args = (1, 256, 418.0, -20.0 / 256, 51.2e-6, 1 << 17, 0.0, 0.1, 64)
    g = np.random.default_rng(12)
    x = g.normal(size=(1, 256, 1 << 17)).astype(np.float32)
    d = oracle.delay_table(args[1], args[2], args[3], args[4], args[6], args[7], args[8])
    ref, ab = oracle.dedisperse(x, d)
    with Plan(args) as p:
        dx = torch.from_numpy(x).cuda()
        out = torch.full((1, 64, 1 << 17), -7, dtype=torch.float32, device="cuda")
        with pytest.raises(m.MdsmError) as ei:
            m.mdsm_dedisperse(p.h, dx, 0, 1, out)
        assert ei.value.status == m.MDSM_EINVAL and "mdsm_plan_reserve" in str(ei.value)
        need = p.info(0)["nyrows"] * (1 << 17) * 4
        torch.cuda.synchronize()
        torch.cuda.empty_cache()
        free, _ = torch.cuda.mem_get_info()
        hog = torch.empty((max(free - need // 2, 0),), dtype=torch.uint8, device="cuda")   # leave half of what one beam needs
        try:
            with pytest.raises(m.MdsmError) as ei:
                m.mdsm_plan_reserve(p.h, m.MDSM_F32, 0)
            assert ei.value.status == m.MDSM_ENOMEM
        finally:
            del hog
            torch.cuda.empty_cache()
        m.mdsm_plan_reserve(p.h, m.MDSM_F32, 0)
        assert p.info(0)["scratch_slots"] == 1 and p.info(0)["scratch_bytes"] == need
        m.mdsm_dedisperse(p.h, dx, 0, 1, out)
        torch.cuda.synchronize()
        got = out_to_numpy(out, p.nsamps_out)
        assert np.all(np.abs(got - ref) <= 1e-5 * ab + 1e-6)


@pytest.mark.parametrize("dtype", [np.float32, np.uint8])
def test_stage_calls_neither_allocate_nor_synchronise(dtype):
    """SURVEY 8(b) "nothing is allocated per call ... no host sync inside": after mdsm_plan_reserve the three stage calls are
    captured into a CUDA graph on a side stream (stream capture fails on any synchronisation or cudaMalloc), free device
    memory does not change, and replaying the graph reproduces the result of the direct calls bit for bit."""
    torch = _torch()
    import paper_1307_5700_b200 as m
    args = (3, 128, 418.0, -20.0 / 128, 51.2e-6, 8192, 0.0, 0.1, 70)
    g = np.random.default_rng(21)
    x = g.normal(5.0, 1.0, size=(3, 128, 8192)).astype(np.float32) if dtype == np.float32 else g.integers(0, 256, size=(3, 128, 8192)).astype(np.uint8)
    mdt = m.MDSM_F32 if dtype == np.float32 else m.MDSM_U8
    with Plan(args) as p:
        m.mdsm_plan_reserve(p.h, mdt, 0)
        pristine = torch.from_numpy(x).cuda()
        work = pristine.clone()
        odt = torch.float32 if dtype == np.float32 else torch.int32
        out = torch.zeros((3, 70, 8192), dtype=odt, device="cuda")
        ev = torch.zeros((1 << 16, 4), dtype=torch.int32, device="cuda")
        cnt = torch.zeros(1, dtype=torch.int64, device="cuda")

        def chain(stream):
            m.mdsm_rfi_clip(p.h, work, 0, 3, 64, 5.0, 5.0, None, None, stream)
            m.mdsm_dedisperse(p.h, work, 0, 3, out, stream)
            m.mdsm_detect(p.h, out, 0, 3, 4.0, ev, 1 << 16, cnt, stream, dtype=mdt)

        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            chain(side)                                        # warm-up outside the capture (lazy module loading)
        side.synchronize()
        work.copy_(pristine); out.zero_(); cnt.zero_()
        torch.cuda.synchronize()
        free0, _ = torch.cuda.mem_get_info()
        chain(side)                                            # the plain calls: device memory must not move
        side.synchronize()
        free1, _ = torch.cuda.mem_get_info()
        assert free1 == free0
        ref_out, ref_cnt = out.clone(), int(cnt.item())
        work.copy_(pristine); out.zero_(); cnt.zero_()
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):             # raises if a call synchronises or allocates
            chain(side)
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, ref_out) and int(cnt.item()) == ref_cnt and ref_cnt > 0


@pytest.mark.parametrize("dtype", [np.float32, np.uint8])
def test_scratch_smaller_than_the_plan_walks_the_beams_through_it(dtype):
    """A reservation for fewer beams than the plan holds (config 5 on a full device): mdsm_dedisperse takes the beams
    through the scratch slots in stream order, for any beam0/nb, and mdsm_pipeline_host keeps to one stream."""
    torch = _torch()
    import paper_1307_5700_b200 as m
    args = (5, 96, 418.0, -20.0 / 96, 51.2e-6, 4096, 0.0, 0.1, 40)
    g = np.random.default_rng(33)
    x = g.normal(size=(5, 96, 4096)).astype(np.float32) if dtype == np.float32 else g.integers(0, 256, size=(5, 96, 4096)).astype(np.uint8)
    d = oracle.delay_table(args[1], args[2], args[3], args[4], args[6], args[7], args[8])
    ref, ab = oracle.dedisperse(x, d)
    mdt = m.MDSM_F32 if dtype == np.float32 else m.MDSM_U8
    with Plan(args) as p:
        per_beam = p.info(mdt)["nyrows"] * 4096 * (4 if dtype == np.float32 else 2)
        m.mdsm_plan_reserve(p.h, mdt, 2 * per_beam + 100)
        assert p.info(mdt)["scratch_slots"] == 2
        p.reserved.add(mdt)
        dx = torch.from_numpy(x).cuda()
        out = p.dedisperse(dx, kernel=2)
        p.dedisperse(dx, beam0=1, nb=3, kernel=2, out=out)                 # again, an odd sub-range
        got = out_to_numpy(out, p.nsamps_out)
        if dtype == np.float32:
            assert np.all(np.abs(got - ref) <= 1e-5 * ab + 1e-6)
        else:
            assert np.array_equal(got, ref)
        # the host pipeline on top of the small scratch
        ev_o, cnt_o, _ = oracle.detect(ref if dtype == np.uint8 else got.astype(np.float64), p.nsamps_out, 4.0)
        h_ev = np.zeros(1 << 16, dtype=m.EVENT_DTYPE)
        rc, cnt = m.mdsm_pipeline_host(p.h, x, 0, 0.0, 0.0, 4.0, h_ev, 1 << 16, 4)
        assert rc == m.MDSM_OK and abs(cnt - cnt_o) <= (0 if dtype == np.uint8 else 3)
        # the pipeline's own mdsm_plan_reserve(plan, dtype, 0) must keep the caller's two-slot cap: only then did the call
        # above take the one-stream branch this test is about
        assert p.info(mdt)["scratch_slots"] == 2
        m.mdsm_plan_reserve(p.h, mdt, 0)
        assert p.info(mdt)["scratch_slots"] == 2
        m.mdsm_plan_reserve(p.h, mdt, 3 * per_beam + 100)                  # an explicit size still replaces it
        assert p.info(mdt)["scratch_slots"] == 3


@pytest.mark.parametrize("G", [1, 2, 3, 4, 5, 6, 7, 8])
def test_every_group_size_matches_the_oracle(G):
    """Plan option group_size: every compiled pre-sum width, both dtypes, on a shape with a ragged last group (nchans not
    a multiple of G for most G), several 256-channel parts, a ragged DM block and unaligned rows (odd nsamps)."""
    torch = _torch()
    args = (2, 601, 418.0, -20.0 / 601, 51.2e-6, 6001, 0.0, 0.05, 83)
    g = np.random.default_rng(40 + G)
    d = oracle.delay_table(args[1], args[2], args[3], args[4], args[6], args[7], args[8])
    xf = g.normal(size=(2, 601, 6001)).astype(np.float32)
    xu = g.integers(0, 256, size=(2, 601, 6001)).astype(np.uint8)
    with Plan(args) as p:
        p.set_option("group_size", G)
        for mdt in (0, 1):
            info = p.info(mdt)
            assert info["kernel"] == "rows" and info["group_size"] == G, info
        ref, ab = oracle.dedisperse(xf, d)
        got = out_to_numpy(p.dedisperse(torch.from_numpy(xf).cuda(), kernel=2), p.nsamps_out)
        assert np.all(np.abs(got - ref) <= 1e-5 * ab + 1e-6)
        refu, _ = oracle.dedisperse(xu, d)
        outu = p.dedisperse(torch.from_numpy(xu).cuda(), kernel=2)
        assert np.array_equal(out_to_numpy(outu, p.nsamps_out), refu)
        assert (outu[:, :, p.nsamps_out:] == -7).all()                       # nothing past nsamps_out is touched


def test_kernel_info_reports_the_direct_kernel_and_its_reason():
    import paper_1307_5700_b200 as m
    args = (1, 64, 418.0, -0.3125, 51.2e-6, 4096, 0.0, 0.1, 32)
    with Plan(args) as p:
        assert p.info(m.MDSM_F32)["kernel"] == "rows"
        p.set_option("dedisp_kernel", 1)
        info = p.info(m.MDSM_U8)
        assert info["kernel"] == "direct" and info["reason"] == "option"
        # option 3 (TMEM operands) exists for fp32 only: kernel_info and mdsm_dedisperse must give the same verdict
        torch = _torch()
        p.set_option("dedisp_kernel", 3)
        info = p.info(m.MDSM_U8)
        assert info["kernel"] == "none" and info["reason"] == "tmem_f32_only"
        m.mdsm_plan_reserve(p.h, m.MDSM_U8, 0)
        x = torch.zeros((1, 64, 4096), dtype=torch.uint8, device="cuda")
        out = torch.zeros((1, 32, 4096), dtype=torch.int32, device="cuda")
        with pytest.raises(m.MdsmError) as ei:
            m.mdsm_dedisperse(p.h, x, 0, 1, out)
        assert ei.value.status == m.MDSM_EINVAL


def test_detect_on_a_series_too_long_for_the_one_launch_kernel_falls_back_by_itself():
    """The fused detection kernel keeps one maximum per 128 samples in shared memory; beyond ~5.2 M samples that no longer
    fits and mdsm_detect must take the two-launch form on its own (it used to return MDSM_EINVAL).  uint32: bit-exact."""
    torch = _torch()
    import paper_1307_5700_b200 as m
    ns = 6_000_000
    args = (1, 8, 418.0, -2.5, 51.2e-6, ns, 0.0, 0.15, 2)
    g = np.random.default_rng(77)
    with Plan(args) as p:
        n = p.nsamps_out
        s = (g.integers(0, 64, size=(1, 2, ns)) + 4000).astype(np.uint32)
        s[0, 1, n - 1] += 700
        s[0, 0, 5_500_000] += 900
        ev_o, cnt_o, _ = oracle.detect(s, n, 6.0)
        l0 = m.mdsm_plan_launch_count(p.h)
        ev_g, cnt_g = p.detect(torch.from_numpy(s.view(np.int32)).cuda(), 6.0)
        assert m.mdsm_plan_launch_count(p.h) - l0 == 2
        assert cnt_g == cnt_o >= 2 and np.array_equal(ev_g, ev_o)
