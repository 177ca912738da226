"""SURVEY 8(f) NEXT-4 on the GPU against the oracle: 16-bit and 4-bit inputs of the dedispersion kernel (bit-exact) and
the 2 x 16 bit -> 2 x 4 bit mu-law quantiser (bit-exact: both sides decide in fp64 on integers)."""
import numpy as np
import pytest

import oracle

from gpu_util import Plan

pytestmark = pytest.mark.gpu

SHAPES = {
    "small": (2, 64, 418.0, -0.3125, 51.2e-6, 4096, 0.0, 0.1, 32),
    "multi_tile": (2, 96, 418.0, -0.2, 51.2e-6, 12288, 1.0, 0.1, 75),
    "wide": (1, 512, 418.0, -20.0 / 512, 51.2e-6, 16384, 0.0, 0.1, 200),
    "ragged": (3, 37, 418.0, -0.5, 51.2e-6, 5002, 0.0, 0.13, 13),
}


def _pack_u4(v):
    return (v[..., 0::2] | (v[..., 1::2] << 4)).astype(np.uint8)


@pytest.mark.parametrize("kernel", [0, 1])
@pytest.mark.parametrize("kind", ["u16", "u4"])
@pytest.mark.parametrize("name", list(SHAPES))
def test_low_precision_inputs_bit_exact(name, kind, kernel):
    import torch
    args = SHAPES[name]
    nb, nc, ns, nd = args[0], args[1], args[5], args[8]
    g = np.random.default_rng(7)
    delay = oracle.delay_table(nc, args[2], args[3], args[4], args[6], args[7], nd)
    if kind == "u16":
        x = g.integers(0, 65536, size=(nb, nc, ns), dtype=np.uint16)
        x[:, :, :64] = 65535                                   # saturated stretch: the 32-bit sums must not wrap
        ref = oracle.dedisperse_u16(x, delay)
        d_in = torch.from_numpy(x.view(np.int16)).cuda()
    else:
        v = g.integers(0, 16, size=(nb, nc, ns), dtype=np.uint8)
        v[:, :, 100:400] = 15                                  # fills the 16-bit lanes as far as they go
        ref = oracle.dedisperse_u16(v.astype(np.uint16), delay)
        assert np.array_equal(oracle.unpack_u4(_pack_u4(v)), v)
        d_in = torch.from_numpy(_pack_u4(v)).cuda()
    with Plan(args) as p:
        m = p.m
        dt = m.MDSM_U16 if kind == "u16" else m.MDSM_U4
        m.mdsm_plan_set_option(p.h, "dedisp_kernel", kernel)
        if kernel != 1:
            m.mdsm_plan_reserve(p.h, dt, 0)
            assert p.info(dt)["kernel"] == "rows"
        out = torch.full((nb, nd, ns), -7, dtype=torch.int32, device="cuda")
        m.mdsm_dedisperse(p.h, d_in, 0, nb, out, dtype=dt)
        torch.cuda.synchronize()
        got = out[:, :, :p.nsamps_out].cpu().numpy().view(np.uint32)
        assert np.array_equal(got, ref)
        assert np.all(out[:, :, p.nsamps_out:].cpu().numpy() == -7)


@pytest.mark.slow
@pytest.mark.parametrize("kind", ["u16", "u4"])
def test_low_precision_inputs_at_config_3_size_one_beam_every_element(kind):
    """One beam of the configuration the headline metric is quoted on (1024 channels x 65536 samples, 640 DM trials, the
    launch geometry bench.py times): every output element of the 16-bit and of the packed 4-bit input path against the oracle,
    bit for bit.  Seeded noise with a saturated stretch and a dispersed pulse."""
    import torch
    from workloads import CONFIGS
    cfg = CONFIGS[3]
    args = (1,) + cfg.plan_args()[1:]
    nc, ns, nd = cfg.nchans, cfg.nsamps, cfg.ndms
    delay = oracle.delay_table(nc, cfg.f_top, cfg.foff, cfg.tsamp, cfg.dm_low, cfg.dm_step, nd)
    g = np.random.default_rng(33)
    top = 65535 if kind == "u16" else 15
    v = g.integers(0, top + 1, size=(1, nc, ns), dtype=np.uint16)
    v[:, :, 5000:5256] = top
    v[0, np.arange(nc), 20000 + delay[333]] = top
    ref = oracle.dedisperse_u16(v, delay)
    d_in = torch.from_numpy(v.view(np.int16)).cuda() if kind == "u16" else torch.from_numpy(_pack_u4(v.astype(np.uint8))).cuda()
    with Plan(args) as p:
        m = p.m
        dt = m.MDSM_U16 if kind == "u16" else m.MDSM_U4
        m.mdsm_plan_reserve(p.h, dt, 0)
        assert p.info(dt)["kernel"] == "rows"
        out = torch.full((1, nd, ns), -7, dtype=torch.int32, device="cuda")
        m.mdsm_dedisperse(p.h, d_in, 0, 1, out, dtype=dt)
        torch.cuda.synchronize()
        got = out[:, :, :p.nsamps_out].cpu().numpy().view(np.uint32)
        assert np.array_equal(got, ref)
        assert int(got[0, 333, 20000]) >= (nc - 1) * top // 2 + top          # the pulse adds up at its DM
        assert np.all(out[:, :, p.nsamps_out:].cpu().numpy() == -7)


def test_u4_4096_channels_one_part_and_odd_nsamps_refused():
    import torch
    args = (1, 4096, 418.0, -20.0 / 4096, 51.2e-6, 8192, 0.0, 0.5, 24)
    g = np.random.default_rng(8)
    v = np.full((1, 4096, 8192), 15, dtype=np.uint8)           # 4096 * 15 = 61440: the most a 16-bit lane is asked to hold
    v[:, ::7, :] = g.integers(0, 16, size=v[:, ::7, :].shape, dtype=np.uint8)
    delay = oracle.delay_table(4096, args[2], args[3], args[4], args[6], args[7], 24)
    ref = oracle.dedisperse_u16(v.astype(np.uint16), delay)
    with Plan(args) as p:
        m = p.m
        m.mdsm_plan_reserve(p.h, m.MDSM_U4, 0)
        out = torch.zeros((1, 24, 8192), dtype=torch.int32, device="cuda")
        m.mdsm_dedisperse(p.h, torch.from_numpy(_pack_u4(v)).cuda(), 0, 1, out, dtype=m.MDSM_U4)
        torch.cuda.synchronize()
        assert np.array_equal(out[:, :, :p.nsamps_out].cpu().numpy().view(np.uint32), ref)
    with Plan((1, 8, 418.0, -1.0, 51.2e-6, 1001, 0.0, 0.1, 2)) as p:
        m = p.m
        m.mdsm_plan_set_option(p.h, "dedisp_kernel", 1)
        with pytest.raises(m.MdsmError):
            m.mdsm_dedisperse(p.h, torch.zeros(8 * 501, dtype=torch.uint8, device="cuda"), 0, 1,
                              torch.zeros((1, 2, 1001), dtype=torch.int32, device="cuda"), dtype=m.MDSM_U4)
        with pytest.raises(m.MdsmError):                       # clip and detect take MDSM_F32 / MDSM_U8 only
            m.mdsm_rfi_clip(p.h, torch.zeros(8 * 1001, dtype=torch.int16, device="cuda"), 0, 1, 1, 5.0, 5.0, dtype=m.MDSM_U16)


@pytest.mark.parametrize("n,mu,amp", [(1, 255.0, 1000), (17, 255.0, 3000), (100003, 255.0, 2000), (1 << 20, 10.0, 12000), (4099, 1e-3, 32767)])
def test_mulaw_c4_bit_exact(n, mu, amp):
    import torch
    import paper_1307_5700_b200 as m
    g = np.random.default_rng(n)
    v = np.clip(np.rint(g.normal(size=(n, 2)) * amp / 3.0), -32768, 32767).astype(np.int16)
    if n > 16:
        v[3] = (0, 0)
        v[5] = (-32768, 32767) if amp == 32767 else (amp, -amp)
    ref, xmax = oracle.mulaw_c4(v, mu)
    dv = torch.from_numpy(v).cuda()
    dp = torch.full((n + 16,), 77, dtype=torch.uint8, device="cuda")
    dx = torch.zeros(9, dtype=torch.int32, device="cuda")
    m.mdsm_mulaw_c4(dv, dp, n, mu, dx)
    torch.cuda.synchronize()
    hx = dx.cpu().numpy()
    assert int(hx[0]) == xmax
    assert np.array_equal(dp.cpu().numpy()[:n], ref) and np.all(dp.cpu().numpy()[n:] == 77)
    # the returned thresholds ARE the law: code k starts at thr[k-1]
    a = np.arange(0, xmax + 1, dtype=np.int32)
    codes, _ = oracle.mulaw_c4(np.stack([a, np.full_like(a, xmax)], axis=1).astype(np.int16), mu) if xmax <= 32767 else (None, None)
    if codes is not None:
        re = (codes & 15).astype(int)
        for k in range(1, 8):
            first = int(np.argmax(re >= k)) if (re >= k).any() else xmax + 1
            assert int(hx[k]) == first


def test_mulaw_c4_all_zero_and_errors():
    import torch
    import paper_1307_5700_b200 as m
    dv = torch.zeros((64, 2), dtype=torch.int16, device="cuda")
    dp = torch.full((64,), 9, dtype=torch.uint8, device="cuda")
    dx = torch.ones(9, dtype=torch.int32, device="cuda")
    m.mdsm_mulaw_c4(dv, dp, 64, 255.0, dx)
    torch.cuda.synchronize()
    assert int(dx[0].item()) == 0 and not dp.cpu().numpy().any()
    with pytest.raises(m.MdsmError):
        m.mdsm_mulaw_c4(dv, dp, 64, 0.0, dx)
    with pytest.raises(m.MdsmError):
        m.mdsm_mulaw_c4(dv, dp, -1, 255.0, dx)
