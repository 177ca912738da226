"""Seeded random plans (channel count, band, sampling time, DM grid, beams, buffer length) through both dedispersion
kernels against the oracle: the tile tables, shears, parts, ragged DM blocks and edge tiles of whatever geometry the
plan picks.  u8 bit-exact, fp32 inside the north_star tolerance."""
import numpy as np
import pytest

import oracle

from gpu_util import Plan, out_to_numpy

pytestmark = pytest.mark.gpu


def _shape(seed):
    g = np.random.default_rng(1000 + seed)
    nchans = int(g.choice([5, 24, 100, 257, 300, 512, 700]))
    bw = float(g.choice([5.0, 20.0, 32.0]))
    f_top = float(g.choice([418.0, 1400.0, 150.0]))
    if f_top - bw < 40.0:
        bw = 5.0
    tsamp = float(g.choice([51.2e-6, 64e-6, 1e-4]))
    ndms = int(g.integers(1, 130))
    dm_low = float(g.choice([0.0, 3.7, 20.0]))
    dm_step = float(g.choice([0.05, 0.1, 0.13, 0.25]))
    nbeams = int(g.integers(1, 4))
    args = [nbeams, nchans, f_top, -bw / nchans, tsamp, 0, dm_low, dm_step, ndms]
    d = oracle.delay_table(nchans, f_top, -bw / nchans, tsamp, dm_low, dm_step, ndms)
    nsamps = int(d.max()) + int(g.integers(1500, 6000))
    nsamps += (-nsamps) % int(g.choice([1, 4, 8, 16]))
    args[5] = nsamps
    return tuple(args), d


@pytest.mark.parametrize("seed", range(int(__import__("os").environ.get("MDSM_FUZZ_SEEDS", "24"))))
def test_random_plan(seed):
    import torch
    args, d = _shape(seed)
    if (args[5] - int(d.max())) * args[0] * args[8] * args[1] > 3e9:
        pytest.skip("oracle too slow for this draw")
    g = np.random.default_rng(seed)
    nb, nc, ns = args[0], args[1], args[5]
    xf = (g.normal(size=(nb, nc, ns)) * g.uniform(0.5, 2.0, size=(1, nc, 1)) + 3.0).astype(np.float32)
    xu = np.clip(np.rint(g.normal(size=(nb, nc, ns)) * 50 + 100), 0, 255).astype(np.uint8)
    with Plan(args) as p:
        n = p.nsamps_out
        assert np.array_equal(p.delays(), d)
        for x in (xf, xu):
            ref, ab = oracle.dedisperse(x, d)
            for kernel in (0, 1):
                out = p.dedisperse(torch.from_numpy(x).cuda(), kernel=kernel)
                got = out_to_numpy(out, n)
                if x.dtype == np.uint8:
                    assert np.array_equal(got, ref), (args, kernel)
                else:
                    assert np.all(np.abs(got.astype(np.float64) - ref) <= 1e-5 * ab + 1e-6), (args, kernel)
                assert bool((out[:, :, n:] == -7).all())


@pytest.mark.parametrize("seed", range(10))
def test_random_plan_u8_chain_bit_exact(seed):
    """clip -> dedisperse -> detect from host buffers (mdsm_pipeline_host) on random plans: the event list must equal
    the oracle's, bit for bit, for uint8 input."""
    import paper_1307_5700_b200 as m
    args, d = _shape(100 + seed)
    args = list(args)
    W = int(np.random.default_rng(seed).choice([8, 16, 64]))
    args[5] += (-args[5]) % W                                   # the clip wants nsamps % window == 0
    if (args[5] - int(d.max())) * args[0] * args[8] * args[1] > 3e9:
        pytest.skip("oracle too slow for this draw")
    g = np.random.default_rng(50 + seed)
    nb, nc, ns = args[0], args[1], args[5]
    x = np.clip(np.rint(g.normal(size=(nb, nc, ns)) * 10 + 64), 0, 255).astype(np.uint8)
    for _ in range(4):                                          # narrow-band bursts, broadband spikes, one pulse
        b, c, t = int(g.integers(nb)), int(g.integers(nc)), int(g.integers(ns - 200))
        x[b, c, t:t + 150] = np.minimum(x[b, c, t:t + 150].astype(int) + 60, 255)
        x[b, :, int(g.integers(ns))] = 200
    k = int(g.integers(args[8]))
    t0 = int(g.integers(0, ns - int(d.max()) - 1))
    x[0, np.arange(nc), t0 + d[k]] = np.minimum(x[0, np.arange(nc), t0 + d[k]].astype(int) + 90, 255)
    xo = x.copy()
    oracle.rfi_clip(xo, W, 5.0, 5.0)
    ref, _ = oracle.dedisperse(xo, d)
    ev_o, cnt_o, _ = oracle.detect(ref, ref.shape[2], 5.0)
    with Plan(tuple(args)) as p:
        hev = np.zeros(1 << 18, dtype=m.EVENT_DTYPE)
        rc, cnt = m.mdsm_pipeline_host(p.h, x, W, 5.0, 5.0, 5.0, hev, len(hev), 3)
        assert rc == m.MDSM_OK and cnt == cnt_o, (args, cnt, cnt_o)
        hev = hev[:cnt]
        hev = hev[np.lexsort((hev["t"], hev["dm_idx"], hev["beam"]))]
        assert np.array_equal(hev, ev_o), args


@pytest.mark.parametrize("G", [0, 8, 3])
def test_wide_sweep_at_low_frequency_picks_a_group_size_whose_pre_pass_fits(G):
    """A low band with a large DM: adjacent channels are thousands of samples apart, so the pre-pass of a wide channel
    group (G rows of chunk + delay range samples in shared memory) does not fit.  The plan must skip such a group size
    when it builds its tables -- or report the direct kernel for an explicit one -- instead of reporting kernel=rows and then
    failing every mdsm_dedisperse call at launch.  Whatever it picks has to run in 'auto' mode and match the oracle."""
    import torch
    import paper_1307_5700_b200 as m
    nchans, f_top, foff, tsamp, dm_low, dm_step, ndms = 48, 60.0, -0.25, 51.2e-6, 0.0, 0.7, 12
    d = oracle.delay_table(nchans, f_top, foff, tsamp, dm_low, dm_step, ndms)
    assert int(np.diff(d[-1]).max()) > 2000                     # adjacent channels, last DM: thousands of samples
    ns = int(d.max()) + 5000
    ns += (-ns) % 16
    args = (1, nchans, f_top, foff, tsamp, ns, dm_low, dm_step, ndms)
    g = np.random.default_rng(7)
    xf = (g.normal(size=(1, nchans, ns)) + 3.0).astype(np.float32)
    xu = g.integers(0, 256, size=(1, nchans, ns)).astype(np.uint8)
    with Plan(args) as p:
        if G:
            p.set_option("group_size", G)
        for x, mdt in ((xf, m.MDSM_F32), (xu, m.MDSM_U8)):
            info = p.info(mdt)
            assert info["kernel"] in ("rows", "direct"), info
            if G == 8 and mdt == m.MDSM_F32:                    # 8 rows x (2048 + ~18000) words = 640 KB (bytes still fit: 177 KB)
                assert info["kernel"] == "direct" and info["reason"] == "no_tables", info
            ref, ab = oracle.dedisperse(x, d)
            got = out_to_numpy(p.dedisperse(torch.from_numpy(x).cuda(), kernel=0), p.nsamps_out)
            if mdt == m.MDSM_U8:
                assert np.array_equal(got, ref), info
            else:
                assert np.all(np.abs(got.astype(np.float64) - ref) <= 1e-5 * ab + 1e-6), info
