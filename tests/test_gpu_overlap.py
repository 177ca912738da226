"""Buffer-to-buffer continuity (reading A3; "a larger temporary GPU buffer to store the shifted samples", Eq. 6
PAPER.md:196-198 budgets (N_s + dt_max) N_c input words): consecutive buffers overlap by max_delay samples, each call produces
nsamps_out = nsamps - max_delay outputs, and the outputs of consecutive calls must join seamlessly -- equal to one long buffer
dedispersed at once, with nothing lost or doubled at the seam."""
import numpy as np
import pytest

import oracle

from gpu_util import Plan, out_to_numpy

pytestmark = pytest.mark.gpu

NC, F_TOP, FOFF, TSAMP, DM_LOW, DM_STEP, NDMS = 160, 418.0, -20.0 / 160, 51.2e-6, 0.0, 0.5, 48


def _geometry(n_out):
    d = oracle.delay_table(NC, F_TOP, FOFF, TSAMP, DM_LOW, DM_STEP, NDMS)
    md = int(d.max())
    return d, md, (2, NC, F_TOP, FOFF, TSAMP, 2 * n_out + md, DM_LOW, DM_STEP, NDMS), (2, NC, F_TOP, FOFF, TSAMP, n_out + md, DM_LOW, DM_STEP, NDMS)


@pytest.mark.parametrize("dtype", [np.uint8, np.float32])
@pytest.mark.parametrize("n_out", [5000, 4097])
def test_two_overlapping_buffers_equal_one_long_buffer(dtype, n_out):
    """One input of 2 n_out + max_delay samples dedispersed by one plan, against two calls of a plan for n_out + max_delay
    samples, the second buffer starting n_out samples later (its first max_delay samples are the first buffer's last).
    uint8: bit for bit.  fp32: both are the same sums of the same terms, possibly in another order -- each within the
    north_star tolerance of the oracle, hence within twice that of each other."""
    import torch
    d, md, long_args, short_args = _geometry(n_out)
    assert md > 1000                                           # a real overlap: the sweep spans many tiles
    g = np.random.default_rng(n_out)
    L = long_args[5]
    x = g.integers(0, 256, size=(2, NC, L)).astype(np.uint8) if dtype == np.uint8 else (g.normal(size=(2, NC, L)) * 2 + 5).astype(np.float32)
    ref, ab = oracle.dedisperse(x, d)
    with Plan(long_args) as p:
        assert p.nsamps_out == 2 * n_out and p.max_delay == md
        whole = out_to_numpy(p.dedisperse(torch.from_numpy(x).cuda(), kernel=0), 2 * n_out)
    halves = []
    with Plan(short_args) as p:
        assert p.nsamps_out == n_out
        for k in range(2):
            buf = np.ascontiguousarray(x[:, :, k * n_out:k * n_out + n_out + md])
            halves.append(out_to_numpy(p.dedisperse(torch.from_numpy(buf).cuda(), kernel=0), n_out).copy())
    joined = np.concatenate(halves, axis=2)
    if dtype == np.uint8:
        assert np.array_equal(whole, ref) and np.array_equal(joined, whole)
    else:
        tol = 1e-5 * ab + 1e-6
        assert np.all(np.abs(whole - ref) <= tol) and np.all(np.abs(joined - ref) <= tol)
        assert np.all(np.abs(joined.astype(np.float64) - whole) <= 2 * tol)


def test_pulses_at_the_seam_are_found_once_through_the_host_pipeline():
    """mdsm_pipeline_host on two consecutive overlapping uint8 buffers.  Three dispersed pulses: one whose sweep starts 5
    samples before the seam (it lives mostly in the overlap and belongs to buffer 1), one starting 7 samples after it
    (buffer 2, t = 7), one in the middle of buffer 2.  Each buffer's event list equals the oracle chain on that buffer bit
    for bit, and across the two lists every pulse peaks exactly once, at its own DM and start time."""
    import paper_1307_5700_b200 as m
    n_out = 6000
    d, md, long_args, short_args = _geometry(n_out)
    L = long_args[5]
    g = np.random.default_rng(99)
    x = np.clip(np.rint(g.normal(size=(2, NC, L)) * 6 + 60), 0, 255).astype(np.uint8)
    pulses = [(0, 30, n_out - 5), (1, 12, n_out + 7), (0, 41, n_out + 3000)]           # (beam, DM index, start sample)
    for b, k, t0 in pulses:
        x[b, np.arange(NC), t0 + d[k]] += 40
    found = []
    with Plan(short_args) as p:
        for buf_no in range(2):
            buf = np.ascontiguousarray(x[:, :, buf_no * n_out:buf_no * n_out + n_out + md])
            ref, _ = oracle.dedisperse(buf, d)
            ev_o, cnt_o, _ = oracle.detect(ref, n_out, 8.0)
            hev = np.zeros(1 << 16, dtype=m.EVENT_DTYPE)
            rc, cnt = m.mdsm_pipeline_host(p.h, buf, 0, 0.0, 0.0, 8.0, hev, len(hev), 2)
            assert rc == m.MDSM_OK and cnt == cnt_o
            hev = hev[:cnt]
            hev = hev[np.lexsort((hev["t"], hev["dm_idx"], hev["beam"]))]
            assert np.array_equal(hev, ev_o)
            for b in range(2):                                  # the strongest event of each beam in this buffer, in stream time
                e = hev[hev["beam"] == b]
                if len(e):
                    top = e[np.argmax(e["snr"])]
                    found.append((b, int(top["dm_idx"]), int(top["t"]) + buf_no * n_out, buf_no))
    # beam 0: pulse at n_out - 5 is buffer 1's strongest, pulse at n_out + 3000 buffer 2's; beam 1: only buffer 2 has one
    assert sorted(found) == sorted([(0, 30, n_out - 5, 0), (0, 41, n_out + 3000, 1), (1, 12, n_out + 7, 1)])
