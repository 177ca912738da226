"""mdsm_detect_noalloc: detection for callers that cannot allocate device memory.

Some users of the detection step cannot call cudaMalloc: a plug-in that runs inside a host application which has
already taken the GPU's memory and only lends out fixed buffers, or the paper's soft-real-time loop, where the
device-wide stall of a cudaMalloc / cudaFree can make other beams miss their deadline.  Every other stage call needs an
mdsm_plan, and creating a plan allocates.  mdsm_detect_noalloc needs no plan: its only scratch (one mean / rms pair per
series) sits in a fixed 512 KB array built into libmdsm.so, which limits a call to MDSM_DETECT_NOALLOC_MAX_SERIES series.

The GPU test compares it with the existing path (mdsm_detect on a plan) on two calls in a row, the second on other
data and a different shape so that values the first call left in the shared array would show.  This file sorts last on
purpose: `pytest -x` stops at the first failure, so a failure here cannot hide any other test.  It passes alone in a
fresh process (then its first call is the one that looks the array's address up) and after the other GPU tests.
"""
import os
import re

import numpy as np
import pytest

from gpu_util import Plan, compare_events_f32

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _sorted_events(m, ev, n, max_events):
    e = ev[: min(n, max_events)].cpu().numpy().view(m.EVENT_DTYPE).reshape(-1)
    return e[np.lexsort((e["t"], e["dm_idx"], e["beam"]))]


def _noalloc_detect(m, torch, d_series, nb, nd, ns, n, thr, max_events=1 << 20, measure_free=False):
    ev = torch.zeros((max_events, 4), dtype=torch.int32, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    dtype = m.MDSM_F32 if d_series.dtype == torch.float32 else m.MDSM_U8
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    m.mdsm_detect_noalloc(d_series, nb, nd, ns, n, thr, ev, max_events, cnt, dtype=dtype)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    if measure_free:
        assert free1 == free0, f"device free memory changed across the call: {free0} -> {free1}"
    c = int(cnt.item())
    return _sorted_events(m, ev, c, max_events), c


def _series(g, nb, nd, ns, n, base):
    s = np.rint(g.normal(size=(nb, nd, ns)) * 40 + base).astype(np.uint32)
    s[nb - 1, nd // 2, min(17, n - 1)] += 900
    s[0, 0, n - 1] += 700                   # last valid sample
    if n < ns:
        s[0, nd - 1, n] += 90000            # first sample past the valid range: must not be seen
    s[nb - 1, nd - 1, :] = 1234             # rms == 0: emits nothing
    return s


@pytest.mark.gpu
def test_noalloc_detect_at_its_series_limit_and_one_past_it():
    """Exactly MDSM_DETECT_NOALLOC_MAX_SERIES series run (the last pair of the array is used: a constant series next to
    a series with one spike); one more series is refused with a message that names the limit, and nothing is launched.
    Uses no plan at all and comes first in this file: run alone, it is the process's first call into libmdsm, so the
    address look-up happens before any other kernel of the library has been loaded on the device."""
    import torch
    import paper_1307_5700_b200 as m
    lim = m.MDSM_DETECT_NOALLOC_MAX_SERIES
    nb, nd, ns = 16, lim // 16, 96
    s = torch.full((nb, nd, ns), 5, dtype=torch.int32, device="cuda")
    s[nb - 1, nd - 1, 40] = 50
    s[0, 0, 3] = 9
    ev, c = _noalloc_detect(m, torch, s, nb, nd, ns, ns, 4.0, max_events=64)
    assert c == 2 and [(int(e["beam"]), int(e["dm_idx"]), int(e["t"])) for e in ev] == [(0, 0, 3), (nb - 1, nd - 1, 40)]
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    evb = torch.zeros((4, 4), dtype=torch.int32, device="cuda")
    with pytest.raises(m.MdsmError, match="MDSM_DETECT_NOALLOC_MAX_SERIES"):
        m.mdsm_detect_noalloc(s, nb, nd + 1, ns, ns, 4.0, evb, 4, cnt, dtype=m.MDSM_U8)
    torch.cuda.synchronize()
    assert int(cnt.item()) == 0


@pytest.mark.gpu
def test_noalloc_detect_matches_the_plan_path_on_two_calls_in_a_row():
    """uint32 series: same events as mdsm_detect, bit for bit (both forms reduce in exact integers), on two calls in a
    row that share the built-in scratch array; then float series within the guard band the other detection tests use.
    The second call has fewer series, other values and another length, so a stale mean / rms pair of the first call
    or a wrong row stride changes its events.  On the second call of each element type the device's free memory must not
    move (the first launch of a kernel may make the CUDA runtime load its code, which is not an allocation of ours)."""
    import torch
    import paper_1307_5700_b200 as m
    g = np.random.default_rng(2024)
    shapes = [(3, 11, 6003, 4000.0), (2, 5, 4100, 900.0)]        # (beams, DMs, samples per row, level)
    for call, (nb, nd, ns, base) in enumerate(shapes):
        args = (nb, 8, 418.0, -2.5, 51.2e-6, ns, 0.0, 0.15, nd)
        with Plan(args) as p:                                      # the existing path: a plan (allocates) + mdsm_detect
            n = p.nsamps_out
            assert n < ns
            s = _series(g, nb, nd, ns, n, base)
            d = torch.from_numpy(s.view(np.int32)).cuda()
            for thr in (3.0, -0.5):
                ev_p, cnt_p = p.detect(d, thr)
                ev_n, cnt_n = _noalloc_detect(m, torch, d, nb, nd, ns, n, thr, measure_free=call > 0)
                assert cnt_n == cnt_p > 10
                assert np.array_equal(ev_n, ev_p)
            # overflow behaves like mdsm_detect: the count keeps counting, what is stored is a subset
            ev_s, cnt_s = _noalloc_detect(m, torch, d, nb, nd, ns, n, 3.0, max_events=5)
            ev_p, cnt_p = p.detect(d, 3.0)
            assert cnt_s == cnt_p and len(ev_s) == 5
            allk = set(zip(ev_p["beam"], ev_p["dm_idx"], ev_p["t"]))
            assert all(k in allk for k in zip(ev_s["beam"], ev_s["dm_idx"], ev_s["t"]))
    # float series, two calls in a row again (after the integer calls above: the array now holds their statistics)
    for call, (nb, nd, ns) in enumerate(((2, 5, 7001), (1, 9, 5000))):
        args = (nb, 8, 418.0, -2.5, 51.2e-6, ns, 0.0, 0.15, nd)
        with Plan(args) as p:
            n = p.nsamps_out
            s = (g.normal(size=(nb, nd, ns)) * 8 + 3).astype(np.float32)
            s[nb - 1, 2, 100:104] += 60
            d = torch.from_numpy(s).cuda()
            ev_p, cnt_p = p.detect(d, 3.0)
            ev_n, cnt_n = _noalloc_detect(m, torch, d, nb, nd, ns, n, 3.0, measure_free=call > 0)
            assert compare_events_f32(ev_n, ev_p, 3.0) > 10
            assert abs(cnt_n - cnt_p) <= 2


def test_noalloc_limit_is_checked_before_any_cuda_call_and_constants_agree():
    """CPU-only: the size check needs no device (it comes before the address look-up), the header's #define equals the
    binding's constant, and detect.cu -- the file that holds the entry point -- contains no allocation call at all."""
    import paper_1307_5700_b200 as m
    hdr = open(os.path.join(ROOT, "include", "mdsm.h")).read()
    assert int(re.search(r"#define\s+MDSM_DETECT_NOALLOC_MAX_SERIES\s+(\d+)", hdr).group(1)) == m.MDSM_DETECT_NOALLOC_MAX_SERIES
    with pytest.raises(m.MdsmError, match="exceed the fixed scratch"):
        m.mdsm_detect_noalloc(0x1000, 2, m.MDSM_DETECT_NOALLOC_MAX_SERIES // 2 + 1, 64, 64, 3.0, 0x2000, 4, 0x3000, stream=0,
                              dtype=m.MDSM_U8)
    with pytest.raises(m.MdsmError, match="nsamps_out"):
        m.mdsm_detect_noalloc(0x1000, 1, 1, 64, 65, 3.0, 0x2000, 4, 0x3000, stream=0, dtype=m.MDSM_U8)
    src = open(os.path.join(ROOT, "paper_1307_5700_b200", "csrc", "detect.cu")).read()
    code = re.sub(r"//[^\n]*", "", src)
    for banned in ("cudaMalloc", "cudaFree", "cudaMallocAsync", "cudaHostAlloc", "cudaMallocManaged"):
        assert banned not in code, banned
    assert "cudaGetSymbolAddress" in code and "static __device__ __align__(256)" in code
