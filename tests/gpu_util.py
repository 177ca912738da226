"""Helpers for the GPU parity tests: run the CUDA path through the C-ABI binding, compare with the oracle."""
from __future__ import annotations

import numpy as np


def torch_cuda():
    import torch
    return torch


class Plan:
    """RAII wrapper used by tests only."""

    def __init__(self, cfg_or_args, scratch_limit=0):
        self.reserved = set()
        self.scratch_limit = scratch_limit
        import paper_1307_5700_b200 as m
        self.m = m
        args = cfg_or_args.plan_args() if hasattr(cfg_or_args, "plan_args") else tuple(cfg_or_args)
        (self.nbeams, self.nchans, self.f_top, self.foff, self.tsamp, self.nsamps, self.dm_low, self.dm_step,
         self.ndms) = args
        self.h = m.mdsm_plan_create(*args)
        self.max_delay = m.mdsm_plan_max_delay(self.h)
        self.nsamps_out = m.mdsm_plan_nsamps_out(self.h)

    def close(self):
        if self.h:
            self.m.mdsm_plan_destroy(self.h)
            self.h = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def info(self, dtype):
        return self.m.mdsm_plan_kernel_info(self.h, dtype)

    def set_option(self, key, value):
        self.m.mdsm_plan_set_option(self.h, key, value)
        if key == "group_size":
            self.reserved.clear()          # the option drops the reservation

    def delays(self):
        return self.m.mdsm_plan_get_delays(self.h, self.ndms, self.nchans)

    def dedisperse(self, d_in, beam0=0, nb=None, kernel=0, out=None):
        torch = torch_cuda()
        nb = self.nbeams - beam0 if nb is None else nb
        odt = torch.float32 if d_in.dtype == torch.float32 else torch.int32      # int32 storage for uint32
        if out is None:
            out = torch.full((self.nbeams, self.ndms, self.nsamps), -7, dtype=odt, device="cuda")
        self.m.mdsm_plan_set_option(self.h, "dedisp_kernel", kernel)
        dtype = self.m.MDSM_F32 if d_in.dtype == torch.float32 else self.m.MDSM_U8
        if kernel != 1 and dtype not in self.reserved:
            self.m.mdsm_plan_reserve(self.h, dtype, self.scratch_limit)
            self.reserved.add(dtype)
        self.m.mdsm_dedisperse(self.h, d_in, beam0, nb, out)
        torch.cuda.synchronize()
        return out

    def clip(self, d_in, window, k_chan, k_spec, beam0=0, nb=None):
        torch = torch_cuda()
        nb = self.nbeams - beam0 if nb is None else nb
        cm = torch.full((self.nbeams, self.nchans, self.nsamps // window), 9, dtype=torch.uint8, device="cuda")
        sm = torch.full((self.nbeams, self.nsamps), 9, dtype=torch.uint8, device="cuda")
        self.m.mdsm_rfi_clip(self.h, d_in, beam0, nb, window, k_chan, k_spec, cm, sm)
        torch.cuda.synchronize()
        return cm.cpu().numpy(), sm.cpu().numpy()

    def detect(self, d_out, thr, max_events=1 << 20, beam0=0, nb=None):
        torch = torch_cuda()
        nb = self.nbeams - beam0 if nb is None else nb
        ev = torch.zeros((max_events, 4), dtype=torch.int32, device="cuda")
        cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
        dtype = self.m.MDSM_F32 if d_out.dtype == torch.float32 else self.m.MDSM_U8
        self.m.mdsm_detect(self.h, d_out, beam0, nb, thr, ev, max_events, cnt, dtype=dtype)
        torch.cuda.synchronize()
        n = int(cnt.item())
        e = ev[: min(n, max_events)].cpu().numpy().view(self.m.EVENT_DTYPE).reshape(-1)
        e = e[np.lexsort((e["t"], e["dm_idx"], e["beam"]))]
        return e, n


def out_to_numpy(out, nso):
    """GPU out [nb][nd][nsamps] -> numpy [nb][nd][nso]; int32 storage is viewed as uint32."""
    a = out[:, :, :nso].cpu().numpy()
    return a.view(np.uint32) if a.dtype == np.int32 else a


def assert_f32_parity(gpu, ref, absum, what=""):
    """north_star tolerance: |gpu - oracle| <= 1e-5 * sum|in| + 1e-6."""
    err = np.abs(gpu.astype(np.float64) - ref)
    tol = 1e-5 * absum + 1e-6
    bad = err > tol
    assert not bad.any(), f"{what}: {bad.sum()} of {bad.size} outside tolerance, worst err/tol={np.max(err / tol):.3g}"
    return float(np.max(err / tol))


def compare_events_f32(ev_g, ev_o, thr, band=1e-3):
    """Reading D-vi: events within `band` of the threshold are optional on either side; all others must
    match on (beam, dm, t) with |dsnr| <= band."""
    def key(e):
        return {(int(a), int(b), int(c)): float(s) for a, b, c, s in zip(e["beam"], e["dm_idx"], e["t"], e["snr"])}
    g, o = key(ev_g), key(ev_o)
    for k, s in g.items():
        if k in o:
            assert abs(s - o[k]) <= band, (k, s, o[k])
        else:
            assert abs(s - thr) <= band, ("extra GPU event", k, s)
    for k, s in o.items():
        if k not in g:
            assert abs(s - thr) <= band, ("missing GPU event", k, s)
    return len(set(g) & set(o))
