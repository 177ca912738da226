"""CPU oracle for the BEST-2 transient-pipeline hot path -- TEST INFRASTRUCTURE ONLY.

Thin ctypes wrapper around ``oracle/mdsm_oracle.c`` (plain C + OpenMP, written from
/root/reference/PAPER.md: Eq. 1 at PAPER.md:93, brute-force dedispersion PAPER.md:96,
channel/spectrum thresholding PAPER.md:79-81, n-sigma detection PAPER.md:110,116).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_1307_5700_b200`` and the CUDA library imports nothing from here.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from ctypes import POINTER, c_double, c_int, c_int32, c_int64, c_uint8, c_uint32, c_void_p

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mdsm_oracle.c")
_SRC_NEXT = os.path.join(_HERE, "mdsm_oracle_next.c")          # the SURVEY 8(f) rows
_LIB = os.path.join(_HERE, "libmdsm_oracle.so")
# -ffp-contract=off / no fast-math: every fp64 op is a single IEEE op in the order written.
CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC", "-Wall"]

# MDSM_ORACLE_SANITIZE=1: the same sources with AddressSanitizer + UndefinedBehaviorSanitizer, in a library of its own
# (SURVEY section 5).  An ASan library only loads into a process that has the ASan runtime first in line:
#   MDSM_ORACLE_SANITIZE=1 LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 \
#       python -m pytest tests -m "not gpu" -q
# (leak detection off: CPython itself never frees everything).  Any finding aborts the process with a report.
SANITIZE = os.environ.get("MDSM_ORACLE_SANITIZE", "0") not in ("", "0")
if SANITIZE:
    _LIB = os.path.join(_HERE, "libmdsm_oracle_san.so")
    CFLAGS = ["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
              "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC", "-Wall"]

EVENT_DTYPE = np.dtype([("beam", "<i4"), ("dm_idx", "<i4"), ("t", "<i4"), ("snr", "<f4")])


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc if the .so is missing or older than the source."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_NEXT)):
        subprocess.run(["gcc", *CFLAGS, "-o", _LIB, _SRC, _SRC_NEXT, "-lm"], check=True)
    return _LIB


_lib = None


def _L():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.orc_detect_f32.restype = c_int64
        _lib.orc_detect_f64.restype = c_int64
        _lib.orc_detect_u32.restype = c_int64
        _lib.orc_num_threads.restype = c_int
        _lib.orc_dbscan.restype = c_int64
        _lib.orc_fdbscan.restype = c_int64
        _lib.orc_dm_response.restype = c_double
        _lib.orc_zeta.restype = c_double
    return _lib


def num_threads() -> int:
    return int(_L().orc_num_threads())


def _p(a):
    return None if a is None else a.ctypes.data_as(c_void_p)


def delay_table(nchans, f_top, foff, tsamp, dm_low, dm_step, ndms) -> np.ndarray:
    """delay[d][c] per Eq. 1 with north_star's constant and rounding."""
    out = np.empty((ndms, nchans), dtype=np.int32)
    _L().orc_delay_table(c_int(nchans), c_double(f_top), c_double(foff), c_double(tsamp),
                         c_double(dm_low), c_double(dm_step), c_int(ndms), _p(out))
    return out


def _check_in(x, dtype):
    assert x.dtype == dtype and x.ndim == 3 and x.flags.c_contiguous, (x.dtype, x.shape)
    return x.shape


def dedisperse(x: np.ndarray, delay: np.ndarray, variant: str = "rows", want_abs: bool = True):
    """out[b][d][t] = sum_c x[b][c][t + delay[d][c]], t < nsamps - max(delay).

    f32 input -> (out fp64, absum fp64 or None); u8 input -> (out uint32, None).
    variant: 'naive' (loops b,d,t,c) or 'rows' (loops b,d,c,t, OpenMP over (b,d)).
    """
    nb, nc, ns = x.shape
    nd = delay.shape[0]
    assert delay.shape == (nd, nc) and delay.dtype == np.int32 and delay.flags.c_contiguous
    nso = ns - int(delay.max())
    assert nso > 0
    L = _L()
    if x.dtype == np.float32:
        _check_in(x, np.float32)
        out = np.empty((nb, nd, nso), dtype=np.float64)
        ab = np.empty((nb, nd, nso), dtype=np.float64) if want_abs else None
        fn = L.orc_dedisperse_f32_naive if variant == "naive" else L.orc_dedisperse_f32_rows
        fn(_p(x), c_int(nb), c_int(nc), c_int64(ns), _p(delay), c_int(nd), c_int64(nso), _p(out), _p(ab))
        return out, ab
    _check_in(x, np.uint8)
    out = np.empty((nb, nd, nso), dtype=np.uint32)
    fn = L.orc_dedisperse_u8_naive if variant == "naive" else L.orc_dedisperse_u8_rows
    fn(_p(x), c_int(nb), c_int(nc), c_int64(ns), _p(delay), c_int(nd), c_int64(nso), _p(out))
    return out, None


def dedisperse_rows(x: np.ndarray, delay: np.ndarray, rows: np.ndarray, want_abs: bool = True):
    """Same definition for selected series only; rows[i] = b*ndms + d."""
    nb, nc, ns = x.shape
    nd = delay.shape[0]
    nso = ns - int(delay.max())
    rows = np.ascontiguousarray(rows, dtype=np.int64)
    assert rows.min() >= 0 and rows.max() < nb * nd
    L = _L()
    if x.dtype == np.float32:
        _check_in(x, np.float32)
        out = np.empty((len(rows), nso), dtype=np.float64)
        ab = np.empty((len(rows), nso), dtype=np.float64) if want_abs else None
        L.orc_dedisperse_f32_sel(_p(x), c_int(nb), c_int(nc), c_int64(ns), _p(delay), c_int(nd), c_int64(nso),
                                 _p(rows), c_int64(len(rows)), _p(out), _p(ab))
        return out, ab
    _check_in(x, np.uint8)
    out = np.empty((len(rows), nso), dtype=np.uint32)
    L.orc_dedisperse_u8_sel(_p(x), c_int(nb), c_int(nc), c_int64(ns), _p(delay), c_int(nd), c_int64(nso),
                            _p(rows), c_int64(len(rows)), _p(out))
    return out, None


def rfi_clip(x: np.ndarray, window: int, k_chan: float, k_spec: float, debug: bool = False):
    """In-place RFI clip of x[b][c][t] (readings B-i..B-viii).

    Returns dict(chan_mask [nb][nc][ns/window] u8, spec_mask [nb][ns] u8) plus, with
    debug=True, chan_mean/chan_sig/chan_thr/repl [nb][nc], spec_thr [nb][3]=(thr,mean,sig),
    spec_sum [nb][ns].
    """
    nb, nc, ns = x.shape
    assert x.flags.c_contiguous and x.flags.writeable
    if window < 1 or ns % window:
        raise ValueError("nsamps must be a multiple of window (reading B-viii)")
    cm = np.empty((nb, nc, ns // window), dtype=np.uint8)
    sm = np.empty((nb, ns), dtype=np.uint8)
    dbg = {}
    if debug:
        dbg = dict(chan_mean=np.empty((nb, nc)), chan_sig=np.empty((nb, nc)), chan_thr=np.empty((nb, nc)),
                   repl=np.empty((nb, nc)), spec_thr=np.empty((nb, 3)), spec_sum=np.empty((nb, ns)))
    fn = {np.dtype(np.float32): _L().orc_rfi_clip_f32, np.dtype(np.uint8): _L().orc_rfi_clip_u8}[x.dtype]
    rc = fn(_p(x), c_int(nb), c_int(nc), c_int64(ns), c_int(window), c_double(k_chan), c_double(k_spec),
            _p(cm), _p(sm), _p(dbg.get("chan_mean")), _p(dbg.get("chan_sig")), _p(dbg.get("chan_thr")),
            _p(dbg.get("repl")), _p(dbg.get("spec_thr")), _p(dbg.get("spec_sum")))
    if rc != 0:
        raise RuntimeError(f"orc_rfi_clip failed rc={rc}")
    return dict(chan_mask=cm, spec_mask=sm, **dbg)


def detect(series: np.ndarray, n_valid: int, snr_thresh: float, max_events: int | None = None):
    """n-sigma detection on series[b][d][stride>=n_valid] (readings D-i..D-vii).

    Returns (events structured array sorted by (beam, dm_idx, t), total_count, stats[nb][nd][2]=(mean,rms)).
    """
    assert series.ndim == 3 and series.flags.c_contiguous
    nb, nd, stride = series.shape
    assert 0 < n_valid <= stride
    if max_events is None:
        max_events = 1 << 22
    ev = np.zeros(max_events, dtype=EVENT_DTYPE)
    stats = np.empty((nb, nd, 2), dtype=np.float64)
    fn = {np.dtype(np.float32): _L().orc_detect_f32, np.dtype(np.float64): _L().orc_detect_f64,
          np.dtype(np.uint32): _L().orc_detect_u32}[series.dtype]
    cnt = fn(_p(series), c_int64(nb * nd), c_int(nd), c_int64(stride), c_int64(n_valid),
             c_double(snr_thresh), _p(ev), c_int64(max_events), _p(stats))
    ev = ev[: min(cnt, max_events)]
    ev = ev[np.lexsort((ev["t"], ev["dm_idx"], ev["beam"]))]
    return ev, int(cnt), stats


def median_filter(series: np.ndarray, n_valid: int, window: int) -> np.ndarray:
    """Windowed median of every series[..., :n_valid] (Eq. 2; reading E-i); the tail is copied."""
    assert series.dtype == np.float32 and series.flags.c_contiguous and window >= 1 and window % 2 == 1 and window <= 1023
    stride = series.shape[-1]
    out = series.copy()
    _L().orc_median_filter_f32(_p(series), c_int64(series.size // stride), c_int64(stride), c_int64(n_valid), c_int(window), _p(out))
    return out


def detrend(series: np.ndarray, n_valid: int):
    """Subtract the least-squares line and divide by the residual's standard deviation (reading E-ii).
    Returns (normalised float32 array, params[..., 3] = mean, slope, std)."""
    assert series.dtype == np.float32 and series.flags.c_contiguous
    stride = series.shape[-1]
    ns = series.size // stride
    out = series.copy()
    params = np.empty(series.shape[:-1] + (3,), dtype=np.float64)
    _L().orc_detrend_f32(_p(series), c_int64(ns), c_int64(stride), c_int64(n_valid), _p(out), _p(params))
    return out, params


def power_i16(volt: np.ndarray) -> np.ndarray:
    """|re + i im|^2 of interleaved int16 voltages [..., 2] -> float32 [...]."""
    assert volt.dtype == np.int16 and volt.shape[-1] == 2 and volt.flags.c_contiguous
    out = np.empty(volt.shape[:-1], dtype=np.float32)
    _L().orc_power_i16(_p(volt), c_int64(out.size), _p(out))
    return out


def mulaw_u8(x: np.ndarray, mu: float):
    """8-bit mu-law codes of a non-negative float32 series (Eq. 5; reading G-i). Returns (codes, xmax)."""
    assert x.dtype == np.float32 and x.flags.c_contiguous and mu > 0
    code = np.empty(x.shape, dtype=np.uint8)
    xmax = np.zeros(1, dtype=np.float32)
    _L().orc_mulaw_u8(_p(x), c_int64(x.size), c_double(mu), _p(code), _p(xmax))
    return code, float(xmax[0])


# ---------------------------------------------------------------- SURVEY 8(f) rows (mdsm_oracle_next.c)
def polyfit_u(y: np.ndarray, order: int) -> np.ndarray:
    """Least-squares coefficients (ascending powers of u = 2c/(n-1) - 1) of an order-p polynomial through y[c]."""
    y = np.ascontiguousarray(y, dtype=np.float64)
    coef = np.zeros(order + 1, dtype=np.float64)
    rc = _L().orc_polyfit_u(_p(y), c_int(y.size), c_int(order), _p(coef))
    if rc != 0:
        raise ValueError("singular fit")
    return coef


def bandpass_clip(x: np.ndarray, window: int, order: int, k_mask: float, k_chan: float, k_spec: float, subtract: bool):
    """The paper's bandpass-fit RFI stage (readings H-*), in place on x [nb][nchans][nsamps] float32.
    Returns dict(chan_mask, spec_mask, fit, bpi, rmse, mean_bp, std_bp, nmasked)."""
    assert x.dtype == np.float32 and x.ndim == 3 and x.flags.c_contiguous
    nb, nc, ns = x.shape
    cm = np.zeros((nb, nc, ns // window), dtype=np.uint8)
    sm = np.zeros((nb, ns), dtype=np.uint8)
    fit = np.zeros((nb, nc), dtype=np.float64)
    bpi = np.zeros((nb, nc), dtype=np.float64)
    st = np.zeros((nb, 4), dtype=np.float64)
    rc = _L().orc_bandpass_clip_f32(_p(x), c_int(nb), c_int(nc), c_int64(ns), c_int(window), c_int(order), c_double(k_mask),
                                    c_double(k_chan), c_double(k_spec), c_int(1 if subtract else 0), _p(cm), _p(sm), _p(fit),
                                    _p(bpi), _p(st))
    if rc != 0:
        raise ValueError(f"orc_bandpass_clip_f32 returned {rc}")
    return {"chan_mask": cm, "spec_mask": sm, "fit": fit, "bpi": bpi, "rmse": st[:, 0].copy(), "mean_bp": st[:, 1].copy(),
            "std_bp": st[:, 2].copy(), "nmasked": st[:, 3].astype(np.int64)}


def _points(pts):
    pts = np.ascontiguousarray(pts, dtype=np.float64)
    assert pts.ndim == 2 and pts.shape[1] == 3
    return pts


def dbscan(pts, eps, min_pts: int):
    """Textbook DBSCAN with a per-dimension box neighbourhood. Returns (labels int32, nclusters)."""
    pts = _points(pts)
    eps = np.ascontiguousarray(eps, dtype=np.float64)
    lab = np.empty(pts.shape[0], dtype=np.int32)
    n = _L().orc_dbscan(_p(pts), c_int64(pts.shape[0]), _p(eps), c_int(min_pts), _p(lab))
    return lab, int(n)


def fdbscan(pts, eps, min_pts: int):
    """FDBSCAN (representative seeds; reading K-ii). Returns (labels, nclusters, region queries made)."""
    pts = _points(pts)
    eps = np.ascontiguousarray(eps, dtype=np.float64)
    lab = np.empty(pts.shape[0], dtype=np.int32)
    nq = np.zeros(1, dtype=np.int64)
    n = _L().orc_fdbscan(_p(pts), c_int64(pts.shape[0]), _p(eps), c_int(min_pts), _p(lab), _p(nq))
    return lab, int(n), int(nq[0])


def dm_response(zeta: float) -> float:
    """Eq. 3."""
    return float(_L().orc_dm_response(c_double(zeta)))


def zeta(ddm: float, bw_mhz: float, w_ms: float, nu_ghz: float) -> float:
    """Eq. 4."""
    return float(_L().orc_zeta(c_double(ddm), c_double(bw_mhz), c_double(w_ms), c_double(nu_ghz)))


def classify_cluster(t, dm_idx, snr, dm_low, dm_step, tsamp, bw_mhz, nu_ghz, k_smooth, rmse_max):
    """The 8-step classifier of PAPER.md:144-156 for one cluster. Returns dict(cls, dm_idx, snr, width_ms, rmse)."""
    t = np.ascontiguousarray(t, dtype=np.int32)
    d = np.ascontiguousarray(dm_idx, dtype=np.int32)
    s = np.ascontiguousarray(snr, dtype=np.float32)
    res = np.zeros(5, dtype=np.float64)
    rc = _L().orc_classify_cluster(_p(t), _p(d), _p(s), c_int64(t.size), c_double(dm_low), c_double(dm_step), c_double(tsamp),
                                   c_double(bw_mhz), c_double(nu_ghz), c_int(k_smooth), c_double(rmse_max), _p(res))
    if rc != 0:
        raise ValueError("bad arguments")
    return {"cls": int(res[0]), "dm_idx": int(res[1]), "snr": float(res[2]), "width_ms": float(res[3]), "rmse": float(res[4])}


def mulaw_c4(volt: np.ndarray, mu: float):
    """2 x 16 bit -> 2 x 4 bit mu-law codes packed into one byte (Eq. 5; reading G-ii). Returns (bytes, xmax)."""
    assert volt.dtype == np.int16 and volt.shape[-1] == 2 and volt.flags.c_contiguous and mu > 0
    out = np.empty(volt.shape[:-1], dtype=np.uint8)
    xmax = np.zeros(1, dtype=np.int32)
    _L().orc_mulaw_c4(_p(volt), c_int64(out.size), c_double(mu), _p(out), _p(xmax))
    return out, int(xmax[0])


def dedisperse_u16(x: np.ndarray, delay: np.ndarray) -> np.ndarray:
    """Brute-force dedispersion of uint16 samples [nb][nchans][nsamps] -> uint32 [nb][ndms][nsamps_out] (exact)."""
    assert x.dtype == np.uint16 and x.ndim == 3 and x.flags.c_contiguous
    delay = np.ascontiguousarray(delay, dtype=np.int32)
    nb, nc, ns = x.shape
    nso = ns - int(delay.max())
    out = np.empty((nb, delay.shape[0], nso), dtype=np.uint32)
    _L().orc_dedisperse_u16_rows(_p(x), c_int(nb), c_int(nc), c_int64(ns), _p(delay), c_int(delay.shape[0]), c_int64(nso), _p(out))
    return out


def unpack_u4(x: np.ndarray) -> np.ndarray:
    """4-bit samples, two per byte along time (low nibble first) [..., nsamps/2] uint8 -> [..., nsamps] uint16."""
    assert x.dtype == np.uint8
    out = np.empty(x.shape[:-1] + (x.shape[-1] * 2,), dtype=np.uint16)
    out[..., 0::2] = x & 15
    out[..., 1::2] = x >> 4
    return out
