"""ctypes binding of libmdsm.so -- argument marshalling only (see include/mdsm.h for semantics).

Every function has the name and argument order of its C counterpart.  Device buffers are
``torch`` CUDA tensors (or raw integer device pointers); streams are ``torch.cuda.Stream``
objects, raw ``cudaStream_t`` integers, or None for torch's current stream.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import (POINTER, c_char_p, c_double, c_int, c_int32, c_int64, c_uint64, c_void_p)

import numpy as np

__all__ = [
    "MDSM_F32", "MDSM_U8", "MDSM_U16", "MDSM_U4", "MDSM_OK", "MDSM_EINVAL", "MDSM_ENOMEM", "MDSM_ECUDA", "MDSM_EOVERFLOW",
    "EVENT_DTYPE", "MdsmError", "lib_path",
    "mdsm_plan_create", "mdsm_plan_destroy", "mdsm_plan_max_delay", "mdsm_plan_nsamps_out",
    "mdsm_plan_get_delays", "mdsm_last_error", "mdsm_plan_set_option", "mdsm_plan_launch_count",
    "mdsm_plan_reserve", "mdsm_plan_kernel_info",
    "mdsm_rfi_clip", "mdsm_bandpass_clip", "mdsm_dedisperse", "mdsm_detect", "mdsm_median_filter", "mdsm_detrend", "mdsm_power_i16", "mdsm_mulaw_u8", "mdsm_pipeline_host", "mdsm_measure_add_peak",
    "mdsm_cluster_events", "mdsm_classify_clusters", "mdsm_mulaw_c4",
    "mdsm_detect_noalloc", "MDSM_DETECT_NOALLOC_MAX_SERIES",
]

MDSM_F32, MDSM_U8, MDSM_U16, MDSM_U4 = 0, 1, 2, 3
MDSM_OK, MDSM_EINVAL, MDSM_ENOMEM, MDSM_ECUDA, MDSM_EOVERFLOW = 0, -1, -2, -3, 1
MDSM_DETECT_NOALLOC_MAX_SERIES = 32768      # the #define of include/mdsm.h (a test keeps the two equal)
EVENT_DTYPE = np.dtype([("beam", "<i4"), ("dm_idx", "<i4"), ("t", "<i4"), ("snr", "<f4")])

_HERE = os.path.dirname(os.path.abspath(__file__))


def lib_path() -> str:
    return os.path.join(_HERE, "libmdsm.so")


class MdsmError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"mdsm status {status}: {msg}")
        self.status = status


def _load():
    path = lib_path()
    if not os.path.exists(path):
        raise ImportError(
            f"{path} is missing: the CUDA extension has not been built "
            "(run `python paper_1307_5700_b200/build.py`). There is no CPU fallback.")
    L = ctypes.CDLL(path)
    L.mdsm_plan_create.restype = c_void_p
    L.mdsm_plan_create.argtypes = [c_int, c_int, c_double, c_double, c_double, c_int64, c_double, c_double, c_int]
    L.mdsm_plan_destroy.restype = None
    L.mdsm_plan_destroy.argtypes = [c_void_p]
    L.mdsm_plan_max_delay.restype = c_int64
    L.mdsm_plan_max_delay.argtypes = [c_void_p]
    L.mdsm_plan_nsamps_out.restype = c_int64
    L.mdsm_plan_nsamps_out.argtypes = [c_void_p]
    L.mdsm_plan_launch_count.restype = c_int64
    L.mdsm_plan_launch_count.argtypes = [c_void_p]
    L.mdsm_plan_get_delays.restype = c_int
    L.mdsm_plan_get_delays.argtypes = [c_void_p, c_void_p]
    L.mdsm_last_error.restype = c_char_p
    L.mdsm_last_error.argtypes = []
    L.mdsm_plan_set_option.restype = c_int
    L.mdsm_plan_set_option.argtypes = [c_void_p, c_char_p, c_int64]
    L.mdsm_plan_reserve.restype = c_int
    L.mdsm_plan_reserve.argtypes = [c_void_p, c_int, c_int64]
    L.mdsm_plan_kernel_info.restype = c_int
    L.mdsm_plan_kernel_info.argtypes = [c_void_p, c_int, c_char_p, c_int64]
    L.mdsm_rfi_clip.restype = c_int
    L.mdsm_rfi_clip.argtypes = [c_void_p, c_void_p, c_int, c_int, c_int, c_int, c_double, c_double, c_void_p,
                                c_void_p, c_void_p]
    L.mdsm_bandpass_clip.restype = c_int
    L.mdsm_bandpass_clip.argtypes = [c_void_p, c_void_p, c_int, c_int, c_int, c_int, c_double, c_double, c_double, c_int,
                                     c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]
    L.mdsm_dedisperse.restype = c_int
    L.mdsm_dedisperse.argtypes = [c_void_p, c_void_p, c_int, c_int, c_int, c_void_p, c_void_p]
    L.mdsm_detect.restype = c_int
    L.mdsm_detect.argtypes = [c_void_p, c_void_p, c_int, c_int, c_int, c_double, c_void_p, c_int64, c_void_p, c_void_p]
    L.mdsm_median_filter.restype = c_int
    L.mdsm_median_filter.argtypes = [c_void_p, c_void_p, c_void_p, c_int, c_int, c_int, c_void_p]
    L.mdsm_detrend.restype = c_int
    L.mdsm_detrend.argtypes = [c_void_p, c_void_p, c_int, c_int, c_void_p, c_void_p]
    L.mdsm_power_i16.restype = c_int
    L.mdsm_power_i16.argtypes = [c_void_p, c_void_p, c_int64, c_void_p]
    L.mdsm_mulaw_u8.restype = c_int
    L.mdsm_mulaw_u8.argtypes = [c_void_p, c_void_p, c_int64, c_double, c_void_p, c_void_p]
    L.mdsm_mulaw_c4.restype = c_int
    L.mdsm_mulaw_c4.argtypes = [c_void_p, c_void_p, c_int64, c_double, c_void_p, c_void_p]
    L.mdsm_cluster_events.restype = c_int
    L.mdsm_cluster_events.argtypes = [c_void_p, c_int64, c_double, c_double, c_double, c_double, c_double, c_int, c_int, c_void_p,
                                      POINTER(c_int64), POINTER(c_int64)]
    L.mdsm_classify_clusters.restype = c_int
    L.mdsm_classify_clusters.argtypes = [c_void_p, c_void_p, c_int64, c_int64, c_double, c_double, c_double, c_double, c_double,
                                         c_int, c_double, c_void_p]
    L.mdsm_pipeline_host.restype = c_int
    L.mdsm_pipeline_host.argtypes = [c_void_p, c_void_p, c_int, c_int, c_double, c_double, c_double, c_void_p,
                                     c_int64, POINTER(c_uint64), c_int]
    L.mdsm_measure_add_peak.restype = c_int
    L.mdsm_measure_add_peak.argtypes = [c_int, POINTER(c_double)]
    L.mdsm_detect_noalloc.restype = c_int
    L.mdsm_detect_noalloc.argtypes = [c_void_p, c_int, c_int, c_int, c_int64, c_int64, c_double, c_void_p, c_int64, c_void_p,
                                      c_void_p]
    return L


_L = _load()


def _ptr(x) -> int | None:
    """Device/host pointer of a torch tensor, numpy array, int or None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    raise TypeError(type(x))


def _stream(s) -> int | None:
    if s is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(s, int):
        return s
    return s.cuda_stream


def _dtype_of(x, dtype):
    if dtype is not None:
        return dtype
    name = str(getattr(x, "dtype", ""))
    if name.endswith("float32"):
        return MDSM_F32
    if name.endswith("uint8") or name.endswith("uint32") or name.endswith("int32"):
        return MDSM_U8
    if name.endswith("uint16") or name.endswith("int16"):
        return MDSM_U16
    raise TypeError(f"cannot infer mdsm dtype from {name!r}")


def _check(rc: int, allow=(MDSM_OK,)):
    if rc not in allow:
        raise MdsmError(rc, mdsm_last_error())
    return rc


def mdsm_last_error() -> str:
    return _L.mdsm_last_error().decode()


def mdsm_plan_create(nbeams, nchans, f_top, foff, tsamp, nsamps, dm_low, dm_step, ndms) -> int:
    h = _L.mdsm_plan_create(nbeams, nchans, f_top, foff, tsamp, nsamps, dm_low, dm_step, ndms)
    if not h:
        raise MdsmError(MDSM_EINVAL, mdsm_last_error())
    return h


def mdsm_plan_destroy(plan) -> None:
    _L.mdsm_plan_destroy(plan)


def mdsm_plan_max_delay(plan) -> int:
    return _L.mdsm_plan_max_delay(plan)


def mdsm_plan_nsamps_out(plan) -> int:
    return _L.mdsm_plan_nsamps_out(plan)


def mdsm_plan_launch_count(plan) -> int:
    return _L.mdsm_plan_launch_count(plan)


def mdsm_plan_get_delays(plan, ndms: int, nchans: int) -> np.ndarray:
    out = np.empty((ndms, nchans), dtype=np.int32)
    _check(_L.mdsm_plan_get_delays(plan, out.ctypes.data))
    return out


def mdsm_plan_set_option(plan, key: str, value: int) -> None:
    _check(_L.mdsm_plan_set_option(plan, key.encode(), value))


def mdsm_plan_reserve(plan, dtype: int, max_bytes: int = 0) -> None:
    _check(_L.mdsm_plan_reserve(plan, dtype, max_bytes))


def mdsm_plan_kernel_info(plan, dtype: int) -> dict:
    """The C call's "key=value ..." description as a dict (integers where they parse)."""
    buf = ctypes.create_string_buffer(512)
    rc = _L.mdsm_plan_kernel_info(plan, dtype, buf, len(buf))
    if rc < 0 and not buf.value:                     # "kernel=none reason=..." comes with MDSM_EINVAL and is still a description
        raise MdsmError(rc, mdsm_last_error())
    info = {}
    for kv in buf.value.decode().split():
        k, _, v = kv.partition("=")
        try:
            info[k] = int(v)
        except ValueError:
            info[k] = v
    return info


def mdsm_rfi_clip(plan, d_in, beam0, nb, window, k_chan, k_spec, d_chan_mask=None, d_spec_mask=None,
                  stream=None, dtype=None) -> None:
    _check(_L.mdsm_rfi_clip(plan, _ptr(d_in), _dtype_of(d_in, dtype), beam0, nb, window, k_chan, k_spec,
                            _ptr(d_chan_mask), _ptr(d_spec_mask), _stream(stream)))


def mdsm_bandpass_clip(plan, d_in, beam0, nb, window, order, k_mask, k_chan, k_spec, subtract, d_chan_mask=None,
                       d_spec_mask=None, d_fit=None, d_stats=None, stream=None) -> None:
    _check(_L.mdsm_bandpass_clip(plan, _ptr(d_in), beam0, nb, window, order, k_mask, k_chan, k_spec, int(bool(subtract)),
                                 _ptr(d_chan_mask), _ptr(d_spec_mask), _ptr(d_fit), _ptr(d_stats), _stream(stream)))


def mdsm_dedisperse(plan, d_in, beam0, nb, d_out, stream=None, dtype=None) -> None:
    _check(_L.mdsm_dedisperse(plan, _ptr(d_in), _dtype_of(d_in, dtype), beam0, nb, _ptr(d_out), _stream(stream)))


def mdsm_detect(plan, d_out, beam0, nb, snr_thresh, d_events, max_events, d_count, stream=None, dtype=None) -> None:
    _check(_L.mdsm_detect(plan, _ptr(d_out), _dtype_of(d_out, dtype), beam0, nb, snr_thresh, _ptr(d_events),
                          max_events, _ptr(d_count), _stream(stream)))


def mdsm_detect_noalloc(d_series, nbeams, ndms, nsamps, nsamps_out, snr_thresh, d_events, max_events, d_count, stream=None,
                        dtype=None) -> None:
    """mdsm_detect without a plan and without any device allocation inside the library, for callers that cannot call
    cudaMalloc (a plug-in in a process whose host application owns the GPU memory; a real-time loop that cannot afford
    cudaMalloc's device-wide stall).  At most MDSM_DETECT_NOALLOC_MAX_SERIES = nbeams * ndms series per call; calls
    share one fixed scratch array per GPU, so do not let two of them overlap on the device.  See include/mdsm.h."""
    _check(_L.mdsm_detect_noalloc(_ptr(d_series), _dtype_of(d_series, dtype), nbeams, ndms, nsamps, nsamps_out, snr_thresh,
                                  _ptr(d_events), max_events, _ptr(d_count), _stream(stream)))


def mdsm_median_filter(plan, d_series, d_filtered, beam0, nb, window, stream=None) -> None:
    _check(_L.mdsm_median_filter(plan, _ptr(d_series), _ptr(d_filtered), beam0, nb, window, _stream(stream)))


def mdsm_detrend(plan, d_series, beam0, nb, d_params=None, stream=None) -> None:
    _check(_L.mdsm_detrend(plan, _ptr(d_series), beam0, nb, _ptr(d_params), _stream(stream)))


def mdsm_power_i16(d_volt, d_power, n, stream=None) -> None:
    _check(_L.mdsm_power_i16(_ptr(d_volt), _ptr(d_power), n, _stream(stream)))


def mdsm_mulaw_u8(d_x, d_code, n, mu, d_xmax, stream=None) -> None:
    _check(_L.mdsm_mulaw_u8(_ptr(d_x), _ptr(d_code), n, mu, _ptr(d_xmax), _stream(stream)))


def mdsm_pipeline_host(plan, h_in, window, k_chan, k_spec, snr_thresh, h_events, max_events, nstreams=4,
                       dtype=None):
    """Returns (status, count); status is MDSM_OK or MDSM_EOVERFLOW."""
    cnt = c_uint64(0)
    rc = _L.mdsm_pipeline_host(plan, _ptr(h_in), _dtype_of(h_in, dtype), window, k_chan, k_spec, snr_thresh,
                               _ptr(h_events), max_events, ctypes.byref(cnt), nstreams)
    _check(rc, allow=(MDSM_OK, MDSM_EOVERFLOW))
    return rc, int(cnt.value)


def mdsm_measure_add_peak(kind: int) -> float:
    v = c_double(0.0)
    _check(_L.mdsm_measure_add_peak(kind, ctypes.byref(v)))
    return float(v.value)


def mdsm_mulaw_c4(d_volt, d_packed, n, mu, d_xmax_thr, stream=None) -> None:
    _check(_L.mdsm_mulaw_c4(_ptr(d_volt), _ptr(d_packed), n, mu, _ptr(d_xmax_thr), _stream(stream)))


def mdsm_cluster_events(h_events: np.ndarray, dm_low, dm_step, eps_t, eps_dm, eps_snr, min_pts, exact=False):
    """Host FDBSCAN / DBSCAN of an EVENT_DTYPE array. Returns (labels int32 [n], nclusters, region queries)."""
    ev = np.ascontiguousarray(h_events, dtype=EVENT_DTYPE)
    labels = np.empty(ev.shape[0], dtype=np.int32)
    ncl, nq = c_int64(0), c_int64(0)
    _check(_L.mdsm_cluster_events(ev.ctypes.data, ev.shape[0], dm_low, dm_step, eps_t, eps_dm, eps_snr, min_pts,
                                  1 if exact else 0, labels.ctypes.data, ctypes.byref(ncl), ctypes.byref(nq)))
    return labels, int(ncl.value), int(nq.value)


def mdsm_classify_clusters(h_events: np.ndarray, h_labels: np.ndarray, nclusters, dm_low, dm_step, tsamp, bw_mhz, nu_ghz,
                           k_smooth, rmse_max) -> np.ndarray:
    """Host DM-SNR classifier. Returns [nclusters][5] = class, dm_idx, snr, width_ms, rmse."""
    ev = np.ascontiguousarray(h_events, dtype=EVENT_DTYPE)
    lab = np.ascontiguousarray(h_labels, dtype=np.int32)
    res = np.zeros((nclusters, 5), dtype=np.float64)
    _check(_L.mdsm_classify_clusters(ev.ctypes.data, lab.ctypes.data, ev.shape[0], nclusters, dm_low, dm_step, tsamp, bw_mhz,
                                     nu_ghz, k_smooth, rmse_max, res.ctypes.data))
    return res
