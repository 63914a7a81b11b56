"""Thin ctypes binding of libgpfc.so (include/gpfc.h) -- argument marshalling only.

Every step of the path runs in the CUDA kernels of the library; torch is used
for device memory and streams.  Functions have the names of the C entry points.
If the library is missing or fails to load this module raises: there is no CPU
fallback and nothing here imports `oracle/`.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgpfc.so")

GPFC_OK = 0
GRID_UNIFORM_FREQUENCY = 0
GRID_UNIFORM_PERIOD = 1
GRID_ENDPOINT_INCLUSIVE = 0
GRID_ENDPOINT_EXCLUSIVE = 2
MAX_NBINS = 4096

EXPORTS = [
    "gpfc_version", "gpfc_last_error", "gpfc_set_stream", "gpfc_workspace_bytes",
    "gpfc_set_workspace", "gpfc_make_period_grid", "gpfc_n_sample", "gpfc_fold",
    "gpfc_normalize", "gpfc_fold_batch", "gpfc_make_period_grid_host",
    "gpfc_fold_batch_host", "gpfc_measure_peaks", "gpfc_profile", "gpfc_profile_read",
    "gpfc_merge_equal_count", "gpfc_init", "gpfc_fold_two_tier", "gpfc_path_counters",
    "gpfc_lc_params_default", "gpfc_make_light_curves", "gpfc_fold_stream", "gpfc_fold_noalloc",
]
OUT_SUM, OUT_COUNT, OUT_NORM = 1, 2, 4


class Chunk(ctypes.Structure):
    """gpfc_chunk of include/gpfc.h."""
    _fields_ = [("curve0", ctypes.c_int64), ("ncurves", ctypes.c_int64),
                ("period0", ctypes.c_int64), ("nperiods", ctypes.c_int64),
                ("nbins", ctypes.c_int32), ("slot", ctypes.c_int32),
                ("sum", ctypes.c_void_p), ("count", ctypes.c_void_p), ("norm", ctypes.c_void_p),
                ("ready", ctypes.c_void_p)]


CHUNK_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.POINTER(Chunk), ctypes.c_void_p, ctypes.c_void_p)


class _DeviceView:
    """Zero-copy view of library-owned device memory for torch.as_tensor."""

    def __init__(self, ptr, shape, typestr):
        self.__cuda_array_interface__ = {"shape": tuple(int(x) for x in shape), "typestr": typestr,
                                         "data": (int(ptr), False), "version": 3, "strides": None}

LC_CENTERED = 1
LC_NO_NOISE = 2
LC_PARAM_NAMES = ("period", "duration", "sigma", "depth", "ratio_r", "epoch", "snr", "has_transit")


class LcParams(ctypes.Structure):
    """gpfc_lc_params of include/gpfc.h (field order and types as declared there)."""
    _fields_ = [(k, ctypes.c_double) for k in (
        "period_lo", "period_hi", "duration_lo", "duration_hi", "ratio_lo", "ratio_hi",
        "sigma_lo", "sigma_hi", "snr_lo", "snr_hi", "transit_fraction", "cadence", "t_start")]
    _fields_ += [("flags", ctypes.c_int32), ("reserved", ctypes.c_int32)]



class GpfcError(RuntimeError):
    pass


_lib = None


def lib() -> ctypes.CDLL:
    """Load libgpfc.so (built in-tree by paper_2312_02063_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise GpfcError("libgpfc.so not found at %s: run `python -m paper_2312_02063_b200.build` "
                        "(there is no CPU fallback)" % LIB_PATH)
    L = ctypes.CDLL(LIB_PATH)
    vp, i64, i32, f64 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double
    L.gpfc_version.restype = ctypes.c_char_p
    L.gpfc_last_error.restype = ctypes.c_char_p
    L.gpfc_set_stream.argtypes = [vp]
    L.gpfc_workspace_bytes.restype = ctypes.c_size_t
    L.gpfc_workspace_bytes.argtypes = [i64, i64, i64, i32]
    L.gpfc_set_workspace.argtypes = [vp, ctypes.c_size_t]
    L.gpfc_make_period_grid.argtypes = [f64, f64, i64, i32, vp]
    L.gpfc_make_period_grid_host.argtypes = [f64, f64, i64, i32, vp]
    L.gpfc_n_sample.restype = f64
    L.gpfc_n_sample.argtypes = [f64, f64, f64]
    L.gpfc_fold.argtypes = [vp, vp, i64, vp, i64, i32, f64, vp, vp]
    L.gpfc_fold_noalloc.argtypes = [vp, vp, i64, vp, i64, i32, f64, vp, vp, vp]
    L.gpfc_normalize.argtypes = [vp, vp, i64, i32, vp]
    fb = [vp, vp, vp, i64, i64, vp, i64, i32, vp, vp, vp, vp]
    L.gpfc_fold_batch.argtypes = fb
    L.gpfc_fold_batch_host.argtypes = fb
    L.gpfc_measure_peaks.argtypes = [vp]
    L.gpfc_profile.argtypes = [i32]
    L.gpfc_merge_equal_count.argtypes = [vp, vp, i64, i32, i32, vp, vp]
    L.gpfc_profile_read.argtypes = [vp, vp, vp]
    L.gpfc_fold_two_tier.argtypes = [vp, vp, vp, i64, i64, vp, i64, i32, i32, vp, vp, vp]
    L.gpfc_path_counters.argtypes = [vp]
    L.gpfc_lc_params_default.argtypes = [vp]
    L.gpfc_make_light_curves.argtypes = [ctypes.c_uint64, i64, i64, vp, vp, vp, vp, vp]
    L.gpfc_fold_stream.argtypes = [vp, vp, vp, i64, i64, vp, i64, i32, vp, i32, ctypes.c_size_t, vp,
                                   CHUNK_FN, vp]
    _lib = L
    return L


def _check(rc: int, what: str):
    if rc != GPFC_OK:
        raise GpfcError("%s failed (status %d): %s"
                        % (what, rc, lib().gpfc_last_error().decode("utf-8", "replace")))


def _dptr(t, dtype, name):
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise GpfcError("%s must be a CUDA tensor" % name)
    if t.dtype != dtype or not t.is_contiguous():
        raise GpfcError("%s must be contiguous %s" % (name, dtype))
    return ctypes.c_void_p(t.data_ptr())


def _hptr(a, dtype, name):
    if a is None:
        return None
    if isinstance(a, torch.Tensor):
        if a.is_cuda or not a.is_contiguous():
            raise GpfcError("%s must be a contiguous host tensor" % name)
        return ctypes.c_void_p(a.data_ptr())
    if not isinstance(a, np.ndarray) or a.dtype != dtype or not a.flags["C_CONTIGUOUS"]:
        raise GpfcError("%s must be a contiguous numpy array of %s" % (name, dtype))
    return ctypes.c_void_p(a.ctypes.data)


def _use_current_stream():
    lib().gpfc_set_stream(ctypes.c_void_p(torch.cuda.current_stream().cuda_stream))


def gpfc_version() -> str:
    return lib().gpfc_version().decode()


def gpfc_last_error() -> str:
    return lib().gpfc_last_error().decode("utf-8", "replace")


def gpfc_set_stream(stream=None) -> None:
    """stream: a torch.cuda.Stream (None = torch's current stream).  The other wrappers call
    this with the current stream before every launch."""
    st = torch.cuda.current_stream() if stream is None else stream
    _check(lib().gpfc_set_stream(ctypes.c_void_p(st.cuda_stream)), "gpfc_set_stream")


def gpfc_n_sample(n_o: float, t_window: float, l_width: float) -> float:
    return float(lib().gpfc_n_sample(n_o, t_window, l_width))


def gpfc_workspace_bytes(ncurves: int, n_total: int, nperiods: int, nbins: int) -> int:
    return int(lib().gpfc_workspace_bytes(ncurves, n_total, nperiods, nbins))


def gpfc_set_workspace(ws) -> None:
    """ws: a CUDA uint8 tensor kept alive by the caller, or None to unregister."""
    if ws is None:
        _check(lib().gpfc_set_workspace(None, 0), "gpfc_set_workspace")
    else:
        _check(lib().gpfc_set_workspace(ctypes.c_void_p(ws.data_ptr()), ws.numel() * ws.element_size()),
               "gpfc_set_workspace")


def gpfc_make_period_grid(pmin, pmax, nperiods, mode_flags=0, out=None, device="cuda"):
    if out is None:
        out = torch.empty(max(int(nperiods), 0), dtype=torch.float64, device=device)
    _use_current_stream()
    _check(lib().gpfc_make_period_grid(float(pmin), float(pmax), int(nperiods), int(mode_flags),
                                       _dptr(out, torch.float64, "periods_out")),
           "gpfc_make_period_grid")
    return out


def gpfc_fold(times, flux, periods, nbins, t0=0.0, out_sum=None, out_count=None):
    n, npd = times.numel(), periods.numel()
    dev = times.device
    if out_sum is None:
        out_sum = torch.empty((npd, nbins), dtype=torch.float32, device=dev)
    if out_count is None:
        out_count = torch.empty((npd, nbins), dtype=torch.int32, device=dev)
    _use_current_stream()
    _check(lib().gpfc_fold(_dptr(times, torch.float64, "times"), _dptr(flux, torch.float32, "flux"),
                           n, _dptr(periods, torch.float64, "periods"), npd, int(nbins), float(t0),
                           _dptr(out_sum, torch.float32, "out_sum"),
                           _dptr(out_count, torch.int32, "out_count")), "gpfc_fold")
    return out_sum, out_count


def gpfc_fold_noalloc(times, flux, periods, nbins, t0, out_sum, out_count, out_norm):
    """gpfc_fold + fused normalisation on the library's static scratch: allocates nothing, so
    the caller passes every output it wants (None = not wanted); see include/gpfc.h for the
    size limits and the rule that overlapping calls race."""
    n, npd = times.numel(), periods.numel()
    _use_current_stream()
    _check(lib().gpfc_fold_noalloc(
        _dptr(times, torch.float64, "times"), _dptr(flux, torch.float32, "flux"), n,
        _dptr(periods, torch.float64, "periods"), npd, int(nbins), float(t0),
        _dptr(out_sum, torch.float32, "out_sum"), _dptr(out_count, torch.int32, "out_count"),
        _dptr(out_norm, torch.float32, "out_norm")), "gpfc_fold_noalloc")
    return out_sum, out_count, out_norm


def gpfc_normalize(sum_, count, out_norm=None):
    nb = sum_.shape[-1]
    nprof = sum_.numel() // nb if nb else 0
    if out_norm is None:
        out_norm = torch.empty_like(sum_)
    _use_current_stream()
    _check(lib().gpfc_normalize(_dptr(sum_, torch.float32, "sum"), _dptr(count, torch.int32, "count"),
                                nprof, nb, _dptr(out_norm, torch.float32, "out_norm")),
           "gpfc_normalize")
    return out_norm


def gpfc_merge_equal_count(sum_, count, nb2, want=("mean", "norm"), out_mean=None, out_norm=None):
    """sum_, count: [..., nb1] device tensors -> (mean, norm) [..., nb2] (None if not wanted)."""
    nb1 = sum_.shape[-1]
    nprof = sum_.numel() // nb1 if nb1 else 0
    shape = tuple(sum_.shape[:-1]) + (int(nb2),)
    if out_mean is None and "mean" in want:
        out_mean = torch.empty(shape, dtype=torch.float32, device=sum_.device)
    if out_norm is None and "norm" in want:
        out_norm = torch.empty(shape, dtype=torch.float32, device=sum_.device)
    _use_current_stream()
    _check(lib().gpfc_merge_equal_count(
        _dptr(sum_, torch.float32, "sum"), _dptr(count, torch.int32, "count"), nprof, nb1, int(nb2),
        _dptr(out_mean, torch.float32, "out_mean"), _dptr(out_norm, torch.float32, "out_norm")),
        "gpfc_merge_equal_count")
    return out_mean, out_norm


def gpfc_fold_batch(times, flux, offsets, periods, nbins, t0=None, out_sum=None, out_count=None,
                    out_norm=None, want=("sum", "count", "norm")):
    """Device tensors in, device tensors out.  `want` selects which outputs are
    allocated when none is passed in; want=("norm",) is the fused path."""
    nc, npd, n_total = offsets.numel() - 1, periods.numel(), times.numel()
    dev = times.device
    shape = (nc, npd, nbins)
    if out_sum is None and out_count is None and out_norm is None:
        if "sum" in want:
            out_sum = torch.empty(shape, dtype=torch.float32, device=dev)
        if "count" in want:
            out_count = torch.empty(shape, dtype=torch.int32, device=dev)
        if "norm" in want:
            out_norm = torch.empty(shape, dtype=torch.float32, device=dev)
    _use_current_stream()
    _check(lib().gpfc_fold_batch(
        _dptr(times, torch.float64, "times"), _dptr(flux, torch.float32, "flux"),
        _dptr(offsets, torch.int64, "offsets"), nc, n_total,
        _dptr(periods, torch.float64, "periods"), npd, int(nbins),
        _dptr(t0, torch.float64, "t0"), _dptr(out_sum, torch.float32, "out_sum"),
        _dptr(out_count, torch.int32, "out_count"), _dptr(out_norm, torch.float32, "out_norm")),
        "gpfc_fold_batch")
    return out_sum, out_count, out_norm


def gpfc_fold_two_tier(times, flux, offsets, periods, nb1, nb2, t0=None, out_mean=None,
                       out_norm=None, want=("mean", "norm")):
    """The paper's complete fold: nb1 intermediary bins merged to nb2 equal-count bins.
    offsets may be None for a single curve.  -> (mean, norm) [ncurves][Np][nb2]."""
    nc = 1 if offsets is None else offsets.numel() - 1
    npd, n_total = periods.numel(), times.numel()
    shape = (nc, npd, int(nb2))
    if out_mean is None and out_norm is None:
        if "mean" in want:
            out_mean = torch.empty(shape, dtype=torch.float32, device=times.device)
        if "norm" in want:
            out_norm = torch.empty(shape, dtype=torch.float32, device=times.device)
    _use_current_stream()
    _check(lib().gpfc_fold_two_tier(
        _dptr(times, torch.float64, "times"), _dptr(flux, torch.float32, "flux"),
        _dptr(offsets, torch.int64, "offsets"), nc, n_total,
        _dptr(periods, torch.float64, "periods"), npd, int(nb1), int(nb2),
        _dptr(t0, torch.float64, "t0"), _dptr(out_mean, torch.float32, "out_mean"),
        _dptr(out_norm, torch.float32, "out_norm")), "gpfc_fold_two_tier")
    return out_mean, out_norm


def gpfc_fold_stream(times, flux, offsets, periods, nbins, consumer, t0=None, want=("norm",),
                     slab_bytes=0, consumer_stream=None):
    """Chunked fold for a downstream consumer.  `consumer(chunk)` is called
    once per chunk with torch's current stream set to the consumer stream, which already waits
    for the chunk; `chunk` is a dict with curve0, ncurves, period0, nperiods, slot and the
    requested arrays "sum" / "count" / "norm" as tensors [ncurves][nperiods][nbins] that alias
    the library's slab: use them only in work enqueued on the current stream during the call
    (a scorer kernel, a copy), and do not block.  Returns once everything is enqueued."""
    nc = 1 if offsets is None else offsets.numel() - 1
    npd, n_total = periods.numel(), times.numel()
    outputs = (OUT_SUM if "sum" in want else 0) | (OUT_COUNT if "count" in want else 0) | \
              (OUT_NORM if "norm" in want else 0)
    cstream = consumer_stream if consumer_stream is not None else torch.cuda.current_stream()
    failure = []

    def on_chunk(chp, _stream, _user):
        try:
            ch = chp.contents
            shape = (ch.ncurves, ch.nperiods, ch.nbins)
            d = {"curve0": ch.curve0, "ncurves": ch.ncurves, "period0": ch.period0,
                 "nperiods": ch.nperiods, "slot": ch.slot}
            for name, ptr, ts in (("sum", ch.sum, "<f4"), ("count", ch.count, "<i4"),
                                  ("norm", ch.norm, "<f4")):
                d[name] = torch.as_tensor(_DeviceView(ptr, shape, ts), device=times.device) if ptr else None
            with torch.cuda.stream(cstream):
                consumer(d)
            return 0
        except BaseException as exc:      # never unwind through the C frame
            failure.append(exc)
            return 1

    cb = CHUNK_FN(on_chunk)
    _use_current_stream()
    rc = lib().gpfc_fold_stream(
        _dptr(times, torch.float64, "times"), _dptr(flux, torch.float32, "flux"),
        _dptr(offsets, torch.int64, "offsets"), nc, n_total, _dptr(periods, torch.float64, "periods"),
        npd, int(nbins), _dptr(t0, torch.float64, "t0"), outputs, int(slab_bytes),
        ctypes.c_void_p(cstream.cuda_stream), cb, None)
    if failure:
        raise failure[0]
    _check(rc, "gpfc_fold_stream")


def gpfc_lc_params_default(**over) -> LcParams:
    """Table 2's ranges, alpha in [6, 10]; keyword arguments override fields."""
    prm = LcParams()
    _check(lib().gpfc_lc_params_default(ctypes.byref(prm)), "gpfc_lc_params_default")
    for k, v in over.items():
        setattr(prm, k, v)
    return prm


def gpfc_make_light_curves(seed, ncurves, n, prm=None, device="cuda", want_times=True,
                           want_offsets=True, want_params=True):
    """Synthetic light curves generated on the device (PAPER.md 2.6).
    -> (times fp64 [ncurves][n] or None, flux fp32 [ncurves][n], offsets int64 [ncurves + 1] or
    None, params fp64 [ncurves][8] or None)."""
    prm = gpfc_lc_params_default() if prm is None else prm
    nc, n = int(ncurves), int(n)
    times = torch.empty((nc, n), dtype=torch.float64, device=device) if want_times else None
    flux = torch.empty((nc, n), dtype=torch.float32, device=device)
    offsets = torch.empty(nc + 1, dtype=torch.int64, device=device) if want_offsets else None
    params = torch.empty((nc, 8), dtype=torch.float64, device=device) if want_params else None
    _use_current_stream()
    _check(lib().gpfc_make_light_curves(
        ctypes.c_uint64(int(seed)), nc, n, ctypes.byref(prm), _dptr(times, torch.float64, "times"),
        _dptr(flux, torch.float32, "flux"), _dptr(offsets, torch.int64, "offsets"),
        _dptr(params, torch.float64, "params_out")), "gpfc_make_light_curves")
    return times, flux, offsets, params


def gpfc_init() -> None:
    _check(lib().gpfc_init(), "gpfc_init")


def gpfc_path_counters() -> dict:
    out = (ctypes.c_int64 * 8)()
    _use_current_stream()
    _check(lib().gpfc_path_counters(out), "gpfc_path_counters")
    return {"generic_kernel_calls": out[0], "exact_path_items": out[1],
            "guard_band_rechecks": out[2], "unfused_two_tier_calls": out[3],
            "count_overflow_refolds": out[4]}


def gpfc_make_period_grid_host(pmin, pmax, nperiods, mode_flags=0):
    out = np.empty(max(int(nperiods), 0), dtype=np.float64)
    _use_current_stream()
    _check(lib().gpfc_make_period_grid_host(float(pmin), float(pmax), int(nperiods),
                                            int(mode_flags), _hptr(out, np.float64, "out")),
           "gpfc_make_period_grid_host")
    return out


def gpfc_fold_batch_host(times, flux, offsets, periods, nbins, t0=None, out_sum=None,
                         out_count=None, out_norm=None):
    """Host buffers (numpy arrays or host torch tensors, pinned or not) in and
    out; the outputs must be passed in (None = not wanted)."""
    nc = offsets.shape[0] - 1
    _use_current_stream()
    _check(lib().gpfc_fold_batch_host(
        _hptr(times, np.float64, "times"), _hptr(flux, np.float32, "flux"),
        _hptr(offsets, np.int64, "offsets"), nc, times.shape[0],
        _hptr(periods, np.float64, "periods"), periods.shape[0], int(nbins),
        _hptr(t0, np.float64, "t0"), _hptr(out_sum, np.float32, "out_sum"),
        _hptr(out_count, np.uint32, "out_count"), _hptr(out_norm, np.float32, "out_norm")),
        "gpfc_fold_batch_host")
    return out_sum, out_count, out_norm


def gpfc_measure_peaks() -> dict:
    out = (ctypes.c_double * 8)()
    _use_current_stream()
    _check(lib().gpfc_measure_peaks(out), "gpfc_measure_peaks")
    return {"smem_atomic_lane_updates_per_s": out[0], "fp64_mul_add_pairs_per_s": out[1],
            "fold_loop_pp_per_s": out[2], "smem_cas_float_lane_updates_per_s": out[3],
            "smem_lds_sts_lane_updates_per_s": out[4]}


def gpfc_profile(enable: bool) -> None:
    _check(lib().gpfc_profile(1 if enable else 0), "gpfc_profile")


def gpfc_profile_read() -> dict:
    ms = ctypes.c_double(0.0)
    nf = ctypes.c_int64(0)
    nk = ctypes.c_int64(0)
    _check(lib().gpfc_profile_read(ctypes.byref(ms), ctypes.byref(nf), ctypes.byref(nk)),
           "gpfc_profile_read")
    return {"fold_kernel_ms": ms.value, "fold_launches": nf.value, "kernel_launches": nk.value}
