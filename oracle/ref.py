"""ctypes loader for the CPU oracle (oracle/gpfc_ref.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It
imports nothing from the CUDA package and holds no arithmetic of its own: every
function marshals numpy arrays into the C oracle and returns what it wrote.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gpfc_ref.c")
_SRCS = [_SRC, os.path.join(_HERE, "gpfc_ref_sim.c")]
_LIB = os.path.join(_HERE, "libgpfc_ref.so")

GRID_UNIFORM_FREQUENCY = 0
GRID_UNIFORM_PERIOD = 1
GRID_ENDPOINT_INCLUSIVE = 0
GRID_ENDPOINT_EXCLUSIVE = 2

CFLAGS = ["-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC"]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no FMA contraction).  Returns the .so path."""
    if (not force and os.path.exists(_LIB)
            and all(os.path.getmtime(_LIB) >= os.path.getmtime(f) for f in _SRCS)):
        return _LIB
    tmp = _LIB + ".tmp.%d" % os.getpid()
    subprocess.check_call(["gcc", *CFLAGS, "-o", tmp, *_SRCS, "-lm"])
    os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        c_dp = ctypes.c_void_p
        L.gpfc_ref_n_sample.restype = ctypes.c_double
        L.gpfc_ref_n_sample.argtypes = [ctypes.c_double] * 3
        L.gpfc_ref_make_period_grid.argtypes = [ctypes.c_double, ctypes.c_double,
                                                ctypes.c_int64, ctypes.c_int, c_dp]
        L.gpfc_ref_bin_index.argtypes = [c_dp, ctypes.c_int64, ctypes.c_double,
                                         ctypes.c_int, ctypes.c_double, c_dp]
        L.gpfc_ref_fold.argtypes = [c_dp, c_dp, ctypes.c_int64, c_dp, ctypes.c_int64,
                                    ctypes.c_int, ctypes.c_double, c_dp, c_dp, c_dp]
        L.gpfc_ref_normalize.argtypes = [c_dp, c_dp, ctypes.c_int64, ctypes.c_int,
                                         c_dp, c_dp]
        L.gpfc_ref_normalize_f64.argtypes = [c_dp, c_dp, ctypes.c_int64, ctypes.c_int,
                                             c_dp, c_dp]
        L.gpfc_ref_fold_batch.argtypes = [c_dp, c_dp, c_dp, ctypes.c_int64, c_dp,
                                          ctypes.c_int64, ctypes.c_int, c_dp,
                                          c_dp, c_dp, c_dp, c_dp, c_dp]
        L.gpfc_ref_two_tier_merge.argtypes = [c_dp, c_dp, ctypes.c_int, ctypes.c_int,
                                              c_dp, c_dp]
        L.gpfc_ref_philox4x32_10.argtypes = [c_dp, c_dp, c_dp]
        L.gpfc_ref_philox4x32_10.restype = None
        for name in ("gpfc_ref_ln", "gpfc_ref_cos2pi"):
            getattr(L, name).restype = ctypes.c_double
            getattr(L, name).argtypes = [ctypes.c_double]
        L.gpfc_ref_u32_to_unit.restype = ctypes.c_double
        L.gpfc_ref_u32_to_unit.argtypes = [ctypes.c_uint32]
        L.gpfc_ref_u52_to_unit.restype = ctypes.c_double
        L.gpfc_ref_u52_to_unit.argtypes = [ctypes.c_uint32, ctypes.c_uint32]
        L.gpfc_ref_normal.restype = ctypes.c_double
        L.gpfc_ref_normal.argtypes = [ctypes.c_uint64, ctypes.c_uint32, ctypes.c_uint32]
        L.gpfc_ref_lc_params_default.argtypes = [c_dp]
        L.gpfc_ref_make_light_curves.argtypes = [ctypes.c_uint64, ctypes.c_int64, ctypes.c_int64,
                                                 c_dp, c_dp, c_dp, c_dp]
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _chk(rc, what):
    if rc != 0:
        raise ValueError("%s failed with status %d" % (what, rc))


def _arr(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def n_sample(n_o: float, t_window: float, l_width: float) -> float:
    return float(lib().gpfc_ref_n_sample(n_o, t_window, l_width))


def make_period_grid(pmin, pmax, nperiods, mode_flags=0) -> np.ndarray:
    out = np.empty(max(int(nperiods), 0), dtype=np.float64)
    _chk(lib().gpfc_ref_make_period_grid(pmin, pmax, int(nperiods), int(mode_flags),
                                         _p(out)), "gpfc_ref_make_period_grid")
    return out


def bin_index(times, period, nbins, t0=0.0) -> np.ndarray:
    times = _arr(times, np.float64)
    out = np.empty(times.shape[0], dtype=np.int32)
    _chk(lib().gpfc_ref_bin_index(_p(times), times.shape[0], float(period), int(nbins),
                                  float(t0), _p(out)), "gpfc_ref_bin_index")
    return out


def fold(times, flux, periods, nbins, t0=0.0, want_sum64=True):
    """-> (sum fp32 [Np][nb], count u32 [Np][nb], sum64 fp64 [Np][nb] or None)."""
    times = _arr(times, np.float64)
    flux = _arr(flux, np.float32)
    periods = _arr(periods, np.float64)
    n, npd = times.shape[0], periods.shape[0]
    assert flux.shape[0] == n
    s = np.empty((npd, nbins), dtype=np.float32)
    c = np.empty((npd, nbins), dtype=np.uint32)
    s64 = np.empty((npd, nbins), dtype=np.float64) if want_sum64 else None
    _chk(lib().gpfc_ref_fold(_p(times), _p(flux), n, _p(periods), npd, int(nbins),
                             float(t0), _p(s), _p(c), _p(s64)), "gpfc_ref_fold")
    return s, c, s64


def fold_threaded(times, flux, periods, nbins, t0=0.0, threads=None, want_sum64=True):
    """Same as fold(); the period axis is split over a thread pool (ctypes drops
    the GIL).  Each period is still folded by the single-threaded C routine."""
    periods = _arr(periods, np.float64)
    npd = periods.shape[0]
    threads = threads or os.cpu_count() or 1
    if npd == 0 or threads <= 1:
        return fold(times, flux, periods, nbins, t0, want_sum64)
    times = _arr(times, np.float64)
    flux = _arr(flux, np.float32)
    n = times.shape[0]
    s = np.empty((npd, nbins), dtype=np.float32)
    c = np.empty((npd, nbins), dtype=np.uint32)
    s64 = np.empty((npd, nbins), dtype=np.float64) if want_sum64 else None
    nchunks = min(npd, threads * 4)
    edges = np.linspace(0, npd, nchunks + 1).astype(np.int64)
    L = lib()

    def work(i):
        lo, hi = int(edges[i]), int(edges[i + 1])
        if hi > lo:
            _chk(L.gpfc_ref_fold(_p(times), _p(flux), n, _p(periods[lo:hi]), hi - lo,
                                 int(nbins), float(t0), _p(s[lo:hi]), _p(c[lo:hi]),
                                 _p(s64[lo:hi]) if s64 is not None else None),
                 "gpfc_ref_fold")

    with ThreadPoolExecutor(max_workers=threads) as ex:
        list(ex.map(work, range(nchunks)))
    return s, c, s64


def normalize(sum32, count, want64=False):
    sum32 = _arr(sum32, np.float32)
    count = _arr(count, np.uint32)
    nb = sum32.shape[-1]
    nprof = sum32.size // nb if nb else 0
    out = np.empty(sum32.shape, dtype=np.float32)
    out64 = np.empty(sum32.shape, dtype=np.float64) if want64 else None
    _chk(lib().gpfc_ref_normalize(_p(sum32), _p(count), nprof, nb, _p(out), _p(out64)),
         "gpfc_ref_normalize")
    return (out, out64) if want64 else out


def normalize_f64(sum64, count, want64=False):
    sum64 = _arr(sum64, np.float64)
    count = _arr(count, np.uint32)
    nb = sum64.shape[-1]
    nprof = sum64.size // nb if nb else 0
    out = np.empty(sum64.shape, dtype=np.float32)
    out64 = np.empty(sum64.shape, dtype=np.float64) if want64 else None
    _chk(lib().gpfc_ref_normalize_f64(_p(sum64), _p(count), nprof, nb, _p(out),
                                      _p(out64)), "gpfc_ref_normalize_f64")
    return (out, out64) if want64 else out


def fold_batch(times, flux, offsets, periods, nbins, t0=None, want_norm=True,
               want64=True):
    """-> dict(sum, count, norm, sum64, norm64), each [ncurves][Np][nb]."""
    times = _arr(times, np.float64)
    flux = _arr(flux, np.float32)
    offsets = _arr(offsets, np.int64)
    periods = _arr(periods, np.float64)
    nc = offsets.shape[0] - 1
    npd = periods.shape[0]
    t0a = None if t0 is None else _arr(t0, np.float64)
    shape = (nc, npd, nbins)
    r = {
        "sum": np.empty(shape, np.float32),
        "count": np.empty(shape, np.uint32),
        "norm": np.empty(shape, np.float32) if want_norm else None,
        "sum64": np.empty(shape, np.float64) if want64 else None,
        "norm64": np.empty(shape, np.float64) if (want64 and want_norm) else None,
    }
    _chk(lib().gpfc_ref_fold_batch(_p(times), _p(flux), _p(offsets), nc, _p(periods),
                                   npd, int(nbins), _p(t0a), _p(r["sum"]),
                                   _p(r["count"]), _p(r["norm"]), _p(r["sum64"]),
                                   _p(r["norm64"])), "gpfc_ref_fold_batch")
    return r


def two_tier_merge(fine_sum64, fine_count, nb2):
    fine_sum64 = _arr(fine_sum64, np.float64)
    fine_count = _arr(fine_count, np.uint32)
    nb1 = fine_sum64.shape[-1]
    lead = fine_sum64.shape[:-1]
    fs = fine_sum64.reshape(-1, nb1)
    fc = fine_count.reshape(-1, nb1)
    osum = np.empty((fs.shape[0], nb2), np.float64)
    omean = np.empty((fs.shape[0], nb2), np.float64)
    for i in range(fs.shape[0]):
        _chk(lib().gpfc_ref_two_tier_merge(_p(fs[i]), _p(fc[i]), nb1, int(nb2),
                                           _p(osum[i]), _p(omean[i])),
             "gpfc_ref_two_tier_merge")
    return osum.reshape(lead + (nb2,)), omean.reshape(lead + (nb2,))


# ---- synthetic light-curve generator (oracle/gpfc_ref_sim.c)
LC_CENTERED = 1
LC_NO_NOISE = 2
LC_PARAM_NAMES = ("period", "duration", "sigma", "depth", "ratio_r", "epoch", "snr", "has_transit")


class LcParams(ctypes.Structure):
    """Mirror of gpfc_ref_lc_params (field order and types as in gpfc_ref_sim.c)."""
    _fields_ = [(k, ctypes.c_double) for k in (
        "period_lo", "period_hi", "duration_lo", "duration_hi", "ratio_lo", "ratio_hi",
        "sigma_lo", "sigma_hi", "snr_lo", "snr_hi", "transit_fraction", "cadence", "t_start")]
    _fields_ += [("flags", ctypes.c_int32), ("reserved", ctypes.c_int32)]


def lc_params_default(**over) -> LcParams:
    prm = LcParams()
    _chk(lib().gpfc_ref_lc_params_default(ctypes.byref(prm)), "gpfc_ref_lc_params_default")
    for k, v in over.items():
        setattr(prm, k, v)
    return prm


def philox4x32_10(ctr, key) -> np.ndarray:
    ctr = _arr(ctr, np.uint32)
    key = _arr(key, np.uint32)
    out = np.empty(4, np.uint32)
    lib().gpfc_ref_philox4x32_10(_p(ctr), _p(key), _p(out))
    return out


def ln(u: float) -> float:
    return float(lib().gpfc_ref_ln(float(u)))


def cos2pi(v: float) -> float:
    return float(lib().gpfc_ref_cos2pi(float(v)))


def u32_to_unit(x: int) -> float:
    return float(lib().gpfc_ref_u32_to_unit(int(x)))


def u52_to_unit(x0: int, x1: int) -> float:
    return float(lib().gpfc_ref_u52_to_unit(int(x0), int(x1)))


def normal(seed: int, curve: int, i: int) -> float:
    return float(lib().gpfc_ref_normal(int(seed), int(curve), int(i)))


def make_light_curves(seed, ncurves, n, prm: LcParams, want_times=True):
    """-> (times fp64 [ncurves][n] or None, flux fp32 [ncurves][n], params fp64 [ncurves][8])."""
    times = np.empty((ncurves, n), np.float64) if want_times else None
    flux = np.empty((ncurves, n), np.float32)
    par = np.empty((ncurves, 8), np.float64)
    _chk(lib().gpfc_ref_make_light_curves(int(seed), int(ncurves), int(n), ctypes.byref(prm),
                                          _p(times), _p(flux), _p(par)),
         "gpfc_ref_make_light_curves")
    return times, flux, par
