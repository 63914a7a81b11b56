"""Seeded synthetic inputs for the five BASELINE.json configs (numpy only).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds
none of the method's arithmetic: it only draws light curves (times, flux) and
names the period-grid parameters.  It imports neither `oracle/` nor the CUDA
binding.  The recipe is SURVEY.md 8(d) / DESIGN.md "Input recipe": the curves
stand in for Kepler DR25 (30,000-70,000 epochs at ~0.0204 d)
and TESS 2-min light curves, which are not available offline.

Every curve: slot index -> time = slot * cadence (fp64, starts at 0), flux =
1 + N(0, sigma) with an optional box transit, cast to fp32, then the fp32
median is subtracted (the paper folds detrended, normalised flux: PAPER.md:71,
Fig. 3(D)).  Seeds: numpy default_rng([config_id, curve_index]); config 0 uses
seed 0 as BASELINE.json states.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

KEPLER_CADENCE_D = 0.020433     # BASELINE.json configs 0-3
TESS_CADENCE_D = 0.0013889      # BASELINE.json config 4

GRID_UNIFORM_FREQUENCY = 0      # mirrors include/gpfc.h
GRID_UNIFORM_PERIOD = 1


@dataclass
class Workload:
    name: str
    config_id: int
    times: np.ndarray            # fp64 [n_total]
    flux: np.ndarray             # fp32 [n_total], median-subtracted
    offsets: np.ndarray          # int64 [ncurves + 1]
    pmin: float
    pmax: float
    nperiods: int
    grid_mode: int
    nbins: int
    fused_normalize: bool        # config 4: only the normalised profile is kept
    truth: list = field(default_factory=list)   # per curve: dict or None (injected box)

    @property
    def ncurves(self) -> int:
        return int(self.offsets.shape[0] - 1)

    @property
    def n_total(self) -> int:
        return int(self.times.shape[0])

    @property
    def point_periods(self) -> int:
        return self.n_total * int(self.nperiods)


def _box_mask(t, p0, dur, epoch):
    """In transit iff the time since (epoch - dur/2), modulo p0, is below dur."""
    ph = (t - epoch + 0.5 * dur) / p0
    ph = ph - np.floor(ph)
    return ph < (dur / p0)


def _finish(flux64):
    f32 = flux64.astype(np.float32)
    med = np.float32(np.median(f32))
    return (f32 - med).astype(np.float32)


def kepler_slots(rng) -> np.ndarray:
    """65,000 valid cadence slots out of 69,156 (1,413 d): three non-overlapping
    245-slot (5-day) gaps at random positions, then exactly 3,421 further slots
    (5.0 %) dropped uniformly at random."""
    nslots, gap, ngaps, ndrop = 69156, 245, 3, 3421
    while True:
        starts = np.sort(rng.integers(0, nslots - gap, size=ngaps))
        if np.all(np.diff(starts) >= gap):
            break
    keep = np.ones(nslots, dtype=bool)
    for s in starts:
        keep[s:s + gap] = False
    idx = np.flatnonzero(keep)
    drop = rng.choice(idx.shape[0], size=ndrop, replace=False)
    keep[idx[drop]] = False
    slots = np.flatnonzero(keep)
    assert slots.shape[0] == 65000
    return slots


def tess_slots() -> np.ndarray:
    """19,440 valid 2-min slots over 28 d: 0..9,719 and 10,440..20,159 (a
    720-slot = 1-day mid-sector gap)."""
    return np.concatenate([np.arange(0, 9720), np.arange(10440, 20160)])


def kepler_curve(rng, sigma, box):
    """box: None or dict(p0, depth, dur) (epoch drawn uniformly in [0, p0))."""
    slots = kepler_slots(rng)
    t = slots.astype(np.float64) * KEPLER_CADENCE_D
    f = 1.0 + rng.normal(0.0, sigma, size=t.shape[0])
    truth = None
    if box is not None:
        epoch = rng.uniform(0.0, box["p0"])
        f = f - box["depth"] * _box_mask(t, box["p0"], box["dur"], epoch)
        truth = dict(box, epoch=float(epoch))
    return t, _finish(f), truth


def _pack(name, cid, curves, pmin, pmax, nperiods, nbins, fused):
    times = np.concatenate([c[0] for c in curves]) if curves else np.zeros(0)
    flux = np.concatenate([c[1] for c in curves]) if curves else np.zeros(0, np.float32)
    lens = np.array([c[0].shape[0] for c in curves], dtype=np.int64)
    offsets = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    return Workload(name=name, config_id=cid, times=np.ascontiguousarray(times, np.float64),
                    flux=np.ascontiguousarray(flux, np.float32), offsets=offsets,
                    pmin=pmin, pmax=pmax, nperiods=int(nperiods),
                    grid_mode=GRID_UNIFORM_FREQUENCY, nbins=nbins,
                    fused_normalize=fused, truth=[c[2] for c in curves])


def config0(nperiods=2000):
    """Tiny single curve (BASELINE.json configs[0]); seed 0."""
    rng = np.random.default_rng(0)
    n = 4000
    t = np.arange(n, dtype=np.float64) * KEPLER_CADENCE_D
    box = dict(p0=0.5, depth=5e-4, dur=0.04, epoch=0.1)
    f = 1.0 + rng.normal(0.0, 1e-3, size=n)
    f = f - box["depth"] * _box_mask(t, box["p0"], box["dur"], box["epoch"])
    return _pack("config0_tiny", 0, [(t, _finish(f), box)], 0.2, 1.0, nperiods, 64, False)


def _config1_curve():
    rng = np.random.default_rng([1, 0])
    p0 = rng.uniform(0.2, 1.0)
    return kepler_curve(rng, 3e-4, dict(p0=float(p0), depth=1e-4, dur=0.03))


def config1(nperiods=200_000):
    """Kepler-shaped single curve (configs[1])."""
    return _pack("config1_kepler_single", 1, [_config1_curve()], 0.2, 1.0, nperiods,
                 256, False)


def config2(ncurves=1024, nperiods=20_000, first_curve=0):
    """Batched Kepler-shaped (configs[2]); even-indexed curves carry a box."""
    curves = []
    for c in range(first_curve, first_curve + ncurves):
        rng = np.random.default_rng([2, c])
        box = None
        if c % 2 == 0:
            p0 = rng.uniform(0.2, 1.0)
            depth = np.exp(rng.uniform(np.log(3e-5), np.log(3e-4)))
            box = dict(p0=float(p0), depth=float(depth), dur=0.03)
        curves.append(kepler_curve(rng, 3e-4, box))
    return _pack("config2_kepler_batch", 2, curves, 0.2, 1.0, nperiods, 256, False)


def config3(nperiods=2_000_000):
    """High-precision grid on config 1's curve (configs[3]); nbins = 1,024."""
    return _pack("config3_fine_grid", 3, [_config1_curve()], 0.2, 1.0, nperiods, 1024,
                 False)


def config4(ncurves=4096, nperiods=50_000, first_curve=0):
    """TESS-shaped batch (configs[4]); every 4th curve carries a box; fold and
    normalisation fused (only the normalised profile is materialised)."""
    slots = tess_slots()
    t = slots.astype(np.float64) * TESS_CADENCE_D
    curves = []
    for c in range(first_curve, first_curve + ncurves):
        rng = np.random.default_rng([4, c])
        f = 1.0 + rng.normal(0.0, 1e-3, size=t.shape[0])
        truth = None
        if c % 4 == 0:
            p0 = rng.uniform(0.2, 1.0)
            depth = np.exp(rng.uniform(np.log(2e-4), np.log(2e-3)))
            dur = rng.uniform(0.02, 0.05)
            epoch = rng.uniform(0.0, p0)
            f = f - depth * _box_mask(t, p0, dur, epoch)
            truth = dict(p0=float(p0), depth=float(depth), dur=float(dur),
                         epoch=float(epoch))
        curves.append((t.copy(), _finish(f), truth))
    return _pack("config4_tess_batch_fused", 4, curves, 0.2, 1.0, nperiods, 128, True)


def paper_fold(nperiods=100_000, n=70_000):
    """The paper's own fold workload (Table 1 :125-142): one
    Kepler-like curve of 70,000 epochs (profiled case), 100,000 trial periods uniform IN PERIOD
    over [0.2, 1.0] d (0.69 s granularity), 4096 intermediary bins merged to 256 equal-count
    bins.  nbins here is the intermediary count; bench.py merges to 256."""
    rng = np.random.default_rng([5, 0])
    nslots = int(round(n / 0.94))
    keep = np.sort(rng.choice(nslots, size=n, replace=False))
    t = keep.astype(np.float64) * KEPLER_CADENCE_D
    p0 = float(rng.uniform(0.2, 1.0))
    box = dict(p0=p0, depth=1e-4, dur=0.03)
    epoch = float(rng.uniform(0.0, p0))
    f = 1.0 + rng.normal(0.0, 3e-4, size=n)
    f = f - box["depth"] * _box_mask(t, p0, box["dur"], epoch)
    w = _pack("paper_fold_two_tier", 5, [(t, _finish(f), dict(box, epoch=epoch))], 0.2, 1.0,
              nperiods, 4096, False)
    w.grid_mode = GRID_UNIFORM_PERIOD
    return w


CONFIGS = {0: config0, 1: config1, 2: config2, 3: config3, 4: config4, 5: paper_fold}


def make(config_id: int, **kw) -> Workload:
    return CONFIGS[config_id](**kw)


def ragged_batch(seed=7, lens=(0, 1, 31, 32, 33, 1000, 4097), nbins=64, nperiods=50,
                 with_nonfinite=True):
    """Edge-case batch for parity tests: ragged and empty curves, irregular
    (non-cadence) timestamps, negative t - t0, a few non-finite samples."""
    rng = np.random.default_rng(seed)
    curves = []
    for ln in lens:
        t = np.sort(rng.uniform(-3.0, 40.0, size=ln))
        f = rng.normal(0.0, 1e-3, size=ln).astype(np.float32)
        if with_nonfinite and ln >= 31:
            t[5] = np.nan
            f[7] = np.inf
            f[11] = np.nan
            t[13] = -np.inf
        curves.append((t, f, None))
    return _pack("ragged_batch", -1, curves, 0.2, 1.0, nperiods, nbins, False)
