"""Pins for the CPU oracle (oracle/gpfc_ref.c) -- CPU only.

The oracle is checked against things other than itself: values the paper
prints (tests/golden/paper_values.json), hand-worked dyadic vectors
(tests/golden/hand_vectors.json), an exact-rational brute force, closed forms
and invariants.  Each test names the mistake it would catch.
"""
import json
import math
import os
from fractions import Fraction

import numpy as np
import pytest

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _golden(name):
    with open(os.path.join(GOLDEN, name)) as f:
        return json.load(f)


# ------------------------------------------------------------------ paper values

def test_eq1_worked_example(ref):
    """2*4*365/0.03 = 97,333 (catches a swapped T/L or dropped N_o)."""
    g = _golden("paper_values.json")["eq1_n_sample"]
    v = ref.n_sample(g["n_o"], g["T_days"], g["L_days"])
    assert int(v) == g["value_printed"]
    assert abs(v - 97333.3333333) < 1e-3


def test_period_mode_granularity_matches_paper(ref):
    """100,000 periods over [0.2, 1.0] d <-> 0.7 s granularity."""
    g = _golden("paper_values.json")["grid_granularity_s"]
    p = ref.make_period_grid(g["pmin"], g["pmax"], g["nperiods"], ref.GRID_UNIFORM_PERIOD)
    assert p.shape == (100000,)
    steps_s = np.diff(p) * 86400.0
    assert round(float(steps_s.mean()), 1) == g["value_printed_s"]
    assert np.allclose(steps_s, 0.8 * 86400 / 99999, rtol=1e-6)
    # last point: 0.2 + (1.0 - 0.2) rounds to 1 + 2^-52 (no endpoint snapping in the formula)
    assert p[0] == 0.2 and abs(p[-1] - 1.0) <= 2.0 ** -52
    assert np.all(np.diff(p) > 0)


def test_points_per_bin_and_attenuation(ref):
    """PAPER.md:105 (65536/256 = 256 points per bin) and :59-61 (1/sqrt(N))."""
    g = _golden("paper_values.json")
    n, nb = g["points_per_bin"]["n"], g["points_per_bin"]["nbins"]
    t = np.arange(n) * 0.020433
    f = np.zeros(n, np.float32)
    _, c, _ = ref.fold(t, f, [0.7131], nb)
    assert c.sum() == n and c.sum() / nb == g["points_per_bin"]["value_printed"]
    lo, hi = g["noise_attenuation"]["range_printed"]
    T = g["noise_attenuation"]["T_days"]
    att = [1 / math.sqrt(T / p) for p in g["noise_attenuation"]["p_range"]]
    assert round(att[0], 2) == lo and round(att[1], 2) == hi


# ------------------------------------------------------------------ grid

def test_frequency_grid_endpoints_order_and_uniformity(ref):
    p = ref.make_period_grid(0.2, 1.0, 2000, ref.GRID_UNIFORM_FREQUENCY)
    assert p[0] == 1.0 and p[-1] == 0.2          # ascending frequency = descending period
    assert np.all(np.diff(p) < 0)
    f = 1.0 / p
    assert np.allclose(np.diff(f), 4.0 / 1999, rtol=1e-9)
    # exclusive endpoint: divisor Np -> f_j = 1 + 4 j / 2000, so j = 500 is exactly 0.5 d
    pe = ref.make_period_grid(0.2, 1.0, 2000,
                              ref.GRID_UNIFORM_FREQUENCY | ref.GRID_ENDPOINT_EXCLUSIVE)
    assert pe[0] == 1.0 and pe[500] == 0.5 and pe[1000] == 1.0 / 3.0
    assert pe[-1] > 0.2
    # the inclusive grid does not contain 0.5 (SURVEY reading 12)
    assert not np.any(p == 0.5)


def test_grid_small_and_invalid(ref):
    assert ref.make_period_grid(0.2, 1.0, 0).shape == (0,)
    assert ref.make_period_grid(0.2, 1.0, 1, ref.GRID_UNIFORM_FREQUENCY)[0] == 1.0
    assert ref.make_period_grid(0.2, 1.0, 1, ref.GRID_UNIFORM_PERIOD)[0] == 0.2
    p2 = ref.make_period_grid(0.25, 0.5, 2)
    assert list(p2) == [0.5, 0.25]
    for bad in [(-1.0, 1.0, 4), (0.0, 1.0, 4), (1.0, 0.5, 4), (0.2, 1.0, -1)]:
        with pytest.raises(ValueError):
            ref.make_period_grid(*bad)


def test_grid_exact_rational(ref):
    """Each grid point is within 1 ulp-ish of the exact rational value (catches
    divide-before-multiply drift and an off-by-one divisor)."""
    n = 1000
    p = ref.make_period_grid(0.2, 1.0, n, ref.GRID_UNIFORM_FREQUENCY)
    fmin, fmax = Fraction(1) / Fraction(1.0), Fraction(1) / Fraction(0.2)
    for j in (0, 1, 17, 500, 998, 999):
        exact = 1 / (fmin + (fmax - fmin) * j / (n - 1))
        assert abs(Fraction(float(p[j])) - exact) <= abs(exact) * Fraction(1, 2 ** 50)
    q = ref.make_period_grid(0.2, 1.0, n, ref.GRID_UNIFORM_PERIOD)
    for j in (0, 1, 17, 500, 998, 999):
        exact = Fraction(0.2) + (Fraction(1.0) - Fraction(0.2)) * j / (n - 1)
        assert abs(Fraction(float(q[j])) - exact) <= abs(exact) * Fraction(1, 2 ** 50)


# ------------------------------------------------------------------ hand vectors

def test_hand_vectors(ref):
    g = _golden("hand_vectors.json")
    t = np.array(g["times"], np.float64)
    f = np.array(g["flux"], np.float32)
    nb = g["nbins"]
    for case in g["cases"]:
        bins = ref.bin_index(t, case["period"], nb, case["t0"])
        assert list(bins) == case["bins"], case
        s, c, s64 = ref.fold(t, f, [case["period"]], nb, case["t0"])
        assert list(c[0]) == case["count"], case
        assert list(s[0]) == case["sum"], case
        assert list(s64[0]) == case["sum"], case


def test_hand_vector_all_periods_in_one_call(ref):
    """Rows are laid out [period][bin] in the order the periods are given."""
    g = _golden("hand_vectors.json")
    t = np.array(g["times"], np.float64)
    f = np.array(g["flux"], np.float32)
    cases = [c for c in g["cases"] if c["t0"] == 0.0]
    s, c, _ = ref.fold(t, f, [k["period"] for k in cases], g["nbins"])
    for j, case in enumerate(cases):
        assert list(c[j]) == case["count"] and list(s[j]) == case["sum"]


def test_phi_rounds_to_one_goes_to_last_bin(ref):
    """t = -2^-60: x + 1 rounds to 1.0; the sample belongs to the last bin (R4)."""
    assert list(ref.bin_index([-2.0 ** -60], 1.0, 4)) == [3]
    assert list(ref.bin_index([-2.0 ** -60], 1.0, 100)) == [99]


def test_hand_normalize(ref):
    g = _golden("hand_vectors.json")["normalize"]
    out, out64 = ref.normalize(np.array([g["sum"]], np.float32),
                               np.array([g["count"]], np.uint32), want64=True)
    assert np.allclose(out64[0], g["out"], rtol=0, atol=1e-15)
    assert np.allclose(out[0], np.array(g["out"], np.float32), rtol=0, atol=0)


# ------------------------------------------------------------------ brute force

def _exact_bin(t, t0, p, nb):
    """Exact rational arithmetic: floor(frac((t - t0)/P) * nb); also the distance
    of the exact scaled phase to the nearest bin edge."""
    x = (Fraction(t) - Fraction(t0)) / Fraction(p)
    phi = x - math.floor(x)
    y = phi * nb
    k = math.floor(y)
    edge = min(y - k, k + 1 - y)
    return k, float(edge)


@pytest.mark.parametrize("nb", [4, 64, 100, 256, 1000, 4096])
def test_bins_against_exact_rational(ref, nb):
    """Brute force on small inputs with exact rationals: catches a wrong sign of
    t0, multiply-for-divide slips larger than rounding, a transposed ratio, an
    off-by-one bin.  Samples whose exact phase sits within 1e-9 of a bin edge are
    decided by fp64 rounding and are excluded (none expected)."""
    rng = np.random.default_rng(nb)
    t = np.sort(rng.uniform(-50.0, 1500.0, size=300))
    t0 = 3.25
    checked = 0
    for p in rng.uniform(0.2, 1.0, size=12):
        got = ref.bin_index(t, p, nb, t0)
        for i in range(t.shape[0]):
            k, edge = _exact_bin(float(t[i]), t0, float(p), nb)
            if edge > 1e-9:
                assert got[i] == k
                checked += 1
    assert checked > 3500


def test_fold_against_python_loop(ref):
    """Counts and sums against a dictionary-based brute force over exact bins."""
    rng = np.random.default_rng(3)
    n, nb = 500, 16
    t = np.sort(rng.uniform(0, 90, n))
    f = rng.normal(0, 1e-3, n).astype(np.float32)
    periods = rng.uniform(0.2, 1.0, 7)
    s, c, s64 = ref.fold(t, f, periods, nb)
    for j, p in enumerate(periods):
        cnt = [0] * nb
        sm = [Fraction(0)] * nb
        for i in range(n):
            k, edge = _exact_bin(float(t[i]), 0.0, float(p), nb)
            assert edge > 1e-9
            cnt[k] += 1
            sm[k] += Fraction(float(f[i]))
        assert list(c[j]) == cnt
        assert np.allclose(s64[j], [float(v) for v in sm], rtol=0, atol=1e-15)
        assert np.array_equal(s[j], s64[j].astype(np.float32))


# ------------------------------------------------------------------ invariants

def _curve(seed, n=3000, dt=0.020433):
    rng = np.random.default_rng(seed)
    keep = np.sort(rng.choice(int(n * 1.1), size=n, replace=False))
    t = keep * dt
    f = rng.normal(0, 3e-4, n).astype(np.float32)
    return t, f


def test_count_and_sum_conservation(ref):
    """Sum_k count = #valid samples; Sum_k sum = Sum_i flux (catches a dropped or
    double-counted sample, e.g. a wrong clamp)."""
    t, f = _curve(1)
    periods = ref.make_period_grid(0.2, 1.0, 200)
    for nb in (1, 7, 64, 256):
        s, c, s64 = ref.fold(t, f, periods, nb)
        assert np.all(c.sum(axis=1) == t.shape[0])
        tot = float(np.sum(f.astype(np.float64)))
        assert np.allclose(s64.sum(axis=1), tot, rtol=0,
                           atol=1e-9 * float(np.abs(f).sum()))


def test_nonfinite_samples_and_bad_periods(ref):
    t, f = _curve(2, n=400)
    t2, f2 = t.copy(), f.copy()
    t2[3] = np.nan
    t2[10] = np.inf
    f2[20] = np.nan
    f2[21] = -np.inf
    ok = np.isfinite(t2) & np.isfinite(f2)
    periods = np.array([0.3, np.nan, 0.0, -1.0, np.inf, 0.77])
    s, c, s64 = ref.fold(t2, f2, periods, 32)
    sv, cv, s64v = ref.fold(t2[ok], f2[ok], periods, 32)
    assert np.array_equal(c, cv) and np.array_equal(s64, s64v)
    assert c[0].sum() == ok.sum() == 396
    for j in (1, 2, 3, 4):
        assert not c[j].any() and not s[j].any()


def test_shift_by_whole_periods_is_invisible(ref):
    """Folding t + m P (dyadic P, dyadic t so that everything is exact) changes
    nothing (the fold is periodic in t with period P)."""
    rng = np.random.default_rng(5)
    t = rng.integers(0, 2 ** 16, 600) / 1024.0
    f = rng.normal(0, 1, 600).astype(np.float32)
    for p in (0.5, 0.625, 1.0):
        a = ref.fold(t, f, [p], 32)
        b = ref.fold(t + 37 * p, f, [p], 32)
        assert np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])
        # and t0 -> t0 + m P is the same statement
        c = ref.fold(t, f, [p], 32, t0=-5 * p)
        assert np.array_equal(a[1], c[1])


def test_permutation_invariance(ref):
    t, f = _curve(6, n=1500)
    perm = np.random.default_rng(0).permutation(t.shape[0])
    periods = [0.2, 0.31234, 0.9999]
    a = ref.fold(t, f, periods, 64)
    b = ref.fold(t[perm], f[perm], periods, 64)
    assert np.array_equal(a[1], b[1])
    assert np.allclose(a[2], b[2], rtol=0, atol=1e-12)


def test_halving_nbins_merges_adjacent_pairs(ref):
    """For power-of-two nb, bin k at nb/2 = bins 2k, 2k+1 at nb (exact scaling)."""
    t, f = _curve(7)
    periods = ref.make_period_grid(0.2, 1.0, 40)
    s1, c1, s641 = ref.fold(t, f, periods, 128)
    s2, c2, s642 = ref.fold(t, f, periods, 64)
    assert np.array_equal(c1[:, 0::2] + c1[:, 1::2], c2)
    assert np.allclose(s641[:, 0::2] + s641[:, 1::2], s642, rtol=0, atol=1e-12)


def test_collapse_closed_forms(ref):
    """Uniform dyadic cadence t_i = i dt, dt = 2^-6 (north_star's 'folding at P and
    at an exact multiple of the baseline gives the expected collapse')."""
    n, nb, dt = 1000, 16, 2.0 ** -6
    t = np.arange(n) * dt
    f = (np.arange(n) % 7).astype(np.float32)
    # P = nb dt  =>  bin = i mod nb
    bins = ref.bin_index(t, nb * dt, nb)
    assert np.array_equal(bins, np.arange(n) % nb)
    _, c, s64 = ref.fold(t, f, [nb * dt], nb)
    assert list(c[0]) == [63] * 8 + [62] * 8
    for k in range(nb):
        assert s64[0, k] == float(f[k::nb].astype(np.float64).sum())
    # P = m * (n dt): baseline (n dt = 15.625, m = 2) => only the first nb/m bins, in time order
    m = 2
    base = 1024 * dt                      # use a power-of-two baseline so bins are exact
    t2 = np.arange(1024) * dt
    f2 = np.ones(1024, np.float32)
    _, c2, _ = ref.fold(t2, f2, [m * base], nb)
    assert list(c2[0]) == [128] * 8 + [0] * 8
    bins2 = ref.bin_index(t2, m * base, nb)
    assert np.all(np.diff(bins2) >= 0)
    # P = baseline: pure time binning, 64 consecutive points per bin
    _, c3, _ = ref.fold(t2, f2, [base], nb)
    assert list(c3[0]) == [64] * 16


def test_noiseless_box_closed_form(ref):
    """Noiseless injected box (north_star): bins wholly inside the transit window
    have mean exactly -d32, bins wholly outside exactly 0, Sum_k sum = -d32 N_in;
    the deepest bin over the grid equals -d32 and is reached at P0."""
    n, dt = 20000, 0.020433
    p0, depth, dur, epoch = 0.5, 5e-4, 0.04, 0.1
    t = np.arange(n) * dt
    ph = (t - epoch + dur / 2) / p0
    intr = (ph - np.floor(ph)) < dur / p0
    flux32 = (1.0 - depth * intr).astype(np.float32)
    centred = flux32 - np.float32(1.0)
    d32 = np.float32(1.0) - np.float32(1.0 - depth)
    assert set(np.unique(centred)) == {np.float32(0.0), -d32}
    nb = 256
    s, c, s64 = ref.fold(t, centred, [p0], nb)
    assert c.sum() == n
    assert s64[0].sum() == pytest.approx(-float(d32) * intr.sum(), rel=1e-12)
    mean = s64[0] / c[0]
    lo, hi = (epoch - dur / 2) / p0, (epoch + dur / 2) / p0    # phase window [0.16, 0.24]
    edges = np.arange(nb + 1) / nb
    inside = (edges[:-1] >= lo + 1e-9) & (edges[1:] <= hi - 1e-9)
    outside = (edges[1:] <= lo - 1e-9) | (edges[:-1] >= hi + 1e-9)
    assert inside.sum() >= 18 and outside.sum() >= 230
    assert np.all(mean[inside] == -float(d32))
    assert np.all(mean[outside] == 0.0)
    # deepest bin over a grid that contains P0 exactly
    grid = ref.make_period_grid(0.2, 1.0, 2000,
                                ref.GRID_UNIFORM_FREQUENCY | ref.GRID_ENDPOINT_EXCLUSIVE)
    assert grid[500] == p0
    sg, cg, s64g = ref.fold_threaded(t, centred, grid, nb)
    with np.errstate(invalid="ignore", divide="ignore"):
        mg = np.where(cg > 0, s64g / np.maximum(cg, 1), 0.0)
    assert mg.min() == -float(d32)
    assert mg[500].min() == -float(d32)
    # half the period: dips dilute to d32/2 (every second fold misses the transit)
    j = int(np.argmin(np.abs(grid - p0 / 2)))
    assert grid[j] == 0.25
    assert mg[j].min() == pytest.approx(-float(d32) / 2, rel=0.06)


def test_sqrt_n_noise_attenuation(ref):
    """noise attenuates as sqrt(N): std of the bin means of a pure
    noise curve ~ sigma sqrt(nb / n)."""
    rng = np.random.default_rng(11)
    n, nb, sigma = 65000, 256, 3e-4
    t = np.arange(n) * 0.020433
    f = rng.normal(0, sigma, n).astype(np.float32)
    periods = rng.uniform(0.2, 1.0, 16)
    _, c, s64 = ref.fold(t, f, periods, nb)
    stds = (s64 / c).std(axis=1)
    assert np.allclose(stds.mean(), sigma * math.sqrt(nb / n), rtol=0.05)


# ------------------------------------------------------------------ normalisation

def test_normalize_invariants_and_numpy(ref):
    """Output keeps the mean and has population std 1 over non-empty bins
    (PAPER.md:63); cross-checked against numpy's mean/std."""
    rng = np.random.default_rng(12)
    nprof, nb = 50, 128
    cnt = rng.integers(0, 5, size=(nprof, nb)).astype(np.uint32)
    cnt[0] = 0                      # K = 0
    cnt[1] = 0
    cnt[1, 5] = 3                   # K = 1
    sm = (rng.normal(0, 1e-3, size=(nprof, nb)) * cnt).astype(np.float32)
    sm[2] = (cnt[2] * 0.25).astype(np.float32)      # s = 0, mu = 0.25
    out, out64 = ref.normalize(sm, cnt, want64=True)
    assert not out64[0].any()
    assert np.all(out64[1] == float(sm[1, 5]) / 3.0)
    assert np.all(out64[2] == 0.25)
    for p in range(3, nprof):
        ne = cnt[p] > 0
        m = sm[p, ne].astype(np.float64) / cnt[p, ne]
        mu, sd = m.mean(), m.std()          # numpy: ddof = 0
        assert out64[p, ne].mean() == pytest.approx(mu, abs=1e-12)
        assert out64[p, ne].std() == pytest.approx(1.0, abs=1e-12)
        assert np.allclose(out64[p, ne], mu + (m - mu) / sd, rtol=0, atol=1e-10)
        assert np.all(out64[p, ~ne] == pytest.approx(mu, abs=1e-15))
        # ddof = 1 would be off by sqrt(K/(K-1)): make sure that is NOT what we get
        assert abs(out64[p, ne].std(ddof=1) - 1.0) > 1e-3
    assert np.array_equal(out, out64.astype(np.float32))


def test_normalize_f64_matches_f32_entry(ref):
    rng = np.random.default_rng(13)
    cnt = rng.integers(1, 9, size=(4, 32)).astype(np.uint32)
    sm = rng.normal(0, 1, size=(4, 32)).astype(np.float32)
    a = ref.normalize(sm, cnt, want64=True)[1]
    b = ref.normalize_f64(sm.astype(np.float64), cnt, want64=True)[1]
    assert np.array_equal(a, b)


# ------------------------------------------------------------------ batch

def test_fold_batch_equals_per_curve(ref):
    from paper_2312_02063_b200 import workloads
    w = workloads.ragged_batch()
    periods = ref.make_period_grid(w.pmin, w.pmax, w.nperiods)
    t0 = np.linspace(-1.0, 2.0, w.ncurves)
    r = ref.fold_batch(w.times, w.flux, w.offsets, periods, w.nbins, t0=t0)
    for c in range(w.ncurves):
        lo, hi = w.offsets[c], w.offsets[c + 1]
        s, cnt, s64 = ref.fold(w.times[lo:hi], w.flux[lo:hi], periods, w.nbins, t0[c])
        assert np.array_equal(r["count"][c], cnt)
        assert np.array_equal(r["sum64"][c], s64)
        assert np.array_equal(r["sum"][c], s)
        nrm = ref.normalize_f64(s64, cnt, want64=True)[1]
        assert np.array_equal(r["norm64"][c], nrm)
    # empty curve: zero rows
    assert not r["count"][0].any() and not r["norm"][0].any()
    # t0 = NULL means 0.0
    r0 = ref.fold_batch(w.times, w.flux, w.offsets, periods, w.nbins, t0=None)
    rz = ref.fold_batch(w.times, w.flux, w.offsets, periods, w.nbins,
                        t0=np.zeros(w.ncurves))
    assert np.array_equal(r0["count"], rz["count"])


def test_config0_recovers_injected_period_statistically(ref):
    """Config 0 (noisy): the count-weighted dip statistic min_k sum/sqrt(count)
    peaks at P0 or 2 P0 (statistical check only)."""
    from paper_2312_02063_b200 import workloads
    w = workloads.config0()
    grid = ref.make_period_grid(w.pmin, w.pmax, w.nperiods,
                                w.grid_mode | ref.GRID_ENDPOINT_EXCLUSIVE)
    _, c, s64 = ref.fold_threaded(w.times, w.flux, grid, w.nbins)
    with np.errstate(invalid="ignore", divide="ignore"):
        stat = np.where(c > 0, s64 / np.sqrt(np.maximum(c, 1)), 0.0).min(axis=1)
    best = grid[int(np.argmin(stat))]
    assert min(abs(best - 0.5), abs(best - 1.0)) < 2e-3


def test_overflowing_quotient_skips_the_sample(ref):
    """R20: a positive period so small that (t - t0) / P overflows gives the sample no phase;
    it is skipped (only t == t0, whose quotient is exactly 0, lands in bin 0)."""
    t = np.array([0.0, 1.0, 2.0, -3.0])
    f = np.array([1.0, 2.0, 4.0, 8.0], np.float32)
    per = np.array([1e-320, 0.5])
    s, c, s64 = ref.fold(t, f, per, 4)
    assert c[0].tolist() == [1, 0, 0, 0] and s64[0].tolist() == [1.0, 0, 0, 0]
    assert c[1].sum() == 4
    assert ref.bin_index(t, 1e-320, 4).tolist() == [0, -1, -1, -1]
