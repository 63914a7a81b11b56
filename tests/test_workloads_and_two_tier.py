"""CPU tests: the synthetic input recipe and the NEXT-row two-tier
merge of the oracle (PAPER.md:105, :111 'Fourthly')."""
import numpy as np
import pytest

from paper_2312_02063_b200 import workloads


def test_config_shapes():
    w0 = workloads.config0()
    assert (w0.ncurves, w0.n_total, w0.nperiods, w0.nbins) == (1, 4000, 2000, 64)
    assert w0.point_periods == 8_000_000
    assert w0.times[0] == 0.0 and w0.times[1] == 0.020433
    assert w0.flux.dtype == np.float32 and w0.times.dtype == np.float64
    assert abs(float(np.median(w0.flux))) < 1e-7
    w1 = workloads.config1()
    assert (w1.n_total, w1.nperiods, w1.nbins) == (65000, 200000, 256)
    assert w1.point_periods == 13_000_000_000
    assert w1.times[-1] < 1413.1 and np.all(np.diff(w1.times) > 0)
    gaps = np.diff(w1.times) / workloads.KEPLER_CADENCE_D
    assert (gaps > 200).sum() >= 3                      # the three 5-day gaps
    # fp32 flux near 1.0 minus an fp32 median: multiples of 2^-24 (lossless fixed point)
    assert np.all(np.mod(w1.flux.astype(np.float64) * 2.0 ** 24, 1.0) == 0.0)
    assert 2.5e-4 < float(w1.flux.std()) < 3.5e-4
    w3 = workloads.config3(nperiods=10)
    assert np.array_equal(w3.times, w1.times) and w3.nbins == 1024


def test_batch_configs_scaled():
    w2 = workloads.config2(ncurves=4, nperiods=100)
    assert w2.ncurves == 4 and list(w2.offsets) == [0, 65000, 130000, 195000, 260000]
    assert [t is not None for t in w2.truth] == [True, False, True, False]
    assert 3e-5 <= w2.truth[0]["depth"] <= 3e-4
    again = workloads.config2(ncurves=2, nperiods=100, first_curve=2)
    assert np.array_equal(again.flux[:65000], w2.flux[130000:195000])   # per-curve seeds
    w4 = workloads.config4(ncurves=8, nperiods=10)
    assert w4.n_total == 8 * 19440 and w4.nbins == 128 and w4.fused_normalize
    assert [t is not None for t in w4.truth] == [True, False, False, False] * 2
    t = w4.times[:19440]
    assert t[-1] < 28.0 and np.max(np.diff(t)) == pytest.approx(721 * 0.0013889)


def test_ragged_batch_has_edge_cases():
    w = workloads.ragged_batch()
    assert w.ncurves == 7 and w.offsets[1] == 0
    assert np.isnan(w.times).sum() > 0 and np.isinf(w.flux).sum() > 0


# ------------------------------------------------------------------ two-tier merge (NEXT)

def test_two_tier_conservation_and_equal_count(ref):
    rng = np.random.default_rng(0)
    n = 5000
    t = np.sort(rng.uniform(0, 300, n))
    f = rng.normal(0, 1e-3, n).astype(np.float32)
    periods = [0.2, 0.37, 0.99]
    _, c, s64 = ref.fold(t, f, periods, 4096)
    osum, omean = ref.two_tier_merge(s64, c, 256)
    assert osum.shape == (3, 256)
    assert np.allclose(osum.sum(axis=1), s64.sum(axis=1), rtol=0, atol=1e-12)
    assert np.allclose(omean * (n / 256), osum, rtol=1e-12, atol=0)


def test_two_tier_exact_when_counts_divide(ref):
    """When every group of nb1/nb2 fine bins already holds N/nb2 points no bin is
    split, and the merge is plain pairwise addition."""
    c = np.full((1, 16), 3, np.uint32)
    s = np.arange(16, dtype=np.float64)[None, :]
    osum, omean = ref.two_tier_merge(s, c, 4)
    assert list(osum[0]) == [0 + 1 + 2 + 3, 4 + 5 + 6 + 7, 8 + 9 + 10 + 11, 12 + 13 + 14 + 15]
    assert list(omean[0]) == [v / 12 for v in osum[0]]


def test_two_tier_split_is_pro_rata(ref):
    """One fine bin of 4 points, flux sum 8, split over 2 output bins: 2 points and
    half the flux each (reading R18)."""
    osum, omean = ref.two_tier_merge(np.array([[8.0, 0.0]]), np.array([[4, 0]], np.uint32), 2)
    assert list(osum[0]) == [4.0, 4.0] and list(omean[0]) == [2.0, 2.0]
    osum, _ = ref.two_tier_merge(np.array([[3.0, 9.0, 0.0]]),
                                 np.array([[1, 3, 0]], np.uint32), 2)
    assert list(osum[0]) == [3.0 + 3.0, 6.0]


def test_two_tier_close_to_sort_based_fold(ref):
    """the two-tier result is a 'near-equivalent' of the sort-based
    fold (sort by residual, split equally).  On tie-free random times the two
    agree closely (correlation > 0.95); this pins the scan direction and the
    equal-count targets, not the split values."""
    rng = np.random.default_rng(1)
    n, nb2 = 65536, 256
    t = np.sort(rng.uniform(0, 1400, n))
    sig = -5e-3 * ((t / 0.61803) % 1.0 < 0.05)
    f = (rng.normal(0, 1e-3, n) + sig).astype(np.float32)
    p = 0.61803
    _, c, s64 = ref.fold(t, f, [p], 4096)
    _, omean = ref.two_tier_merge(s64, c, nb2)
    order = np.argsort((t / p) % 1.0, kind="stable")
    sort_mean = f[order].astype(np.float64).reshape(nb2, n // nb2).mean(axis=1)
    r = np.corrcoef(omean[0], sort_mean)[0, 1]
    assert r > 0.95
    assert int(np.argmin(omean[0])) in range(0, 14)
