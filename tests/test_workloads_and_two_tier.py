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

def _interp_merge(s64, c, nb2):
    """R18 in a different formulation from the oracle's left-to-right scan: the cumulative flux
    is piecewise linear in cumulative count (knots after every non-empty fine bin); output bin b
    is the difference of that function at b N/nb2 and (b + 1) N/nb2."""
    ne = c > 0
    xc = np.concatenate([[0.0], np.cumsum(c[ne].astype(np.float64))])
    xs = np.concatenate([[0.0], np.cumsum(s64[ne])])
    n = xc[-1]
    edges = np.arange(nb2 + 1, dtype=np.float64) * (n / nb2)
    edges[-1] = n
    return np.diff(np.interp(edges, xc, xs))


def test_two_tier_hand_vectors_fractional_split(ref):
    """tests/golden/hand_vectors.json 'two_tier_merge': N/nb2 is fractional, fine bins are cut
    by one and by three boundaries, empty fine bins sit between populated ones.  An oracle that
    rounded its targets to whole points, split by bin width instead of by count, or scanned
    right to left fails these."""
    import json
    import os
    g = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "hand_vectors.json")))
    for case in g["two_tier_merge"]["cases"]:
        osum, omean = ref.two_tier_merge(np.array([case["sum"]], np.float64),
                                         np.array([case["count"]], np.uint32), case["nb2"])
        assert list(osum[0]) == case["out_sum"], case["_work"]
        assert list(omean[0]) == case["out_mean"], case["_work"]


def test_two_tier_paper_example_256_points_per_bin(ref):
    """'given a light curve comprising 65,536 data points, each of the 256 bins
    will accommodate 65536/256 = 256 data points'.  Folding unit flux makes out_sum[b] the
    number of points of output bin b: exactly 256 everywhere, whatever the period."""
    n = 65536
    t = np.arange(n, dtype=np.float64) * 0.0204
    f = np.ones(n, np.float32)
    periods = [0.2, 0.6852, 1.0, 12 * 0.0204]            # the last: cadence-commensurate, sparse
    _, c, s64 = ref.fold(t, f, periods, 4096)
    assert (c[3] == 0).sum() > 4000                      # nearly all fine bins empty there
    osum, omean = ref.two_tier_merge(s64, c, 256)
    assert np.allclose(osum, 256.0, rtol=0, atol=1e-9)
    assert np.allclose(omean, 1.0, rtol=0, atol=1e-12)


def test_two_tier_conservation_and_interp_formulation(ref):
    rng = np.random.default_rng(0)
    n = 5000                                             # 5000 / 256 is fractional
    t = np.sort(rng.uniform(0, 300, n))
    f = rng.normal(0, 1e-3, n).astype(np.float32)
    periods = [0.2, 0.37, 0.99]
    _, c, s64 = ref.fold(t, f, periods, 4096)
    osum, omean = ref.two_tier_merge(s64, c, 256)
    assert osum.shape == (3, 256)
    assert np.allclose(osum.sum(axis=1), s64.sum(axis=1), rtol=0, atol=1e-12)
    for j in range(3):
        want = _interp_merge(s64[j], c[j], 256)
        assert np.allclose(osum[j], want, rtol=0, atol=1e-15 + 1e-12 * np.abs(want).max())
        assert np.allclose(omean[j], want / (n / 256), rtol=0, atol=1e-14)
    # ragged bin counts, nb1 not a multiple of nb2, more output than input bins
    for nb1, nb2 in [(37, 5), (8, 12), (100, 7)]:
        cc = rng.integers(0, 9, nb1).astype(np.uint32)
        cc[rng.integers(0, nb1, nb1 // 3)] = 0
        ss = rng.normal(0, 1, nb1) * (cc > 0)
        osum, _ = ref.two_tier_merge(ss[None, :], cc[None, :], nb2)
        assert np.allclose(osum[0], _interp_merge(ss, cc, nb2), rtol=0, atol=1e-12)


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
