"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(-m gpu).  The whole output is produced by one gpfc_fold_batch call per config; the oracle
checks a sample of (curve, period) rows one by one (all periods of a few curves, random and
cadence-commensurate periods of many curves), and properties that hold at any size are checked
on every row on the device (torch is plumbing here): counts of a row sum to the number of
valid samples, sums of a row sum to the curve's total flux, normalised rows have the mean of
the bin means and unit population std.
"""
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

from paper_2312_02063_b200 import workloads

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def gp():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2312_02063_b200 import binding
    binding.lib()
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def oracle_rows(ref, w, periods, pairs):
    """pairs: dict curve -> sorted array of period indices.  Returns dict curve -> oracle dict."""
    tasks = []
    threads = os.cpu_count() or 1
    for c, idx in pairs.items():
        nsplit = max(1, min(len(idx) // 64, threads))       # short lists: one task per curve
        for part in np.array_split(np.asarray(idx), nsplit):
            if len(part):
                tasks.append((c, part))
    out = {c: {} for c in pairs}

    def work(task):
        c, part = task
        a, b = int(w.offsets[c]), int(w.offsets[c + 1])
        r = ref.fold_batch(w.times[a:b], w.flux[a:b], np.array([0, b - a], np.int64), periods[part],
                           w.nbins)
        return c, part, r

    with ThreadPoolExecutor(max_workers=threads) as ex:
        for c, part, r in ex.map(work, tasks):
            out[c][tuple(part)] = r
    return out


def compare_rows(g_sum, g_cnt, g_norm, c, part, r, exact_sums=True):
    idx = torch.as_tensor(np.asarray(part), device="cuda")
    if g_cnt is not None:
        gc = g_cnt[c].index_select(0, idx).cpu().numpy().view(np.uint32)
        assert np.array_equal(gc, r["count"][0]), "counts differ (curve %d)" % c
    if g_sum is not None:
        gs = g_sum[c].index_select(0, idx).cpu().numpy()
        cnt = np.maximum(r["count"][0], 1).astype(np.float64)
        assert np.max(np.abs(gs.astype(np.float64) / cnt - r["sum64"][0] / cnt)) <= 1e-6
        if exact_sums:
            assert np.array_equal(gs, r["sum"][0]), "fp32 sums differ on lattice input"
    if g_norm is not None:
        gn = g_norm[c].index_select(0, idx).cpu().numpy().astype(np.float64)
        ref64 = r["norm64"][0]
        err = np.abs(gn - ref64)
        tol = 1e-4 * np.maximum(1.0, np.abs(ref64))
        assert np.all(err <= tol), "normalised row off by %g x tol (curve %d)" % ((err / tol).max(), c)


def degenerate_indices(periods, dt, ks=(10, 12, 15, 16, 20, 24, 25, 30, 32, 40, 45, 48)):
    """Grid periods nearest to k * cadence: thousands of samples in a few bins, empty bins."""
    return sorted({int(np.argmin(np.abs(periods - k * dt))) for k in ks
                   if periods.min() <= k * dt <= periods.max()})


def device_invariants(w, g_sum, g_cnt, g_norm, nvalid, flux_tot):
    """Properties of every row, checked on the device."""
    nv = torch.as_tensor(nvalid, device="cuda").view(-1, 1)
    if g_cnt is not None:
        rows = g_cnt.sum(dim=2, dtype=torch.int64)
        assert bool((rows == nv).all()), "a row's counts do not sum to the number of samples"
    if g_sum is not None:
        ft = torch.as_tensor(flux_tot, device="cuda").view(-1, 1)
        rows = g_sum.sum(dim=2, dtype=torch.float64)
        assert float((rows - ft).abs().max()) <= 1e-6
    if g_norm is not None:
        chunk = max(1, (1 << 28) // (g_norm.shape[1] * g_norm.shape[2]))
        for c0 in range(0, g_norm.shape[0], chunk):
            x = g_norm[c0:c0 + chunk].double()
            if g_cnt is not None:
                ne = g_cnt[c0:c0 + chunk] > 0
                k = ne.sum(dim=2).clamp(min=1)
                mu = (x * ne).sum(dim=2) / k
                var = (((x - mu.unsqueeze(2)) ** 2) * ne).sum(dim=2) / k
                assert float((var - 1.0).abs().max()) <= 1e-4, "normalised rows: std != 1"
            else:
                # fused path: every bin non-empty for these shapes except degenerate rows;
                # empty bins hold mu, which leaves the mean unchanged and lowers the variance
                var = x.var(dim=2, unbiased=False)
                assert float(var.max()) <= 1.0 + 1e-4 and float(var.median()) >= 1.0 - 1e-4
            assert bool(torch.isfinite(x).all())


def totals(w):
    nvalid = np.diff(w.offsets)
    flux_tot = np.array([w.flux[a:b].astype(np.float64).sum()
                         for a, b in zip(w.offsets[:-1], w.offsets[1:])])
    return nvalid, flux_tot


def run_full(gp, w, want):
    torch.cuda.empty_cache()
    periods_d = gp.gpfc_make_period_grid(w.pmin, w.pmax, w.nperiods, w.grid_mode)
    s, c, nrm = gp.gpfc_fold_batch(dev(w.times), dev(w.flux), dev(w.offsets), periods_d, w.nbins,
                                   want=want)
    torch.cuda.synchronize()
    return periods_d.cpu().numpy(), s, c, nrm


def test_config1_full_all_rows(gp, ref):
    """65,000 samples x 200,000 periods: every row against the oracle."""
    w = workloads.config1()
    periods, s, c, nrm = run_full(gp, w, ("sum", "count", "norm"))
    assert np.array_equal(periods, ref.make_period_grid(w.pmin, w.pmax, w.nperiods, w.grid_mode))
    device_invariants(w, s, c, nrm, *totals(w))
    rows = oracle_rows(ref, w, periods, {0: np.arange(w.nperiods)})
    for part, r in rows[0].items():
        compare_rows(s, c, nrm, 0, part, r)


def test_config2_full_sampled(gp, ref):
    """1,024 curves x 20,000 periods (bench.py's launch): all periods of 2 curves, and for EVERY
    curve a fixed set of periods (the cadence-commensurate ones + 8 fixed random ones, >= 16 in
    all), plus 48 random periods of every 8th curve."""
    w = workloads.config2()
    periods, s, c, nrm = run_full(gp, w, ("sum", "count", "norm"))
    device_invariants(w, s, c, nrm, *totals(w))
    rng = np.random.default_rng(123)
    deg = degenerate_indices(periods, workloads.KEPLER_CADENCE_D)
    assert len(deg) >= 8
    fixed = sorted(set(deg) | set(rng.integers(0, w.nperiods, 8).tolist()) | {0, w.nperiods - 1})
    assert len(fixed) >= 16
    pairs = {cu: np.array(fixed) for cu in range(w.ncurves)}
    pairs[0] = pairs[1023] = np.arange(w.nperiods)
    for cu in range(5, w.ncurves, 8):
        pairs[cu] = np.array(sorted(set(rng.integers(0, w.nperiods, 48).tolist()) | set(fixed)))
    rows = oracle_rows(ref, w, periods, pairs)
    for cu, parts in rows.items():
        for part, r in parts.items():
            compare_rows(s, c, nrm, cu, part, r)


def test_config3_full_sampled(gp, ref):
    """65,000 samples x 2,000,000 periods, nbins = 1,024: 6,000 random rows + degenerate ones."""
    w = workloads.config3()
    periods, s, c, _ = run_full(gp, w, ("sum", "count"))
    device_invariants(w, s, c, None, *totals(w))
    rng = np.random.default_rng(321)
    deg = degenerate_indices(periods, workloads.KEPLER_CADENCE_D)
    idx = np.array(sorted(set(rng.integers(0, w.nperiods, 6000).tolist()) | set(deg)
                          | {0, w.nperiods - 1}))
    rows = oracle_rows(ref, w, periods, {0: idx})
    for part, r in rows[0].items():
        compare_rows(s, c, None, 0, part, r)


def test_config4_full_fused_sampled(gp, ref):
    """4,096 curves x 50,000 periods, nbins = 128, fold + normalise fused (only the
    normalised profile is materialised: 105 GB)."""
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    w = workloads.config4()
    need = w.ncurves * w.nperiods * w.nbins * 4 + (3 << 30)
    if free < need:
        pytest.skip("needs %.0f GB of free HBM" % (need / 1e9))
    periods, s, c, nrm = run_full(gp, w, ("norm",))
    assert s is None and c is None
    device_invariants(w, None, None, nrm, *totals(w))
    rng = np.random.default_rng(77)
    deg = degenerate_indices(periods, workloads.TESS_CADENCE_D, ks=(144, 180, 200, 240, 288, 360, 400,
                                                                   480, 500, 600, 700, 720))
    fixed = sorted(set(deg) | set(rng.integers(0, w.nperiods, 8).tolist()) | {0, w.nperiods - 1})
    assert len(fixed) >= 16
    pairs = {cu: np.array(fixed) for cu in range(w.ncurves)}          # every curve
    pairs[0], pairs[4095] = np.arange(0, w.nperiods, 25), np.arange(7, w.nperiods, 25)
    for cu in range(3, w.ncurves, 16):
        pairs[cu] = np.array(sorted(set(rng.integers(0, w.nperiods, 40).tolist()) | set(fixed)))
    rows = oracle_rows(ref, w, periods, pairs)
    for cu, parts in rows.items():
        for part, r in parts.items():
            compare_rows(None, None, nrm, cu, part, r)


def oracle_two_tier_rows(ref, w, periods, nb1, nb2):
    """fp64 fold at nb1 bins + gpfc_ref_two_tier_merge + normalisation of the merged means."""
    threads = os.cpu_count() or 1
    s32, cnt, s64 = ref.fold_threaded(w.times, w.flux, periods, nb1, threads=threads)
    _, omean = ref.two_tier_merge(s64, cnt, nb2)
    ones = np.ones((len(periods), nb2), np.uint32)
    onorm = ref.normalize_f64(omean, ones, want64=True)[1]
    return s32, cnt, omean, onorm


def check_two_tier_sample(gp, ref, w, periods_all, mean_d, norm_d, idx, nb1=4096, nb2=256):
    idx = np.asarray(idx)
    per = periods_all[idx]
    s32, cnt, omean, onorm = oracle_two_tier_rows(ref, w, per, nb1, nb2)
    ti = torch.as_tensor(idx, device="cuda")
    gm = mean_d[0].index_select(0, ti).cpu().numpy().astype(np.float64)
    gn = norm_d[0].index_select(0, ti).cpu().numpy().astype(np.float64)
    assert np.all(np.abs(gm - omean) <= 1e-6), np.abs(gm - omean).max()      # north_star: bin means
    scale = np.maximum(np.abs(omean).max(axis=-1, keepdims=True), 1e-30)
    assert np.all(np.abs(gm - omean) <= 2e-7 * scale + 1e-12)                # lattice input: fp32 rounding only
    defined = omean.std(axis=-1) >= 1e-11 * np.abs(omean).max(axis=-1)       # bound: test_gpu_two_tier.py
    err, tol = np.abs(gn - onorm), 1e-4 * np.maximum(1.0, np.abs(onorm))
    assert np.all(err[defined] <= tol[defined]), float((err[defined] / tol[defined]).max())
    # tier 1 itself, bit for bit, through the same kernel's bin epilogue
    s, c = gp.gpfc_fold(dev(w.times), dev(w.flux), dev(per), nb1)
    torch.cuda.synchronize()
    assert np.array_equal(c.cpu().numpy().view(np.uint32), cnt), "tier-1 counts differ"
    assert np.array_equal(s.cpu().numpy(), s32), "tier-1 sums differ"
    return int(defined.sum())


def test_config5_paper_fold_full_sampled(gp, ref):
    """The paper's own workload at full scale (Table 1): 70,000
    epochs x 100,000 periods uniform IN PERIOD over [0.2, 1.0] d, 4096 intermediary -> 256
    equal-count bins, in bench.py --config 5's launch (gpfc_fold_two_tier, one kernel).  The
    oracle recomputes 2,048 random rows + every cadence-commensurate period + both ends: merged
    means, normalised profile, and tier 1 bit for bit."""
    w = workloads.paper_fold()
    assert w.n_total == 70000 and w.nperiods == 100000
    periods_d = gp.gpfc_make_period_grid(w.pmin, w.pmax, w.nperiods, w.grid_mode)
    gp.gpfc_profile(True)
    mean, norm = gp.gpfc_fold_two_tier(dev(w.times), dev(w.flux), dev(w.offsets), periods_d, 4096, 256)
    torch.cuda.synchronize()
    counters = gp.gpfc_path_counters()
    gp.gpfc_profile(False)
    assert counters["unfused_two_tier_calls"] == 0 and counters["generic_kernel_calls"] == 0
    assert counters["exact_path_items"] == 0
    periods = periods_d.cpu().numpy()
    assert np.array_equal(periods, ref.make_period_grid(0.2, 1.0, 100000, workloads.GRID_UNIFORM_PERIOD))
    # 0.7 s granularity
    assert abs((periods[1] - periods[0]) * 86400.0 - 0.6912) < 1e-3
    rng = np.random.default_rng(2312)
    deg = degenerate_indices(periods, workloads.KEPLER_CADENCE_D,
                             ks=tuple(range(10, 49)))
    idx = sorted(set(rng.integers(0, w.nperiods, 2048).tolist()) | set(deg) | {0, w.nperiods - 1})
    assert len(idx) >= 2000 and len(deg) >= 30
    ncmp = check_two_tier_sample(gp, ref, w, periods, mean, norm, idx)
    assert ncmp >= len(idx) - len(deg)
    # every row on the device: finite, mean of the normalised row = mean of the merged means,
    # population std 1 (every final bin holds N/256 points, none is empty)
    m, x = mean[0].double(), norm[0].double()
    assert bool(torch.isfinite(x).all()) and bool(torch.isfinite(m).all())
    assert float((x.mean(dim=1) - m.mean(dim=1)).abs().max()) <= 1e-6
    var = x.var(dim=1, unbiased=False)
    flat = m.std(dim=1, unbiased=False) <= 1e-11 * m.abs().amax(dim=1).clamp(min=1e-30)
    assert float((var[~flat] - 1.0).abs().max()) <= 1e-4
    # equal-count property: the merged means average to the curve's mean flux
    assert float((m.mean(dim=1) - float(w.flux.astype(np.float64).mean())).abs().max()) <= 1e-9


def test_wider_period_range_1_to_10_days(gp, ref):
    """the method carries over to longer periods.  20,000 periods uniform in
    period over [1, 10] d on the 70,000-epoch curve: the two-tier fold and the plain 256-bin
    fold against the oracle on sampled rows (longer periods: fewer cycles, smaller rp, the
    guard band shrinks; nothing takes the exact path)."""
    w = workloads.paper_fold(nperiods=20000)
    periods_d = gp.gpfc_make_period_grid(1.0, 10.0, 20000, workloads.GRID_UNIFORM_PERIOD)
    periods = periods_d.cpu().numpy()
    assert np.array_equal(periods, ref.make_period_grid(1.0, 10.0, 20000, workloads.GRID_UNIFORM_PERIOD))
    gp.gpfc_profile(True)
    mean, norm = gp.gpfc_fold_two_tier(dev(w.times), dev(w.flux), dev(w.offsets), periods_d, 4096, 256)
    s, c, nrm = gp.gpfc_fold_batch(dev(w.times), dev(w.flux), dev(w.offsets), periods_d, 256)
    torch.cuda.synchronize()
    counters = gp.gpfc_path_counters()
    gp.gpfc_profile(False)
    assert counters["exact_path_items"] == 0 and counters["unfused_two_tier_calls"] == 0
    rng = np.random.default_rng(356)
    dt = workloads.KEPLER_CADENCE_D
    deg = sorted({int(np.argmin(np.abs(periods - k * dt))) for k in (49, 50, 60, 64, 75, 100, 128, 200, 256, 400)})
    idx = sorted(set(rng.integers(0, 20000, 500).tolist()) | set(deg) | {0, 19999})
    check_two_tier_sample(gp, ref, w, periods, mean, norm, idx)
    w256 = workloads.Workload(**{**w.__dict__, "nbins": 256})
    rows = oracle_rows(ref, w256, periods, {0: np.array(idx)})
    for part, r in rows[0].items():
        compare_rows(s, c, nrm, 0, part, r)
    device_invariants(w256, s, c, nrm, *totals(w256))
