"""NEXT row, -m gpu: the paper's step 4 -- equal-count merge of the
intermediary bins (PAPER.md:105, :111 'Fourthly') -- gpfc_merge_equal_count against the oracle's
gpfc_ref_two_tier_merge on the same folded profiles.  Counts and sums fed to both sides are the
(bit-identical) outputs of the fold; the merged means are fp64 on both sides, compared at fp32
resolution.  The pro-rata split itself is reading R18 (pinned on the oracle side by hand-worked
fractional merges, tests/test_workloads_and_two_tier.py)."""
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


def check_merge(gp, ref, s32, cnt, nb2):
    mean, norm = gp.gpfc_merge_equal_count(dev(s32), dev(cnt.view(np.int32)), nb2)
    torch.cuda.synchronize()
    mean, norm = mean.cpu().numpy(), norm.cpu().numpy()
    osum, omean = ref.two_tier_merge(s32.astype(np.float64), cnt, nb2)
    scale = np.maximum(np.abs(omean).max(axis=-1, keepdims=True), 1e-30)
    assert np.all(np.abs(mean - omean) <= 2e-7 * scale + 1e-12), np.abs(mean - omean).max()
    # normalised: every final bin non-empty (count 1), profiles without points stay zero; both
    # sides normalise their fp64 merged means
    has = cnt.reshape(-1, cnt.shape[-1]).sum(axis=-1) > 0
    on = ref.normalize_f64(omean.reshape(-1, nb2),
                           np.where(has[:, None], 1, 0).astype(np.uint32) * np.ones((1, nb2), np.uint32),
                           want64=True)[1]
    err = np.abs(norm.reshape(-1, nb2) - on)
    tol = 1e-4 * np.maximum(1.0, np.abs(on))
    # Every row is compared, except profiles whose spread is at the rounding level of their
    # own means.  Bound: either side's merged means carry a relative rounding error of a few
    # ulp (<= 4 eps each, eps = 2^-53), so two correct evaluations differ by delta <= 8 eps mag,
    # and (m - mu)/s turns that into 8 eps mag / s: above the 1e-4 tolerance only when
    # s < 8 eps mag / 1e-4 ~ 1e-11 mag.  Such rows (none in the folded-curve tests, asserted
    # there; here: equal means whose spread is one rounding) have no defined scale -- dividing
    # rounding noise by its own std gives O(1) numbers on either side -- so only finiteness
    # is required of them.
    sd = omean.reshape(-1, nb2).std(axis=-1)
    mag = np.abs(omean.reshape(-1, nb2)).max(axis=-1)
    ok_rows = (sd >= 1e-11 * mag) | (sd == 0)
    assert np.all(err[ok_rows] <= tol[ok_rows]), float((err[ok_rows] / tol[ok_rows]).max())
    assert np.all(np.isfinite(norm))
    return mean, omean, int(ok_rows.sum())


def test_merge_hand_cases(gp, ref):
    # counts divide evenly: 8 fine bins of 2 points -> 4 bins of 4 points: plain pair sums
    s = np.array([[1, 2, 3, 4, 5, 6, 7, 8]], np.float32)
    c = np.full((1, 8), 2, np.uint32)
    mean, _, _ = check_merge(gp, ref, s, c, 4)
    assert np.allclose(mean[0], [3 / 4, 7 / 4, 11 / 4, 15 / 4])
    # everything in one fine bin: every final bin gets that bin's mean
    s = np.array([[0, 0, 12, 0]], np.float32)
    c = np.array([[0, 0, 6, 0]], np.uint32)
    mean, _, _ = check_merge(gp, ref, s, c, 3)
    assert np.allclose(mean[0], [2, 2, 2])
    # no points -> zeros; nb1 < nb2 (every fine bin split); nb1 not a multiple of 32
    s = np.zeros((1, 16), np.float32)
    c = np.zeros((1, 16), np.uint32)
    mean, _, _ = check_merge(gp, ref, s, c, 8)
    assert not mean.any()
    rng = np.random.default_rng(3)
    for nb1, nb2 in [(4, 8), (37, 5), (100, 100), (4096, 256), (4096, 4096), (1, 7)]:
        c = rng.integers(0, 50, (6, nb1)).astype(np.uint32)
        c[2, : nb1 // 2] = 0
        s = (rng.integers(-1000, 1000, (6, nb1)) * c).astype(np.float32) * np.float32(2.0 ** -10)
        check_merge(gp, ref, s, c, nb2)


def test_merge_of_folded_kepler_profiles(gp, ref):
    """Config-1 curve folded at 4096 intermediary bins (the paper's tier 1) over ordinary and
    cadence-commensurate periods, merged to 256 equal-count bins (the paper's tier 2)."""
    w = workloads.config1(nperiods=48)
    grid = ref.make_period_grid(w.pmin, w.pmax, 100000, workloads.GRID_UNIFORM_PERIOD)
    dt = workloads.KEPLER_CADENCE_D
    periods = np.concatenate([grid[np.linspace(0, 99999, 40).astype(int)],
                              [10 * dt, 16 * dt, 20 * dt, 25 * dt, 32 * dt, 0.5, 0.25, 1.0]])
    s, c = gp.gpfc_fold(dev(w.times), dev(w.flux), dev(periods), 4096)
    torch.cuda.synchronize()
    s, c = s.cpu().numpy(), c.cpu().numpy().view(np.uint32)
    rs, rc, _ = ref.fold(w.times, w.flux, periods, 4096)
    assert np.array_equal(c, rc) and np.array_equal(s, rs)
    mean, omean, ncmp = check_merge(gp, ref, s, c, 256)
    assert ncmp == len(periods)                          # every folded profile was compared
    # equal-count property: the merged means average to the curve's mean flux
    assert np.allclose(mean.mean(axis=1), w.flux.astype(np.float64).mean(), atol=1e-9)


# ------------------------------------------------------------------ fused fold + merge

def oracle_two_tier(ref, times, flux, periods, nb1, nb2, t0=0.0):
    """The oracle's own path: fp64 fold at nb1 bins, then gpfc_ref_two_tier_merge, then the
    normalisation of the merged means (every final bin non-empty unless the profile is empty)."""
    _, c, s64 = ref.fold(times, flux, periods, nb1, t0=t0)
    _, omean = ref.two_tier_merge(s64, c, nb2)
    has = c.sum(axis=-1) > 0
    cnt1 = np.where(has[:, None], 1, 0).astype(np.uint32) * np.ones((1, nb2), np.uint32)
    onorm = ref.normalize_f64(omean, cnt1, want64=True)[1]
    return omean, onorm, has


def check_fused(gp, ref, times, flux, periods, nb1, nb2, t0=None, offsets=None, lattice=True):
    off = np.array([0, len(times)], np.int64) if offsets is None else offsets
    t0d = None if t0 is None else dev(np.asarray(t0, np.float64))
    mean, norm = gp.gpfc_fold_two_tier(dev(times), dev(flux), dev(off), dev(periods), nb1, nb2, t0=t0d)
    torch.cuda.synchronize()
    mean, norm = mean.cpu().numpy(), norm.cpu().numpy()
    for c in range(len(off) - 1):
        a, b = int(off[c]), int(off[c + 1])
        omean, onorm, has = oracle_two_tier(ref, times[a:b], flux[a:b], periods, nb1, nb2,
                                            0.0 if t0 is None else float(t0[c]))
        # north_star: bin means within 1e-6 absolute (observed: fp32 rounding of the output)
        assert np.all(np.abs(mean[c] - omean) <= 1e-6), np.abs(mean[c] - omean).max()
        if lattice:
            # flux on the curve's fixed-point lattice: the sums are exact, what is
            # left is the fp32 rounding of the output
            scale = np.maximum(np.abs(omean).max(axis=-1, keepdims=True), 1e-30)
            assert np.all(np.abs(mean[c] - omean) <= 2e-7 * scale + 1e-12)
        tol = 1e-4 * np.maximum(1.0, np.abs(onorm))
        err = np.abs(norm[c] - onorm)
        # a profile whose spread is the rounding noise of equal means has no defined scale
        # (bound as in check_merge: below 1e-11 of the magnitude the 1e-4 bar cannot hold for
        # two correct evaluation orders; happens when every point sits in one intermediary bin)
        sd = omean.std(axis=-1)
        defined = sd >= 1e-11 * np.abs(omean).max(axis=-1)
        assert np.all(err[defined] <= tol[defined]), float((err[defined] / tol[defined]).max())
        assert np.all(norm[c][~has] == 0) and np.all(mean[c][~has] == 0)
    return mean, norm


@pytest.mark.parametrize("nb1,nb2", [(4096, 256), (2048, 128), (1024, 64), (4096, 200), (4096, 1),
                                     (2048, 100), (1024, 33)])
def test_fused_two_tier_matches_oracle(gp, ref, nb1, nb2):
    """gpfc_fold_two_tier (one kernel: fold at nb1 rows, equal-count merge from the exact sums
    in shared memory) against fold + gpfc_ref_two_tier_merge + normalise of the oracle:
    ordinary, cadence-commensurate (sparse), invalid and tiny periods."""
    w = workloads.config1(nperiods=8)
    grid = ref.make_period_grid(w.pmin, w.pmax, 100000, workloads.GRID_UNIFORM_PERIOD)
    dt = workloads.KEPLER_CADENCE_D
    periods = np.concatenate([grid[np.linspace(0, 99999, 37).astype(int)],
                              [10 * dt, 16 * dt, 20 * dt, 25 * dt, 32 * dt, 0.5, 0.25, 1.0, dt,
                               np.nan, -1.0, 3.0, 1e-3]])
    check_fused(gp, ref, w.times, w.flux, periods, nb1, nb2)
    c = gp.gpfc_path_counters()
    assert c["unfused_two_tier_calls"] == 0


def test_fused_two_tier_ragged_batch_and_t0(gp, ref):
    """Ragged / empty curves, NaN samples, negative t - t0, per-curve t0."""
    w = workloads.ragged_batch(nperiods=70)
    periods = ref.make_period_grid(0.3, 7.0, w.nperiods, workloads.GRID_UNIFORM_PERIOD)
    t0 = np.linspace(-1.0, 2.0, w.ncurves)
    check_fused(gp, ref, w.times, w.flux, periods, 4096, 256, t0=t0, offsets=w.offsets, lattice=False)
    check_fused(gp, ref, w.times, w.flux, periods, 2048, 64, t0=t0, offsets=w.offsets, lattice=False)


def test_two_tier_long_curve_count_flush(gp, ref):
    """70,000 and 140,000 epochs: more samples than a 16-bit count half
    holds, so the packed counts are flushed once / twice; all samples at ONE phase (P = cadence)
    puts every point in a single intermediary bin."""
    dt = workloads.KEPLER_CADENCE_D
    for n in (70000, 140000):
        w = workloads.paper_fold(nperiods=8, n=n)
        periods = np.array([0.2, 0.37, 0.731, 1.0, dt, 2 * dt, 0.5, 10 * dt])
        check_fused(gp, ref, w.times, w.flux, periods, 4096, 256)
        # the unfused route through the same kernel's bin epilogue: bit-exact tier 1
        s, c = gp.gpfc_fold(dev(w.times), dev(w.flux), dev(periods), 4096)
        torch.cuda.synchronize()
        rs, rc, _ = ref.fold(w.times, w.flux, periods, 4096)
        assert np.array_equal(c.cpu().numpy().view(np.uint32), rc)
        assert np.array_equal(s.cpu().numpy(), rs)
        s, c = gp.gpfc_fold(dev(w.times), dev(w.flux), dev(periods), 1024)
        torch.cuda.synchronize()
        rs, rc, _ = ref.fold(w.times, w.flux, periods, 1024)
        assert np.array_equal(c.cpu().numpy().view(np.uint32), rc)
        assert np.array_equal(s.cpu().numpy(), rs)


def test_two_tier_unfused_fallback(gp, ref):
    """(nb1, nb2) that the fused kernel does not cover go through fold + merge kernels."""
    w = workloads.config1(nperiods=8)
    periods = np.array([0.2, 0.3333, 0.5, 0.77, 1.0, 16 * workloads.KEPLER_CADENCE_D])
    gp.gpfc_profile(False)
    check_fused(gp, ref, w.times, w.flux, periods, 512, 64)
    check_fused(gp, ref, w.times, w.flux, periods, 1000, 100)
    check_fused(gp, ref, w.times, w.flux, periods, 4096, 1024)
    check_fused(gp, ref, w.times, w.flux, periods, 4096, 300)
    assert gp.gpfc_path_counters()["unfused_two_tier_calls"] == 4


@pytest.mark.parametrize("seed", range(16))
def test_fused_two_tier_fuzz(gp, ref, seed):
    """Seeded random cases of the whole two-tier fold: batch of 1-3 curves (regular cadence with
    drops, or irregular times; flux off the lattice, any scale), 1-40 periods, (nb1, nb2) from
    the fused and the unfused pairs, optional per-curve t0."""
    rng = np.random.default_rng([105, 111, seed])
    nb1 = int(rng.choice([1024, 2048, 4096]))
    nb2 = int(rng.choice([1, 2, 7, 32, 64, 100, 128, 200, 256, 300]))
    nc = int(rng.integers(1, 4))
    scale = float(2.0 ** rng.integers(-20, 6))
    ts, fs, off = [], [], [0]
    for _ in range(nc):
        n = int(rng.choice([0, 1, 3, 40, int(rng.integers(100, 5000))]))
        if rng.random() < 0.5:
            t = np.cumsum(1 + (rng.random(n) < 0.05)) * workloads.KEPLER_CADENCE_D
        else:
            t = np.sort(rng.uniform(0.0, 60.0, n))
        ts.append(t)
        fs.append(((1.0 + rng.normal(0.0, 1e-3, n)) * scale).astype(np.float32))
        off.append(off[-1] + n)
    times, flux = np.concatenate(ts), np.concatenate(fs)
    periods = np.sort(rng.uniform(0.2, float(rng.choice([1.0, 10.0])), int(rng.integers(1, 41))))
    t0 = rng.uniform(-1.0, 1.0, nc) if rng.random() < 0.5 else None
    off = np.asarray(off, np.int64)
    # check_fused's absolute 1e-6 bar is for relative flux: scale the curves back for it
    m, _ = check_fused(gp, ref, times, (flux.astype(np.float64) / scale).astype(np.float32), periods,
                       nb1, nb2, t0=t0, offsets=off, lattice=False)
    assert np.all(np.isfinite(m))
    # and at the drawn scale: merged means relative to the profile's magnitude
    mean, norm = gp.gpfc_fold_two_tier(dev(times), dev(flux), dev(off), dev(periods), nb1, nb2,
                                       t0=None if t0 is None else dev(t0))
    torch.cuda.synchronize()
    for c in range(nc):
        a, b = int(off[c]), int(off[c + 1])
        omean, onorm, has = oracle_two_tier(ref, times[a:b], flux[a:b], periods, nb1, nb2,
                                            0.0 if t0 is None else float(t0[c]))
        assert np.all(np.abs(mean[c].cpu().numpy() - omean) <= 1e-6 * scale * 2.0)
        sd = omean.std(axis=-1)
        defined = sd >= 1e-9 * np.abs(omean).max(axis=-1)
        err = np.abs(norm[c].cpu().numpy() - onorm)
        assert np.all(err[defined] <= 1e-4 * np.maximum(1.0, np.abs(onorm[defined])))
