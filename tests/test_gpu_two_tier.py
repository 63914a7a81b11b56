"""NEXT row, -m gpu: the paper's step 4 -- equal-count merge of the
intermediary bins (PAPER.md:105, :111 'Fourthly') -- gpfc_merge_equal_count against the oracle's
gpfc_ref_two_tier_merge on the same folded profiles.  Counts and sums fed to both sides are the
(bit-identical) outputs of the fold; the merged means are fp64 on both sides, compared at fp32
resolution.  The pro-rata split itself is reading R18 (parity with the oracle, which is pinned
only by conservation / equal-count / sort-fold properties for the split values)."""
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
    # normalised: every final bin non-empty (count 1), profiles without points stay zero
    has = cnt.reshape(-1, cnt.shape[-1]).sum(axis=-1) > 0
    on = ref.normalize(omean.reshape(-1, nb2).astype(np.float32),
                       np.where(has[:, None], 1, 0).astype(np.uint32) * np.ones((1, nb2), np.uint32),
                       want64=True)[1]
    # the oracle normalises the fp32-rounded means, the kernel the fp64 ones: 1e-4 bar (R14)
    err = np.abs(norm.reshape(-1, nb2) - on)
    flat = np.abs(omean.reshape(-1, nb2)).max(axis=-1) == 0
    tol = 1e-4 * np.maximum(1.0, np.abs(on))
    sd = omean.reshape(-1, nb2).std(axis=-1)
    ok_rows = (sd > 1e-3 * np.abs(omean.reshape(-1, nb2)).max(axis=-1)) | flat
    assert np.all(err[ok_rows] <= tol[ok_rows]), float((err[ok_rows] / tol[ok_rows]).max())
    return mean, omean


def test_merge_hand_cases(gp, ref):
    # counts divide evenly: 8 fine bins of 2 points -> 4 bins of 4 points: plain pair sums
    s = np.array([[1, 2, 3, 4, 5, 6, 7, 8]], np.float32)
    c = np.full((1, 8), 2, np.uint32)
    mean, _ = check_merge(gp, ref, s, c, 4)
    assert np.allclose(mean[0], [3 / 4, 7 / 4, 11 / 4, 15 / 4])
    # everything in one fine bin: every final bin gets that bin's mean
    s = np.array([[0, 0, 12, 0]], np.float32)
    c = np.array([[0, 0, 6, 0]], np.uint32)
    mean, _ = check_merge(gp, ref, s, c, 3)
    assert np.allclose(mean[0], [2, 2, 2])
    # no points -> zeros; nb1 < nb2 (every fine bin split); nb1 not a multiple of 32
    s = np.zeros((1, 16), np.float32)
    c = np.zeros((1, 16), np.uint32)
    mean, _ = check_merge(gp, ref, s, c, 8)
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
    mean, omean = check_merge(gp, ref, s, c, 256)
    # equal-count property: the merged means average to the curve's mean flux
    assert np.allclose(mean.mean(axis=1), w.flux.astype(np.float64).mean(), atol=1e-9)
