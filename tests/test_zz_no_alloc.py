"""-m gpu, collected last: gpfc_fold_noalloc (fold + fused normalisation of one curve on the
library's static device scratch, no allocation of any kind) against the existing path
(gpfc_fold_batch, which takes its scratch from the workspace or the stream-ordered allocator),
on two calls in a row that share the static array -- the second with a shorter curve, other
periods and another kernel, so that it runs over the first call's leftovers -- and then the
first call again.  Bars as in test_gpu_parity.py: counts bit-exact, bin means within 1e-6,
normalised profiles within 1e-4 max(1, |ref|).  Also: the documented limits are refused with a
clear message, and a registered workspace is left as it was."""
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
    binding.lib()          # must load: no fallback
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def both_paths(gp, times, flux, periods, nbins, t0):
    """-> (noalloc outputs, existing-path outputs), each (sum, count, norm) as numpy."""
    t, f, p = dev(times), dev(flux), dev(periods)
    shape = (periods.shape[0], nbins)
    os_ = torch.full(shape, -7.0, dtype=torch.float32, device="cuda")
    oc = torch.full(shape, -7, dtype=torch.int32, device="cuda")
    on = torch.full(shape, -7.0, dtype=torch.float32, device="cuda")
    gp.gpfc_fold_noalloc(t, f, p, nbins, t0, os_, oc, on)
    off = dev(np.array([0, times.shape[0]], np.int64))
    rs, rc, rn = gp.gpfc_fold_batch(t, f, off, p, nbins, t0=dev(np.array([t0], np.float64)))
    torch.cuda.synchronize()
    new = (os_.cpu().numpy(), oc.cpu().numpy().view(np.uint32), on.cpu().numpy())
    old = (rs.cpu().numpy()[0], rc.cpu().numpy().view(np.uint32)[0], rn.cpu().numpy()[0])
    return new, old


def check_same(new, old):
    (s, c, nrm), (rs, rc, rn) = new, old
    assert np.array_equal(c, rc), "bin counts differ"
    k = np.maximum(rc, 1).astype(np.float64)
    assert np.max(np.abs(s.astype(np.float64) / k - rs.astype(np.float64) / k), initial=0.0) <= 1e-6
    err = np.abs(nrm.astype(np.float64) - rn.astype(np.float64))
    assert np.all(err <= 1e-4 * np.maximum(1.0, np.abs(rn))), float(err.max())


def test_noalloc_matches_existing_path_on_consecutive_calls(gp):
    w = workloads.config1(nperiods=8)                      # one Kepler-shaped curve, 65,000 samples
    grid = np.linspace(1.0, 5.0, 777)
    cases = [
        (w.times[:60000], w.flux[:60000], 1.0 / grid, 256, 0.0),                 # fold_lp, 256 rows
        (w.times[100:9100], w.flux[100:9100], 1.0 / grid[::3][:200], 1024, 0.37),    # fold_pk<10>, shorter
        (w.times[:60000], w.flux[:60000], 1.0 / grid, 256, 0.0),                 # the first one again
        (w.times[:5000], w.flux[:5000], np.array([0.3, np.nan, 0.71, -1.0, 0.5]), 100, -2.0),   # any-nbins kernel
    ]
    first = None
    for i, (t, f, p, nb, t0) in enumerate(cases):
        new, old = both_paths(gp, t, f, p, nb, t0)
        check_same(new, old)
        assert new[1].sum() > 0
        if i == 0:
            first = new
        if i == 2:                                          # same inputs, same kernels: same bits
            for a, b in zip(new, first):
                assert np.array_equal(a, b)


def test_noalloc_subset_of_outputs_and_workspace_untouched(gp):
    w = workloads.config1(nperiods=8)
    t, f = dev(w.times[:20000]), dev(w.flux[:20000])
    p = dev(1.0 / np.linspace(1.0, 5.0, 96))
    ws = torch.empty(1 << 20, dtype=torch.uint8, device="cuda")      # far too small for a fold
    gp.gpfc_set_workspace(ws)
    try:
        on = torch.empty((96, 128), dtype=torch.float32, device="cuda")
        gp.gpfc_fold_noalloc(t, f, p, 128, 0.0, None, None, on)
        _, _, rn = gp.gpfc_fold_batch(t, f, dev(np.array([0, 20000], np.int64)), p, 128, want=("norm",))
        torch.cuda.synchronize()
        assert np.array_equal(on.cpu().numpy(), rn.cpu().numpy()[0])
    finally:
        gp.gpfc_set_workspace(None)


def test_noalloc_limits_are_refused(gp):
    small = torch.zeros(8, dtype=torch.float64, device="cuda")
    out = torch.zeros((8, 32), dtype=torch.float32, device="cuda")
    big_t = torch.zeros(131073, dtype=torch.float64, device="cuda")
    big_f = torch.zeros(131073, dtype=torch.float32, device="cuda")
    with pytest.raises(gp.GpfcError, match="GPFC_NOALLOC_MAX_SAMPLES"):
        gp.gpfc_fold_noalloc(big_t, big_f, small, 32, 0.0, out, None, None)
    many = torch.ones(262145, dtype=torch.float64, device="cuda")
    with pytest.raises(gp.GpfcError, match="GPFC_NOALLOC_MAX_PERIODS"):
        gp.gpfc_fold_noalloc(big_t[:100], big_f[:100], many, 32, 0.0, out, None, None)
    out4k = torch.zeros((8, 4096), dtype=torch.float32, device="cuda")
    with pytest.raises(gp.GpfcError, match="65408"):
        gp.gpfc_fold_noalloc(big_t[:70000], big_f[:70000], small, 4096, 0.0, out4k, None, None)
    # 70,000 samples are fine at nbins <= 256
    periods = dev(np.array([0.2, 0.5, 0.9, 1.0, 0.33, 0.47, 0.61, 0.83]))
    times = dev(np.arange(70000) * 0.020433)
    cnt = torch.zeros((8, 32), dtype=torch.int32, device="cuda")
    gp.gpfc_fold_noalloc(times, big_f[:70000], periods, 32, 0.0, None, cnt, None)
    torch.cuda.synchronize()
    assert np.all(cnt.cpu().numpy().sum(axis=1) == 70000)
