"""-m gpu: seeded differential fuzzing of gpfc_fold_batch against the oracle.

Every case draws its own shape (curves of 0 .. 3,000 samples, 1 .. 160 periods, nbins from every
kernel's range), its own time structure (regular cadence with gaps and drops, uniform random
times, unsorted times, duplicates, times before t0), flux scale and offset, a few non-finite
samples and invalid periods, and a subset of the outputs.  Bars as in test_gpu_parity.py: counts
bit-exact, bin means within 1e-6 of the flux scale, normalised profiles within 1e-4 max(1, |ref|)
(profiles whose spread is at the rounding level of their own means excepted, as in
test_gpu_two_tier.py).  The cases are fixed by their seeds: a failure names the seed."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

NBINS = [1, 5, 32, 64, 100, 128, 250, 256, 512, 1000, 1024, 2048, 4096]


@pytest.fixture(scope="module")
def gp():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2312_02063_b200 import binding
    binding.lib()          # must load: no fallback
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def draw_case(seed):
    rng = np.random.default_rng([2312, 2063, seed])
    nbins = int(NBINS[seed % len(NBINS)])
    ncurves = int(rng.integers(1, 5))
    scale = float(2.0 ** rng.integers(-30, 11))
    offset = float(rng.choice([0.0, 0.0, 1.0, -3.0]))
    times, flux, offs = [], [], [0]
    for _ in range(ncurves):
        n = int(rng.choice([0, 1, 2, 31, 33, 127, 129, int(rng.integers(200, 3000))]))
        kind = int(rng.integers(0, 4))
        if kind == 0:                                   # cadence with gaps and dropped slots
            slots = np.cumsum(1 + (rng.random(n) < 0.05) + 200 * (rng.random(n) < 0.003))
            t = slots * 0.020433
        elif kind == 1:                                 # irregular
            t = np.sort(rng.uniform(0.0, 90.0, n))
        elif kind == 2:                                 # unsorted, with duplicates
            t = rng.uniform(-5.0, 40.0, n)
            if n > 4:
                t[rng.integers(0, n, n // 8)] = t[0]
        else:                                           # short baseline, fine structure
            t = rng.uniform(0.0, 2.0, n) + 2455000.0
        f = (offset + rng.normal(0.0, 1e-3, n)) * scale
        f32 = f.astype(np.float32)
        if n > 8:
            bad = rng.integers(0, n, 3)
            f32[bad[0]] = np.nan
            t[bad[1]] = np.inf
            f32[bad[2]] = -np.inf
        times.append(t)
        flux.append(f32)
        offs.append(offs[-1] + n)
    times = np.concatenate(times) if times else np.zeros(0)
    flux = np.concatenate(flux) if flux else np.zeros(0, np.float32)
    nper = int(rng.integers(1, 160))
    lo = float(rng.choice([0.05, 0.2, 1.0, 7.0]))
    periods = np.sort(rng.uniform(lo, lo * float(rng.choice([1.5, 5.0, 40.0])), nper))
    if nper > 6:
        periods[int(rng.integers(0, nper))] = np.nan
        periods[int(rng.integers(0, nper))] = -1.0
    t0 = None
    if rng.random() < 0.5:
        t0 = rng.uniform(-1.0, 3.0, ncurves) + (2455000.0 if times.size and times[np.isfinite(times)].max(initial=0) > 1e6 else 0.0)
    wants = [("sum", "count", "norm"), ("norm",), ("sum", "count"), ("count", "norm"), ("sum",)]
    want = wants[int(rng.integers(0, len(wants)))]
    return dict(nbins=nbins, times=times.astype(np.float64), flux=flux, offsets=np.asarray(offs, np.int64),
                periods=periods, t0=t0, want=want, scale=scale * max(1.0, abs(offset)))


@pytest.mark.parametrize("seed", range(52))
def test_fold_batch_fuzz(gp, ref, seed):
    c = draw_case(seed)
    s, cnt, nrm = gp.gpfc_fold_batch(dev(c["times"]), dev(c["flux"]), dev(c["offsets"]), dev(c["periods"]),
                                     c["nbins"], t0=None if c["t0"] is None else dev(c["t0"]), want=c["want"])
    torch.cuda.synchronize()
    r = ref.fold_batch(c["times"], c["flux"], c["offsets"], c["periods"], c["nbins"], t0=c["t0"])
    if "count" in c["want"]:
        assert np.array_equal(cnt.cpu().numpy().view(np.uint32), r["count"]), "bin counts differ"
    else:
        assert cnt is None
    k = np.maximum(r["count"], 1).astype(np.float64)
    if "sum" in c["want"]:
        dmean = np.abs(s.cpu().numpy().astype(np.float64) / k - r["sum64"] / k)
        assert dmean.max(initial=0.0) <= 1e-6 * c["scale"], dmean.max()
    else:
        assert s is None
    if "norm" in c["want"]:
        g = nrm.cpu().numpy().astype(np.float64)
        assert np.all(np.isfinite(g))
        ref_n = r["norm64"]
        err = np.abs(g - ref_n)
        tol = 1e-4 * np.maximum(1.0, np.abs(ref_n))
        # rows whose spread is rounding noise of their own means have no defined scale
        mean = r["sum64"] / k
        filled = r["count"] > 0
        nf = np.maximum(filled.sum(axis=-1), 1)
        mu = (mean * filled).sum(axis=-1) / nf
        sd = np.sqrt((((mean - mu[..., None]) * filled) ** 2).sum(axis=-1) / nf)
        mag = np.abs(mean).max(axis=-1)
        ok_rows = (sd >= 1e-9 * mag) | (sd == 0)
        assert np.all(err[ok_rows] <= tol[ok_rows]), float((err[ok_rows] / tol[ok_rows]).max())
    else:
        assert nrm is None
