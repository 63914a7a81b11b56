"""GPU parity tests (-m gpu): the CUDA path through the C ABI against the CPU
oracle, element by element, on the same seeded inputs.

Bars (BASELINE.json north_star): bin counts bit-exact; bin means within 1e-6
absolute; normalised profiles within 1e-4 * max(1, |ref|) (reading R14).  For the
config inputs (flux on the 2^-24 lattice) the fixed-point sums are exact, so the
fp32 sums are compared bit for bit as well.
"""
import dataclasses

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


def run_gpu(gp, w, periods, t0=None, want=("sum", "count", "norm")):
    s, c, nrm = gp.gpfc_fold_batch(dev(w.times), dev(w.flux), dev(w.offsets), dev(periods),
                                   w.nbins, t0=None if t0 is None else dev(t0), want=want)
    torch.cuda.synchronize()
    out = {}
    out["sum"] = None if s is None else s.cpu().numpy()
    out["count"] = None if c is None else c.cpu().numpy().view(np.uint32)
    out["norm"] = None if nrm is None else nrm.cpu().numpy()
    return out


def check(g, r, exact_sums=False):
    assert np.array_equal(g["count"], r["count"]), "bin counts differ"
    cnt = np.maximum(r["count"], 1).astype(np.float64)
    mean_g = g["sum"].astype(np.float64) / cnt
    mean_r = r["sum64"] / cnt
    assert np.max(np.abs(mean_g - mean_r), initial=0.0) <= 1e-6
    if exact_sums:
        assert np.array_equal(g["sum"], r["sum"]), "fp32 sums differ on lattice input"
    if g.get("norm") is not None:
        ref = r["norm64"]
        err = np.abs(g["norm"].astype(np.float64) - ref)
        tol = 1e-4 * np.maximum(1.0, np.abs(ref))
        assert np.all(err <= tol), "normalised profile off by %g" % float((err / tol).max())


def test_grid_bit_identical(gp, ref):
    for mode in (0, 1, 2, 3):
        for (pmin, pmax, n) in [(0.2, 1.0, 2000), (0.2, 1.0, 1), (0.25, 0.5, 2), (0.2, 1.0, 100000),
                                (0.3, 17.0, 12345)]:
            g = gp.gpfc_make_period_grid(pmin, pmax, n, mode).cpu().numpy()
            r = ref.make_period_grid(pmin, pmax, n, mode)
            assert np.array_equal(g, r), (mode, pmin, pmax, n)
    h = gp.gpfc_make_period_grid_host(0.2, 1.0, 5000, 0)
    assert np.array_equal(h, ref.make_period_grid(0.2, 1.0, 5000, 0))
    assert gp.gpfc_make_period_grid(0.2, 1.0, 0).numel() == 0
    with pytest.raises(gp.GpfcError):
        gp.gpfc_make_period_grid(-1.0, 1.0, 10)
    assert int(gp.gpfc_n_sample(2, 4 * 365, 0.03)) == 97333


def test_hand_vectors_on_gpu(gp):
    """The same hand-worked dyadic vectors the oracle is pinned with."""
    import json, os
    g = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "hand_vectors.json")))
    t = dev(np.array(g["times"], np.float64))
    f = dev(np.array(g["flux"], np.float32))
    for case in g["cases"]:
        s, c = gp.gpfc_fold(t, f, dev(np.array([case["period"]])), g["nbins"], t0=case["t0"])
        assert c.cpu().tolist()[0] == case["count"], case
        assert s.cpu().tolist()[0] == case["sum"], case
    nz = g["normalize"]
    out = gp.gpfc_normalize(dev(np.array([nz["sum"]], np.float32)),
                            dev(np.array([nz["count"]], np.int32)))
    assert np.allclose(out.cpu().numpy()[0], nz["out"], rtol=0, atol=1e-6)


def test_config0_full(gp, ref):
    w = workloads.config0()
    periods = ref.make_period_grid(w.pmin, w.pmax, w.nperiods, w.grid_mode)
    g = run_gpu(gp, w, periods)
    r = ref.fold_batch(w.times, w.flux, w.offsets, periods, w.nbins)
    check(g, r, exact_sums=True)


@pytest.mark.parametrize("nbins", [32, 64, 128, 256, 512, 1024, 2048, 4096])
def test_pow2_nbins_kepler_slice(gp, ref, nbins):
    """Config-1 curve (65,000 samples: many tiles + ragged tail) over a slice of the
    grid that includes cadence-commensurate (degenerate) periods; 37 periods is not
    a multiple of any period-group size, so the ragged last group is exercised."""
    w = workloads.config1(nperiods=37)
    grid = ref.make_period_grid(w.pmin, w.pmax, 200000, w.grid_mode)
    idx = np.linspace(0, 199999, 30).astype(int)
    dt = workloads.KEPLER_CADENCE_D
    periods = np.concatenate([grid[idx], [10 * dt, 12 * dt, 16 * dt, 20 * dt, 0.5, 0.25, 1.0]])
    w.nbins = nbins
    g = run_gpu(gp, w, periods)
    r = ref.fold_batch(w.times, w.flux, w.offsets, periods, nbins)
    check(g, r, exact_sums=True)


@pytest.mark.parametrize("nbins", [1, 2, 7, 16, 100, 1000, 4095])
def test_generic_nbins(gp, ref, nbins):
    w = workloads.config0(nperiods=25)
    w.nbins = nbins
    periods = ref.make_period_grid(w.pmin, w.pmax, 25, w.grid_mode)
    g = run_gpu(gp, w, periods)
    r = ref.fold_batch(w.times, w.flux, w.offsets, periods, nbins)
    check(g, r, exact_sums=True)


@pytest.mark.parametrize("nbins", [1, 3, 8, 31, 33, 100, 200, 250, 255])
def test_any_nbins_up_to_256_on_the_fast_kernel(gp, ref, nbins):
    """nbins <= 256 that are not a power of two >= 32 run on fold_lp_kernel<true> (bin =
    high word of frac(u/P) 2^32 * nbins), not on the generic kernel: Kepler-shaped curve with
    many tiles and a ragged tail, 37 periods incl. cadence-commensurate ones, all outputs."""
    w = workloads.config1(nperiods=37)
    grid = ref.make_period_grid(w.pmin, w.pmax, 200000, w.grid_mode)
    dt = workloads.KEPLER_CADENCE_D
    periods = np.concatenate([grid[np.linspace(0, 199999, 30).astype(int)],
                              [10 * dt, 12 * dt, 16 * dt, 20 * dt, 0.5, 0.25, 1.0]])
    w.nbins = nbins
    gp.gpfc_profile(False)
    g = run_gpu(gp, w, periods)
    c = gp.gpfc_path_counters()
    assert c["generic_kernel_calls"] == 0 and c["exact_path_items"] == 0
    r = ref.fold_batch(w.times, w.flux, w.offsets, periods, nbins)
    check(g, r, exact_sums=True)
    # fused normalisation only
    g2 = run_gpu(gp, w, periods, want=("norm",))
    err = np.abs(g2["norm"].astype(np.float64) - r["norm64"])
    assert np.all(err <= 1e-4 * np.maximum(1.0, np.abs(r["norm64"])))


@pytest.mark.parametrize("nbins", [64, 100, 256])
def test_ragged_batch_edge_cases(gp, ref, nbins):
    """Empty and tiny curves, irregular times, negative t - t0, non-finite samples,
    invalid periods, per-curve t0, flux off the lattice."""
    w = workloads.ragged_batch(nbins=nbins)
    periods = ref.make_period_grid(w.pmin, w.pmax, w.nperiods, w.grid_mode)
    periods[3] = np.nan
    periods[4] = 0.0
    periods[5] = -0.5
    periods[6] = np.inf
    periods[7] = 1e-9            # x far outside the fast range
    periods[8] = 1e9
    periods[9] = 1e-320          # (t - t0) / P overflows: samples skipped (R20)
    t0 = np.linspace(-1.0, 2.0, w.ncurves)
    g = run_gpu(gp, w, periods, t0=t0)
    r = ref.fold_batch(w.times, w.flux, w.offsets, periods, nbins, t0=t0)
    check(g, r)
    for j in (3, 4, 5, 6):
        assert not g["count"][:, j].any() and not g["sum"][:, j].any() and not g["norm"][:, j].any()
    # t0 = NULL
    g0 = run_gpu(gp, w, periods)
    r0 = ref.fold_batch(w.times, w.flux, w.offsets, periods, nbins)
    check(g0, r0)


@pytest.mark.parametrize("nbins", [64, 256, 512, 1024])
def test_packed_counts_long_and_short_curves(gp, ref, nbins):
    """fold_pk (nbins 512 ... 4096) packs the counts of rows k and k + rows/2 in the two
    half-words of one word, which cannot wrap for curves of up to 65,535 samples; longer curves
    in the same batch are folded without a flush first, checked, and folded again with the counts
    flushed to a 32-bit side array only if a half-word wrapped (fold_lp, nbins <= 256, keeps
    32-bit counts).  Cadence-locked periods put thousands of samples in one bin."""
    rng = np.random.default_rng(11)
    dt = workloads.KEPLER_CADENCE_D
    curves = []
    for n in (70000, 65535, 65536, 300):
        t = np.arange(n, dtype=np.float64) * dt
        f = (rng.integers(-4000, 4000, n).astype(np.float32)) * np.float32(2.0 ** -24)
        curves.append((t, f, None))
    periods = np.array([16 * dt, 20 * dt, 0.5, 0.7310371, 1.0, 0.2, np.nan, 25 * dt])
    w = workloads._pack("packed", -1, curves, 0.2, 1.0, periods.shape[0], nbins, False)
    g = run_gpu(gp, w, periods)
    r = ref.fold_batch(w.times, w.flux, w.offsets, periods, nbins)
    check(g, r, exact_sums=True)
    assert g["count"].max() > 4000           # the degenerate bins are really there


def test_guard_band_samples_match_division(gp, ref):
    """Samples that sit exactly on bin edges (t = k P / nb, t = t0) and their
    fp64 neighbours: the reciprocal fast path must fall back to the division."""
    nb = 256
    rng = np.random.default_rng(5)
    periods = np.concatenate([rng.uniform(0.2, 1.0, 30), [0.5, 0.25, 0.75, 1.0, 0.3]])
    ts = [np.zeros(3)]
    for p in periods[:12]:
        k = rng.integers(0, 200000, 400)
        e = (k * p) / nb
        ts += [e, np.nextafter(e, np.inf), np.nextafter(e, -np.inf), k.astype(np.float64) * p]
    t = np.sort(np.concatenate(ts))
    f = rng.integers(-1000, 1000, t.shape[0]).astype(np.float32) * np.float32(2.0 ** -20)
    w = workloads._pack("edges", -1, [(t, f, None)], 0.2, 1.0, periods.shape[0], nb, False)
    for nbins in (64, 256, 1024, 4096):
        w.nbins = nbins
        g = run_gpu(gp, w, periods)
        r = ref.fold_batch(w.times, w.flux, w.offsets, periods, nbins)
        check(g, r, exact_sums=True)
    # bin counts that are not a power of two: the oracle rounds phi * nbins once, so an edge
    # sample can land on either side of k / nbins; edges of 100, 96 and 255 bins and neighbours
    for nbins in (100, 96, 255, 3):
        ts = [np.zeros(2)]
        for p in periods[:12]:
            k = rng.integers(0, 200000, 300)
            e = (k * p) / nbins
            ts += [e, np.nextafter(e, np.inf), np.nextafter(e, -np.inf), k.astype(np.float64) * p]
        t = np.sort(np.concatenate(ts))
        f = rng.integers(-1000, 1000, t.shape[0]).astype(np.float32) * np.float32(2.0 ** -20)
        w2 = workloads._pack("edges", -1, [(t, f, None)], 0.2, 1.0, periods.shape[0], nbins, False)
        g = run_gpu(gp, w2, periods)
        r = ref.fold_batch(w2.times, w2.flux, w2.offsets, periods, nbins)
        check(g, r, exact_sums=True)


def test_uncentred_flux_is_centred_internally(gp, ref):
    """Flux around 1.0 (not median-subtracted): the library removes a per-curve
    constant before quantising; means still agree to 1e-6."""
    w = workloads.config0(nperiods=40)
    w.flux = (w.flux + np.float32(1.0)).astype(np.float32)
    periods = ref.make_period_grid(w.pmin, w.pmax, 40, w.grid_mode)
    g = run_gpu(gp, w, periods, want=("sum", "count"))
    r = ref.fold_batch(w.times, w.flux, w.offsets, periods, w.nbins)
    check(g, r)


def test_batch_configs_scaled(gp, ref):
    """Config 2 and 4 shapes with fewer curves / periods (full parity)."""
    w2 = workloads.config2(ncurves=3, nperiods=40)
    p2 = ref.make_period_grid(w2.pmin, w2.pmax, 40, w2.grid_mode)
    check(run_gpu(gp, w2, p2), ref.fold_batch(w2.times, w2.flux, w2.offsets, p2, w2.nbins),
          exact_sums=True)
    w4 = workloads.config4(ncurves=5, nperiods=50)
    p4 = ref.make_period_grid(w4.pmin, w4.pmax, 50, w4.grid_mode)
    g4 = run_gpu(gp, w4, p4, want=("norm",))         # fused: only the normalised profile
    r4 = ref.fold_batch(w4.times, w4.flux, w4.offsets, p4, w4.nbins)
    err = np.abs(g4["norm"].astype(np.float64) - r4["norm64"])
    assert np.all(err <= 1e-4 * np.maximum(1.0, np.abs(r4["norm64"])))
    assert g4["sum"] is None and g4["count"] is None


def test_single_curve_fold_and_normalize_entry_points(gp, ref):
    w = workloads.config0(nperiods=64)
    periods = ref.make_period_grid(w.pmin, w.pmax, 64, w.grid_mode)
    s, c = gp.gpfc_fold(dev(w.times), dev(w.flux), dev(periods), w.nbins, t0=0.37)
    nrm = gp.gpfc_normalize(s, c)
    torch.cuda.synchronize()
    rs, rc, rs64 = ref.fold(w.times, w.flux, periods, w.nbins, t0=0.37)
    assert np.array_equal(c.cpu().numpy().view(np.uint32), rc)
    assert np.array_equal(s.cpu().numpy(), rs)
    rn = ref.normalize(rs, rc, want64=True)[1]
    err = np.abs(nrm.cpu().numpy().astype(np.float64) - rn)
    assert np.all(err <= 1e-4 * np.maximum(1.0, np.abs(rn)))


def test_host_entry_point_and_workspace(gp, ref):
    w = workloads.config2(ncurves=2, nperiods=24)
    periods = ref.make_period_grid(w.pmin, w.pmax, 24, w.grid_mode)
    shape = (w.ncurves, 24, w.nbins)
    s = np.empty(shape, np.float32)
    c = np.empty(shape, np.uint32)
    nrm = np.empty(shape, np.float32)
    gp.gpfc_fold_batch_host(w.times, w.flux, w.offsets, periods, w.nbins, out_sum=s, out_count=c,
                            out_norm=nrm)
    r = ref.fold_batch(w.times, w.flux, w.offsets, periods, w.nbins)
    check({"sum": s, "count": c, "norm": nrm}, r, exact_sums=True)
    # caller-owned workspace
    need = gp.gpfc_workspace_bytes(w.ncurves, w.n_total, 24, w.nbins)
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    gp.gpfc_set_workspace(ws)
    try:
        g = run_gpu(gp, w, periods)
    finally:
        gp.gpfc_set_workspace(None)
    check(g, r, exact_sums=True)


def test_empty_and_error_paths(gp):
    e64 = torch.empty(0, dtype=torch.float64, device="cuda")
    e32 = torch.empty(0, dtype=torch.float32, device="cuda")
    per = dev(np.array([0.5, 0.7]))
    s, c = gp.gpfc_fold(e64, e32, per, 16)                  # n = 0: zero rows
    assert not s.cpu().numpy().any() and not c.cpu().numpy().any()
    s, c = gp.gpfc_fold(e64, e32, e64, 16)                  # nperiods = 0: no-op
    assert s.shape == (0, 16)
    with pytest.raises(gp.GpfcError):
        gp.gpfc_fold(e64, e32, per, 0)
    with pytest.raises(gp.GpfcError):
        gp.gpfc_fold(e64, e32, per, 5000)
    with pytest.raises(gp.GpfcError):
        gp.gpfc_fold(torch.empty(4, dtype=torch.float64), e32, per, 16)   # host tensor


def test_host_path_streams_several_chunks(gp, ref):
    """gpfc_fold_batch_host folds the curves in chunks of about 512 MB of output and copies
    chunk k back while chunk k+1 is folded: 20 curves x 20,000 periods x 256 bins x 3 arrays
    = 1.2 GB = 3 chunks.  Per-curve t0, ragged lengths; sampled rows against the oracle."""
    rng = np.random.default_rng(21)
    curves = []
    for c in range(20):
        n = int(rng.integers(2000, 6000))
        t = np.sort(rng.uniform(0.0, 90.0, n))
        f = (rng.integers(-3000, 3000, n).astype(np.float32)) * np.float32(2.0 ** -22)
        curves.append((t, f, None))
    npd = 20000
    w = workloads._pack("host_chunks", -1, curves, 0.2, 1.0, npd, 256, False)
    periods = ref.make_period_grid(w.pmin, w.pmax, npd, w.grid_mode)
    t0 = np.linspace(-2.0, 2.0, w.ncurves)
    shape = (w.ncurves, npd, 256)
    s = np.empty(shape, np.float32)
    c = np.empty(shape, np.uint32)
    nrm = np.empty(shape, np.float32)
    gp.gpfc_fold_batch_host(w.times, w.flux, w.offsets, periods, 256, t0=t0, out_sum=s,
                            out_count=c, out_norm=nrm)
    idx = np.array(sorted(set(rng.integers(0, npd, 25).tolist()) | {0, npd - 1}))
    for cu in (0, 7, 8, 15, 16, 19):          # first / last curves of each chunk
        a, b = int(w.offsets[cu]), int(w.offsets[cu + 1])
        r = ref.fold_batch(w.times[a:b], w.flux[a:b], np.array([0, b - a], np.int64), periods[idx],
                           256, t0=t0[cu:cu + 1])
        check({"sum": s[cu:cu + 1, idx], "count": c[cu:cu + 1, idx], "norm": nrm[cu:cu + 1, idx]}, r,
              exact_sums=True)
    assert np.array_equal(c.sum(axis=2, dtype=np.int64), np.broadcast_to(
        np.diff(w.offsets)[:, None], (w.ncurves, npd)))


def test_flat_and_sparse_profiles_fused_normalise(gp, ref):
    """Degenerate profiles through the fused epilogue: constant flux (every bin mean equal:
    s = 0 -> mu everywhere, exactly as the oracle), two samples, one sample, samples in one bin."""
    t = np.arange(5000, dtype=np.float64) * 0.0137
    curves = [(t, np.full(5000, np.float32(3.0 * 2.0 ** -12)), None),
              (t, np.zeros(5000, np.float32), None),
              (np.array([0.3, 0.9]), np.array([1.0, -1.0], np.float32) * np.float32(2.0 ** -10), None),
              (np.array([0.3]), np.array([2.0 ** -9], np.float32), None),
              (np.full(40, 0.25) + np.arange(40) * 0.5, np.linspace(-1, 1, 40).astype(np.float32), None)]
    periods = np.array([0.5, 0.37, 1.0, 0.25, 0.713])
    for nbins in (32, 128, 256, 1024):
        w = workloads._pack("flat", -1, curves, 0.2, 1.0, periods.shape[0], nbins, False)
        g = run_gpu(gp, w, periods)
        r = ref.fold_batch(w.times, w.flux, w.offsets, periods, nbins)
        check(g, r)
        # constant-flux curves: the normalised profile is exactly flat
        assert np.array_equal(g["norm"][0], np.full_like(g["norm"][0], np.float32(3.0 * 2.0 ** -12)))
        assert not g["norm"][1].any()
        gf = run_gpu(gp, w, periods, want=("norm",))
        assert np.array_equal(gf["norm"], g["norm"])


def test_profile_hooks_count_launches(gp):
    """gpfc_profile_read: one event pair per fold-kernel launch, and every kernel of the
    library counted where it is launched (grid, two prepass kernels, fold), for each of the
    three fold kernels."""
    w = workloads.config0(nperiods=64)
    periods = gp.gpfc_make_period_grid(w.pmin, w.pmax, 64, w.grid_mode)
    t, f, off = dev(w.times), dev(w.flux), dev(w.offsets)
    for nbins in (w.nbins, 1024, 4096, 100):
        gp.gpfc_profile(True)
        for _ in range(3):
            gp.gpfc_make_period_grid(w.pmin, w.pmax, 64, w.grid_mode, out=periods)
            gp.gpfc_fold_batch(t, f, off, periods, nbins)
        p = gp.gpfc_profile_read()
        gp.gpfc_profile(False)
        assert p["fold_launches"] == 3 and p["kernel_launches"] == 3 * 4, (nbins, p)
        assert 0.0 < p["fold_kernel_ms"] < 1000.0
    gp.gpfc_profile(True)
    gp.gpfc_fold(t, f, periods, 64)                    # single-curve entry: + the offsets kernel
    gp.gpfc_normalize(*gp.gpfc_fold(t, f, periods, 64))
    p = gp.gpfc_profile_read()
    gp.gpfc_profile(False)
    assert p["fold_launches"] == 2 and p["kernel_launches"] == 2 * 4 + 1


# ------------------------------------------------------------------ any sample order (gpfc.h)

@pytest.mark.parametrize("nbins", [256, 1024, 4096, 100])
def test_unsorted_and_duplicate_times(gp, ref, nbins):
    """gpfc.h: samples may come in any order.  A shuffled Kepler-shaped curve (tiles then span
    the whole baseline: the kernels take the exact division for every point-period), the same
    curve with every 7th time stamp duplicated, and a curve sorted in DEScending order: bins,
    counts and sums identical to the sorted fold, and the slow path is reported."""
    w = workloads.config1(nperiods=40)
    rng = np.random.default_rng(11)
    periods = ref.make_period_grid(w.pmin, w.pmax, w.nperiods)
    n = 20000
    t, f = w.times[:n].copy(), w.flux[:n].copy()
    dup = np.arange(0, n - 1, 7)
    t[dup] = t[dup + 1]                                  # duplicate time stamps
    rs, rc, _ = ref.fold(t, f, periods, nbins)
    perm = rng.permutation(n)
    gp.gpfc_profile(False)
    for order in (perm, np.arange(n)[::-1].copy(), np.arange(n)):
        s, c = gp.gpfc_fold(dev(t[order]), dev(f[order]), dev(periods), nbins)
        torch.cuda.synchronize()
        assert np.array_equal(c.cpu().numpy().view(np.uint32), rc)
        assert np.array_equal(s.cpu().numpy(), rs)       # exact integer sums: order-free
    counters = gp.gpfc_path_counters()
    assert counters["generic_kernel_calls"] == 0
    if nbins != 100:
        # the shuffled call took the exact path (at 100 bins the DFMA counts cycles, not rows:
        # even a tile spanning the whole baseline stays inside the fast path's range)
        assert counters["exact_path_items"] > 0


def test_outputs_with_4_byte_alignment(gp, ref):
    """Outputs that are contiguous but only 4-byte aligned (a view at offset 1 of a larger
    buffer) are accepted: scalar stores instead of vector stores."""
    w = workloads.config2(ncurves=2, nperiods=70)
    periods = ref.make_period_grid(w.pmin, w.pmax, w.nperiods)
    for nbins in (64, 256, 1024):
        r = ref.fold_batch(w.times, w.flux, w.offsets, periods, nbins)
        shape = (w.ncurves, w.nperiods, nbins)
        nel = int(np.prod(shape))
        bs = torch.zeros(nel + 3, dtype=torch.float32, device="cuda")
        bc = torch.zeros(nel + 3, dtype=torch.int32, device="cuda")
        bn = torch.zeros(nel + 3, dtype=torch.float32, device="cuda")
        os_, oc, on = (b[1:1 + nel].view(shape) for b in (bs, bc, bn))
        assert os_.data_ptr() % 16 == 4
        gp.gpfc_fold_batch(dev(w.times), dev(w.flux), dev(w.offsets), dev(periods), nbins,
                           out_sum=os_, out_count=oc, out_norm=on)
        torch.cuda.synchronize()
        assert np.array_equal(oc.cpu().numpy().view(np.uint32), r["count"])
        assert np.array_equal(os_.cpu().numpy(), r["sum"])
        err = np.abs(on.cpu().numpy().astype(np.float64) - r["norm64"])
        assert np.all(err <= 1e-4 * np.maximum(1.0, np.abs(r["norm64"])))
        for b in (bs, bc, bn):                            # nothing written outside the view
            assert float(b[0]) == 0 and float(b[nel + 1]) == 0 and float(b[nel + 2]) == 0


def test_fold_batch_in_a_cuda_graph(gp, ref):
    """Device-pointer calls never synchronise: with a registered workspace the whole step
    (grid + batched fold + normalise) is captured in a CUDA graph and replayed."""
    w = workloads.config2(ncurves=2, nperiods=96)
    t, f, off = dev(w.times), dev(w.flux), dev(w.offsets)
    shape = (w.ncurves, w.nperiods, w.nbins)
    periods = torch.empty(w.nperiods, dtype=torch.float64, device="cuda")
    s = torch.empty(shape, dtype=torch.float32, device="cuda")
    c = torch.empty(shape, dtype=torch.int32, device="cuda")
    nrm = torch.empty(shape, dtype=torch.float32, device="cuda")
    ws = torch.empty(gp.gpfc_workspace_bytes(w.ncurves, w.n_total, w.nperiods, w.nbins),
                     dtype=torch.uint8, device="cuda")
    gp.gpfc_set_workspace(ws)
    try:
        gp.gpfc_init()
        g = torch.cuda.CUDAGraph()
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            with torch.cuda.graph(g, stream=side):
                gp.gpfc_make_period_grid(w.pmin, w.pmax, w.nperiods, w.grid_mode, out=periods)
                gp.gpfc_fold_batch(t, f, off, periods, w.nbins, out_sum=s, out_count=c, out_norm=nrm)
        torch.cuda.current_stream().wait_stream(side)
        for _ in range(2):
            s.zero_(); c.zero_(); nrm.zero_(); periods.zero_()
            g.replay()
            torch.cuda.synchronize()
            pr = ref.make_period_grid(w.pmin, w.pmax, w.nperiods, w.grid_mode)
            assert np.array_equal(periods.cpu().numpy(), pr)
            r = ref.fold_batch(w.times, w.flux, w.offsets, pr, w.nbins)
            assert np.array_equal(c.cpu().numpy().view(np.uint32), r["count"])
            assert np.array_equal(s.cpu().numpy(), r["sum"])
    finally:
        gp.gpfc_set_workspace(None)


def test_second_device_if_present(gp, ref):
    """Per-device library state: the same process folds on cuda:1 after cuda:0."""
    if torch.cuda.device_count() < 2:
        pytest.skip("one CUDA device")
    w = workloads.config2(ncurves=1, nperiods=64)
    periods = ref.make_period_grid(w.pmin, w.pmax, w.nperiods)
    r = ref.fold_batch(w.times, w.flux, w.offsets, periods, 1024)
    for d in (0, 1, 0):
        with torch.cuda.device(d):
            to = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda(d)
            s, c, _ = gp.gpfc_fold_batch(to(w.times), to(w.flux), to(w.offsets), to(periods), 1024,
                                         want=("sum", "count"))
            torch.cuda.synchronize(d)
            assert np.array_equal(c.cpu().numpy().view(np.uint32), r["count"])
            assert np.array_equal(s.cpu().numpy(), r["sum"])


def test_two_host_threads_on_their_own_streams(gp, ref):
    """The stream, the workspace, the error text and the launch counters are per calling
    thread (gpfc.h): two threads fold different batches at the same time on their own streams
    and each gets what a lone call gives."""
    import threading
    ws = [workloads.config2(ncurves=3, nperiods=400), workloads.config4(ncurves=5, nperiods=300)]
    pers = [ref.make_period_grid(w.pmin, w.pmax, w.nperiods, w.grid_mode) for w in ws]
    alone = [gp.gpfc_fold_batch(dev(w.times), dev(w.flux), dev(w.offsets), dev(p), w.nbins)
             for w, p in zip(ws, pers)]
    torch.cuda.synchronize()
    got, errs = [None, None], []

    def work(k):
        try:
            st = torch.cuda.Stream()
            w, p = ws[k], pers[k]
            with torch.cuda.stream(st):
                t, f, o, pd = dev(w.times), dev(w.flux), dev(w.offsets), dev(p)
                buf = torch.empty(gp.gpfc_workspace_bytes(w.ncurves, w.n_total, w.nperiods, w.nbins),
                                  dtype=torch.uint8, device="cuda")
                gp.gpfc_set_workspace(buf)
                for _ in range(5):
                    out = gp.gpfc_fold_batch(t, f, o, pd, w.nbins)
                gp.gpfc_set_workspace(None)
                st.synchronize()
            got[k] = out
        except BaseException as exc:      # surfaced in the main thread
            errs.append(exc)

    th = [threading.Thread(target=work, args=(k,)) for k in range(2)]
    for t_ in th:
        t_.start()
    for t_ in th:
        t_.join()
    assert not errs, errs
    for k in range(2):
        for x, y in zip(got[k], alone[k]):
            assert torch.equal(x, y)


@pytest.mark.parametrize("nbins", [128, 250, 256, 1024, 4096])
def test_every_subset_of_outputs(gp, ref, nbins):
    """The epilogues are specialised per set of requested outputs (all three, the normalised
    profile alone, anything else): every subset gives the same arrays as the full call, and
    the full call matches the oracle.  Several curves share t0 with their first samples
    (zero-time samples are added to bin 0 apart from the fold)."""
    w = workloads.config2(ncurves=3, nperiods=101)
    w.times[w.offsets[1] + 1] = w.times[w.offsets[1]]          # two samples at t == t0
    periods = ref.make_period_grid(w.pmin, w.pmax, w.nperiods)
    periods[17] = np.nan
    r = ref.fold_batch(w.times, w.flux, w.offsets, periods, nbins)
    full = run_gpu(gp, dataclasses.replace(w, nbins=nbins), periods)
    check(full, r, exact_sums=True)
    for want in (("sum",), ("count",), ("norm",), ("sum", "count"), ("sum", "norm"), ("count", "norm")):
        g = run_gpu(gp, dataclasses.replace(w, nbins=nbins), periods, want=want)
        for k in ("sum", "count", "norm"):
            if k in want:
                assert np.array_equal(g[k], full[k]), (want, k)
            else:
                assert g[k] is None


@pytest.mark.parametrize("nbins", [128, 256, 1024, 4096])
def test_normalised_profile_does_not_depend_on_the_flux_scale(gp, ref, nbins):
    """The epilogues keep fp32 deviations in units of the curve's fixed-point quantum, so a
    curve scaled by 2^-123 (fp32 denormals: flux of order 1e-40, bin-mean deviations of order
    2^-140, which fp32 itself would keep to 9 bits) or by 2^40 still gives the oracle's
    normalised profile: the z-score part is scale-free, only the profile mean carries the scale."""
    w = workloads.config2(ncurves=2, nperiods=64)
    periods = ref.make_period_grid(w.pmin, w.pmax, w.nperiods)
    for scale in (2.0 ** -123, 2.0 ** 40):
        flux = (w.flux.astype(np.float64) * scale).astype(np.float32)
        ws = dataclasses.replace(w, flux=flux, nbins=nbins)
        g = run_gpu(gp, ws, periods)
        r = ref.fold_batch(ws.times, ws.flux, ws.offsets, periods, nbins)
        assert np.array_equal(g["count"], r["count"])
        ok = np.abs(g["sum"].astype(np.float64) - r["sum64"]) <= 1e-6 * scale * np.maximum(r["count"], 1)
        assert ok.all()
        err = np.abs(g["norm"].astype(np.float64) - r["norm64"])
        assert np.all(err <= 1e-4 * np.maximum(1.0, np.abs(r["norm64"])))


@pytest.mark.parametrize("nbins,nperiods", [(256, 14500), (100, 14500), (128, 96 * 148 + 1), (256, 96 * 148)])
def test_item_counts_around_one_wave(gp, ref, nbins, nperiods):
    """One curve over a few more than 148 work items of 96 periods (a second, nearly empty
    wave of the persistent grid: those groups run as single-slot items of fold_lp_tail_kernel),
    a last group of a single period, exactly 148 items (no tail kernel)."""
    w = workloads.config1(nperiods=8)
    n = 3000
    periods = ref.make_period_grid(0.2, 1.0, nperiods)
    periods[[5, nperiods - 97]] = np.nan
    ws = dataclasses.replace(w, times=w.times[:n], flux=w.flux[:n], offsets=np.array([0, n], np.int64), nbins=nbins)
    g = run_gpu(gp, ws, periods)
    r = ref.fold_batch(ws.times, ws.flux, ws.offsets, periods, nbins)
    check(g, r, exact_sums=True)


@pytest.mark.parametrize("nbins", [64, 100, 256])
def test_edge_cases_through_the_main_fold_lp_kernel(gp, ref, nbins):
    """Calls of fewer than ~50 work items run entirely on fold_lp_tail_kernel (single-slot
    items), which is where the small edge-case tests above end up.  The same edge cases with
    enough periods for whole waves of three-slot items on fold_lp_kernel: the ragged batch
    (empty and tiny curves, NaN samples, negative t - t0, per-curve t0, invalid and extreme
    periods), flat and sparse profiles, 4-byte-aligned outputs."""
    w = workloads.ragged_batch(nbins=nbins)
    nper = 96 * (148 // w.ncurves + 2) + 5            # > 148 items, a partial last group per curve
    periods = ref.make_period_grid(0.2, 3.0, nper, workloads.GRID_UNIFORM_PERIOD)
    periods[[3, 200, nper - 1]] = np.nan
    periods[[4, 97]] = [0.0, -0.5]
    periods[[7, 300]] = [1e-9, 1e9]
    periods[9] = 1e-320
    t0 = np.linspace(-1.0, 2.0, w.ncurves)
    ws = dataclasses.replace(w, nperiods=nper)
    g = run_gpu(gp, ws, periods, t0=t0)
    r = ref.fold_batch(w.times, w.flux, w.offsets, periods, nbins, t0=t0)
    check(g, r)
    c = gp.gpfc_path_counters()
    assert c["generic_kernel_calls"] == 0
    # flat / sparse profiles, outputs at offset 4 bytes
    t = np.arange(3000, dtype=np.float64) * 0.0137
    curves = [(t, np.full(3000, np.float32(3.0 * 2.0 ** -12)), None),
              (np.array([0.3, 0.9]), np.array([1.0, -1.0], np.float32) * np.float32(2.0 ** -10), None),
              (np.array([0.3]), np.array([2.0 ** -9], np.float32), None)]
    nper2 = 96 * 52
    p2 = ref.make_period_grid(0.25, 1.0, nper2)
    wf = workloads._pack("flat", -1, curves, 0.25, 1.0, nper2, nbins, False)
    r2 = ref.fold_batch(wf.times, wf.flux, wf.offsets, p2, nbins)
    shape = (wf.ncurves, nper2, nbins)
    nel = int(np.prod(shape))
    bufs = [torch.zeros(nel + 3, dtype=dt, device="cuda") for dt in (torch.float32, torch.int32, torch.float32)]
    os_, oc, on = (b[1:1 + nel].view(shape) for b in bufs)
    gp.gpfc_fold_batch(dev(wf.times), dev(wf.flux), dev(wf.offsets), dev(p2), nbins,
                       out_sum=os_, out_count=oc, out_norm=on)
    torch.cuda.synchronize()
    g2 = {"sum": os_.cpu().numpy(), "count": oc.cpu().numpy().view(np.uint32), "norm": on.cpu().numpy()}
    check(g2, r2)
    assert np.array_equal(g2["norm"][0], np.full_like(g2["norm"][0], np.float32(3.0 * 2.0 ** -12)))
    for b in bufs:
        assert float(b[0]) == 0 and float(b[nel + 1]) == 0
