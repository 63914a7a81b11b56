"""GPU parity of the on-device light-curve generator (-m gpu): gpfc_make_light_curves through
the C ABI against oracle/gpfc_ref_sim.c for the same (seed, curve, sample) counters.  Both
sides implement the generator specified in include/gpfc.h operation by operation, so the bar
is bit-exact: time stamps, fp32 flux, drawn parameters.  (PAPER.md 2.6: Eq. 2 :162, Table 2
:176-180, trapezoid :170.)"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def gp():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2312_02063_b200 import binding
    binding.lib()          # must load: no fallback
    return binding


FIELDS = ("period_lo", "period_hi", "duration_lo", "duration_hi", "ratio_lo", "ratio_hi",
          "sigma_lo", "sigma_hi", "snr_lo", "snr_hi", "transit_fraction", "cadence", "t_start", "flags")


def both(gp, ref, **over):
    a, b = gp.gpfc_lc_params_default(**over), ref.lc_params_default(**over)
    for k in FIELDS:     # the two defaults are written independently: they must agree (Table 2)
        assert getattr(a, k) == getattr(b, k), k
    return a, b


def compare(gp, ref, seed, nc, n, **over):
    pg, po = both(gp, ref, **over)
    t, f, off, par = gp.gpfc_make_light_curves(seed, nc, n, pg)
    torch.cuda.synchronize()
    rt, rf, rpar = ref.make_light_curves(seed, nc, n, po)
    assert np.array_equal(off.cpu().numpy(), np.arange(nc + 1, dtype=np.int64) * n)
    assert np.array_equal(par.cpu().numpy(), rpar), "drawn parameters differ"
    assert np.array_equal(t.cpu().numpy(), rt), "time stamps differ"
    g = f.cpu().numpy()
    assert np.array_equal(g.view(np.uint32), rf.view(np.uint32)), \
        "flux differs in %d of %d samples" % (int((g != rf).sum()), g.size)
    return g, rpar


@pytest.mark.parametrize("n", [1, 255, 1024, 1025, 5000])
def test_generator_matches_oracle_default_ranges(gp, ref, n):
    """Table 2's ranges, several chunks of 1,024 samples and ragged tails."""
    compare(gp, ref, 20231204, 37, n)


def test_generator_flags_start_time_and_seeds(gp, ref):
    compare(gp, ref, 1, 9, 3000, flags=gp.LC_CENTERED)
    compare(gp, ref, 2, 9, 3000, flags=gp.LC_NO_NOISE)
    compare(gp, ref, 3, 9, 3000, flags=gp.LC_NO_NOISE | gp.LC_CENTERED, t_start=131.51, cadence=0.0013889)
    compare(gp, ref, 2 ** 63 + 12345, 5, 2000, transit_fraction=1.0)      # high key word in use
    compare(gp, ref, 4, 5, 2000, transit_fraction=0.0)
    # degenerate ranges (every draw the same number) and the TESS cadence
    compare(gp, ref, 5, 4, 19440, period_lo=0.5, period_hi=0.5, ratio_lo=0.09, ratio_hi=0.09,
            duration_lo=0.001, duration_hi=1.0, sigma_lo=1e-3, sigma_hi=1e-3, snr_lo=8.0, snr_hi=8.0,
            cadence=0.0013889, transit_fraction=1.0)
    # a duration window that no draw can meet: the 64th draw is clamped on both sides alike
    compare(gp, ref, 6, 6, 500, duration_lo=0.2, duration_hi=0.3)


def test_generator_empty_and_invalid(gp, ref):
    t, f, off, par = gp.gpfc_make_light_curves(1, 0, 100)
    assert f.shape == (0, 100)
    t, f, off, par = gp.gpfc_make_light_curves(1, 3, 0)
    torch.cuda.synchronize()
    assert f.shape == (3, 0) and np.array_equal(off.cpu().numpy(), [0, 0, 0, 0])
    assert np.array_equal(par.cpu().numpy(), ref.make_light_curves(1, 3, 0, ref.lc_params_default())[2])
    with pytest.raises(gp.GpfcError):
        gp.gpfc_make_light_curves(1, 2, 10, gp.gpfc_lc_params_default(cadence=0.0))
    with pytest.raises(gp.GpfcError):
        gp.gpfc_make_light_curves(1, 2, 10, gp.gpfc_lc_params_default(sigma_lo=2e-4, sigma_hi=1e-4))
    # optional outputs
    t, f, off, par = gp.gpfc_make_light_curves(7, 3, 777, want_times=False, want_offsets=False,
                                               want_params=False)
    torch.cuda.synchronize()
    assert t is None and off is None and par is None
    assert np.array_equal(f.cpu().numpy(), ref.make_light_curves(7, 3, 777, ref.lc_params_default())[1])


def test_generator_full_size_batch_sampled(gp, ref):
    """BASELINE config 2's shape (1,024 curves x 65,000 samples) generated on the device; the
    oracle recomputes every 61st curve in full and the first and last 64 samples of every curve."""
    nc, n = 1024, 65000
    pg, po = both(gp, ref, flags=gp.LC_CENTERED)
    t, f, off, par = gp.gpfc_make_light_curves(99, nc, n, pg)
    torch.cuda.synchronize()
    g = f.cpu().numpy()
    _, _, rpar = ref.make_light_curves(99, nc, 1, ref.lc_params_default(flags=ref.LC_CENTERED),
                                       want_times=False)
    gpar = par.cpu().numpy()
    # p, L, sigma, r, tc, alpha, has do not depend on n; the depth does (Eq. 2)
    for col in (0, 1, 2, 4, 5, 6, 7):
        assert np.array_equal(gpar[:, col], rpar[:, col]), col
    sel = np.arange(0, nc, 61)
    # the oracle draws curve c from counter c: generate the first max(sel) + 1 curves' selection
    rt, rf, rp = ref.make_light_curves(99, int(sel.max()) + 1, n, po)
    assert np.array_equal(g[sel].view(np.uint32), rf[sel].view(np.uint32))
    assert np.array_equal(gpar[sel], rp[sel])
    assert np.array_equal(t.cpu().numpy()[sel], rt[sel])
    # moments of the whole batch: noise of the drawn sigma around zero (centred output)
    sig = gpar[:, 2]
    has = gpar[:, 7] == 1.0
    sd = g[~has].astype(np.float64).std(axis=1)
    assert np.all(np.abs(sd / sig[~has] - 1.0) < 0.02)
    assert abs(has.mean() - 0.5) < 0.06


def test_generated_curves_fold_like_the_oracles(gp, ref):
    """Device-generated curves go straight into the fold (no host round trip): the folded
    profiles equal the oracle's fold of the oracle's curves, and the transit shows up at the
    injected period as the deepest bin mean."""
    nc, n, nb = 6, 20000, 64
    pg, po = both(gp, ref, flags=gp.LC_CENTERED, transit_fraction=1.0, snr_lo=30.0, snr_hi=30.0)
    t, f, off, par = gp.gpfc_make_light_curves(31, nc, n, pg)
    p_true = par.cpu().numpy()[:, 0]
    periods = np.concatenate([np.linspace(0.31, 0.99, 41), p_true])
    s, c, nrm = gp.gpfc_fold_batch(t.reshape(-1), f.reshape(-1), off,
                                   torch.from_numpy(periods).cuda(), nb)
    torch.cuda.synchronize()
    rt, rf, _ = ref.make_light_curves(31, nc, n, po)
    r = ref.fold_batch(rt.reshape(-1), rf.reshape(-1), np.arange(nc + 1, dtype=np.int64) * n, periods, nb)
    assert np.array_equal(c.cpu().numpy().view(np.uint32), r["count"])
    assert np.array_equal(s.cpu().numpy(), r["sum"])
    err = np.abs(nrm.cpu().numpy() - r["norm64"])
    assert np.all(err <= 1e-4 * np.maximum(1.0, np.abs(r["norm64"])))
    mean = s.cpu().numpy().astype(np.float64) / np.maximum(c.cpu().numpy().view(np.uint32), 1)
    for k in range(nc):
        depth_at = mean[k].min(axis=1)           # deepest bin mean of every trial period
        assert np.argmin(depth_at) == 41 + k     # ... is deepest at the curve's own period
