"""Pins of the generator oracle (oracle/gpfc_ref_sim.c; PAPER.md 2.6: Eq. 2 :162, Table 2
:176-180, trapezoid :170, Fig. 7 :188).  CPU only.  Each check is chosen so that a plausible
mistake (a wrong Philox constant or round count, a dropped series term, a wrong octant sign,
Eq. 2 inverted the wrong way, duration measured at the base instead of at half depth) fails."""
import json
import math
import os

import numpy as np
import pytest

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def test_philox_known_answers(ref):
    kat = json.load(open(os.path.join(GOLDEN, "philox_kat.json")))["vectors"]
    assert len(kat) == 3
    for v in kat:
        ctr = [int(x, 16) for x in v["ctr"]]
        key = [int(x, 16) for x in v["key"]]
        out = ref.philox4x32_10(ctr, key)
        assert [int(x) for x in out] == [int(x, 16) for x in v["out"]]


def test_uniform_maps_are_exact_and_open(ref):
    assert ref.u32_to_unit(0) == 2.0 ** -33
    assert ref.u32_to_unit(0xffffffff) == 1.0 - 2.0 ** -33
    assert ref.u32_to_unit(0x80000000) == 0.5 + 2.0 ** -33
    assert ref.u52_to_unit(0, 0) == 2.0 ** -53
    assert ref.u52_to_unit(0xffffffff, 0xffffffff) == 1.0 - 2.0 ** -53
    # the low 12 bits of the second word are not used
    assert ref.u52_to_unit(5, 0x00001fff) == ref.u52_to_unit(5, 0x00001000)
    assert ref.u52_to_unit(1, 0) == (2.0 ** 20 + 0.5) * 2.0 ** -52


def test_ln_series_against_libm(ref):
    rng = np.random.default_rng(11)
    us = np.concatenate([rng.random(4000), 2.0 ** -rng.integers(1, 53, 500) * (1 + rng.random(500)),
                         [2.0 ** -53, 1.0 - 2.0 ** -53, 0.5, 0.70710678118654752, 0.7071067811865476,
                          0.25, 1.0]])
    us = us[(us > 0) & (us <= 1.0)]
    for u in us:
        got, want = ref.ln(float(u)), math.log(float(u))
        assert abs(got - want) <= 4 * abs(np.spacing(want)) + 1e-300, (u, got, want)
    assert ref.ln(1.0) == 0.0


def test_cos2pi_series_against_libm(ref):
    rng = np.random.default_rng(12)
    vs = np.concatenate([rng.random(4000), np.arange(0, 16) / 16.0, np.arange(0, 16) / 16.0 + 2.0 ** -33,
                         [1.0 - 2.0 ** -33]])
    two_pi = 2 * np.longdouble("3.14159265358979323846264338327950288")
    assert np.finfo(np.longdouble).eps < 2e-19               # x87 extended: cosl is the reference
    for v in vs:
        got, want = ref.cos2pi(float(v)), float(np.cos(two_pi * np.longdouble(float(v))))
        assert abs(got - want) <= 2.5e-16, (v, got, want)    # |cos| <= 1: an ulp of 1
    # exact values on the axes and the octant signs
    assert ref.cos2pi(0.0) == 1.0 and ref.cos2pi(0.5) == -1.0
    assert abs(ref.cos2pi(0.25)) < 1e-16 and abs(ref.cos2pi(0.75)) < 1e-16
    assert ref.cos2pi(0.125) > 0 and ref.cos2pi(0.375) < 0 and ref.cos2pi(0.625) < 0 and ref.cos2pi(0.875) > 0


def test_normal_deviates_are_standard_normal(ref):
    from scipy import stats
    z = np.array([ref.normal(20231204, c, i) for c in range(4) for i in range(50000)])
    n = z.size
    assert abs(z.mean()) < 4.0 / math.sqrt(n)
    assert abs(z.var() - 1.0) < 4.0 * math.sqrt(2.0 / n)
    assert abs(stats.skew(z)) < 4.0 * math.sqrt(6.0 / n)
    assert abs(stats.kurtosis(z)) < 4.0 * math.sqrt(24.0 / n)
    assert stats.kstest(z, "norm").pvalue > 1e-3
    # different curves and different seeds give different streams
    a = np.array([ref.normal(1, 0, i) for i in range(1000)])
    b = np.array([ref.normal(1, 1, i) for i in range(1000)])
    c = np.array([ref.normal(2, 0, i) for i in range(1000)])
    assert abs(np.corrcoef(a, b)[0, 1]) < 0.15 and abs(np.corrcoef(a, c)[0, 1]) < 0.15


def fixed(ref, **kw):
    """Degenerate ranges: every drawn parameter is the given number."""
    base = dict(period_lo=0.5, period_hi=0.5, ratio_lo=0.09, ratio_hi=0.09,
                duration_lo=0.001, duration_hi=1.0, sigma_lo=3e-4, sigma_hi=3e-4,
                snr_lo=6.0, snr_hi=6.0, transit_fraction=2.0, cadence=0.0125, t_start=0.0)
    base.update(kw)
    return ref.lc_params_default(**base)


def test_eq2_depth_hand_worked(ref):
    """PAPER.md:162 Eq. 2 solved for d.  n = 40,000, L/p = 0.09: n L/p = 3,600 points in
    transit, sqrt = 60; alpha = 6, sigma = 3e-4: d = 6 * 3e-4 / 60 = 3e-5."""
    prm = fixed(ref, flags=ref.LC_NO_NOISE)
    _, _, par = ref.make_light_curves(5, 3, 40000, prm)
    for row in par:
        assert row[0] == 0.5 and abs(row[1] - 0.045) < 1e-17 and row[2] == 3e-4 and row[6] == 6.0
        assert row[7] == 1.0
        assert abs(row[3] - 3e-5) < 1e-19
    # four times the points: half the depth; twice the SNR: twice the depth
    _, _, par4 = ref.make_light_curves(5, 1, 160000, prm)
    assert abs(par4[0, 3] - 1.5e-5) < 1e-19
    _, _, par2 = ref.make_light_curves(5, 1, 40000, fixed(ref, snr_lo=12.0, snr_hi=12.0, flags=ref.LC_NO_NOISE))
    assert abs(par2[0, 3] - 6e-5) < 1e-19


def test_noiseless_trapezoid_closed_forms(ref):
    """Fig. 7 / PAPER.md:170: duration L at HALF depth, short base = r * long base.  With a
    cadence far below the ramp the sampled model integrates to d * L per transit, bottoms out
    at 1 - d, and is below 1 - d/2 for L/p of the time."""
    n, cad = 200000, 0.00025                    # 50 d, 100 transits at p = 0.5
    prm = fixed(ref, cadence=cad, flags=ref.LC_NO_NOISE)
    t, f, par = ref.make_light_curves(9, 6, n, prm)
    for c in range(6):
        p, L, d, r = par[c, 0], par[c, 1], par[c, 3], par[c, 4]
        dip = 1.0 - f[c].astype(np.float64)
        assert dip.min() >= 0.0 and abs(dip.max() - d) <= 2.0 ** -24
        ntr = n * cad / p
        area = dip.sum() * cad / ntr
        assert abs(area - d * L) <= 2e-3 * d * L, (area, d * L)
        half = (dip > 0.5 * d).mean()
        assert abs(half - L / p) <= 2 * cad / p + 1e-4
        # long base 2L/(1+r): the fraction of samples touched by the transit
        touched = (dip > 2.0 ** -25).mean()
        assert abs(touched - (2 * L / (1 + r)) / p) <= 4 * cad / p + 5e-3
        # flat bottom r * long base
        flat = (dip >= d - 2.0 ** -24).mean()
        assert abs(flat - (r * 2 * L / (1 + r)) / p) <= 4 * cad / p + 5e-3
    # the transits sit at epoch + k p
    c = 0
    p, tc = par[c, 0], par[c, 5]
    deepest = t[c][np.argmax(1.0 - f[c])]
    y = (deepest - tc) / p
    assert abs(y - round(y)) * p <= par[c, 1]
    # no transit -> exactly 1
    _, f0, par0 = ref.make_light_curves(9, 2, 1000, fixed(ref, transit_fraction=0.0, flags=ref.LC_NO_NOISE))
    assert np.all(f0 == 1.0) and np.all(par0[:, 3] == 0.0) and np.all(par0[:, 7] == 0.0)


def test_table2_ranges_and_joint_rule(ref):
    """Table 2: every drawn p, L, L/p, sigma inside its range; alpha in [6, 10]
    (PAPER.md:190); r in (0, 1); epoch in [0, p); about half the curves carry a transit."""
    prm = ref.lc_params_default()
    _, _, par = ref.make_light_curves(123, 20000, 1, prm, want_times=False)
    p, L, sig, d, r, tc, al, has = par.T
    assert p.min() > 0.3 and p.max() < 1.0
    assert L.min() >= 0.03 and L.max() <= 0.09
    assert (L / p).min() > 0.04 - 1e-12 and (L / p).max() < 0.12 + 1e-12
    assert sig.min() > 1e-4 and sig.max() < 5e-4
    assert al.min() > 6.0 and al.max() < 10.0
    assert r.min() > 0.0 and r.max() < 1.0
    assert np.all(tc >= 0) and np.all(tc < p)
    assert abs(has.mean() - 0.5) < 0.02
    assert np.all((d > 0) == (has == 1.0))
    # the ranges are used, not just a corner of them
    assert p.max() - p.min() > 0.6 and sig.max() - sig.min() > 3.5e-4 and al.max() - al.min() > 3.5


def test_noise_level_and_recovered_snr(ref):
    """sigma is the per-point noise (Eq. 2's sigma), and the injected transit has the requested
    SNR: (mean out - mean in) / (sigma / sqrt(n_in)) ~ alpha up to the trapezoid's ramps."""
    n = 65536
    prm = fixed(ref, cadence=0.020433, snr_lo=40.0, snr_hi=40.0)
    t, f, par = ref.make_light_curves(77, 8, n, prm)
    prm0 = fixed(ref, cadence=0.020433, snr_lo=40.0, snr_hi=40.0, flags=ref.LC_NO_NOISE)
    _, model, _ = ref.make_light_curves(77, 8, n, prm0)
    for c in range(8):
        resid = f[c].astype(np.float64) - model[c].astype(np.float64)
        assert abs(resid.std() - par[c, 2]) < 0.02 * par[c, 2]
        assert abs(resid.mean()) < 5 * par[c, 2] / math.sqrt(n)
        dip = 1.0 - model[c].astype(np.float64)
        # matched-filter SNR of the model in white noise of this sigma
        snr = math.sqrt((dip ** 2).sum()) / par[c, 2]
        # box of depth d over n L/p points gives alpha exactly; the ramps change it by < 20 %
        assert 0.8 * 40.0 < snr < 1.1 * 40.0, snr
    # centred output: the same numbers minus one, in fp32
    prm_c = fixed(ref, cadence=0.020433, snr_lo=40.0, snr_hi=40.0, flags=ref.LC_CENTERED)
    _, fc, _ = ref.make_light_curves(77, 2, n, prm_c)
    assert np.array_equal(fc, f[:2] - np.float32(1.0))


def test_times_and_argument_checks(ref):
    prm = ref.lc_params_default(cadence=0.020433, t_start=131.5)
    t, f, _ = ref.make_light_curves(3, 2, 100, prm)
    assert np.array_equal(t[0], 131.5 + np.arange(100) * 0.020433) and np.array_equal(t[0], t[1])
    assert not np.array_equal(f[0], f[1])
    t2, f2, _ = ref.make_light_curves(3, 2, 100, prm)
    assert np.array_equal(f, f2)                                   # a pure function of the seed
    _, f3, _ = ref.make_light_curves(4, 2, 100, prm)
    assert not np.array_equal(f, f3)
    # a longer series starts with the shorter one's noise (counter = sample index); only the
    # depth (Eq. 2 has n in it) changes
    _, f_long, _ = ref.make_light_curves(3, 1, 200, ref.lc_params_default(transit_fraction=0.0))
    _, f_short, _ = ref.make_light_curves(3, 1, 100, ref.lc_params_default(transit_fraction=0.0))
    assert np.array_equal(f_long[0, :100], f_short[0])
    with pytest.raises(ValueError):
        ref.make_light_curves(3, 1, 10, ref.lc_params_default(cadence=0.0))
    with pytest.raises(ValueError):
        ref.make_light_curves(3, 1, 10, ref.lc_params_default(period_lo=1.0, period_hi=0.3))
    assert ref.make_light_curves(3, 0, 10, prm)[1].shape == (0, 10)
