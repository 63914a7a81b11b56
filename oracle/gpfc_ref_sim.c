/*
 * gpfc_ref_sim.c -- CPU ORACLE for the synthetic light-curve generator
 * (PAPER.md 2.6 "Light Curve Simulation": Eq. 2 :162,
 * parameter ranges :166-170, Table 2 :176-180, trapezoid model :170, Fig. 7 :188).
 *
 * THIS FILE IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as gpfc_ref.c:
 * only tests/, __graft_entry__.smoke() and bench.py's oracle legs may use it; it
 * shares no code, header, table or helper with paper_2312_02063_b200/csrc/).
 *
 * A generator draws random numbers, so "the same result" needs the same
 * generator on both sides: include/gpfc.h ("Generator specification") fixes a
 * counter-based one, and this file and csrc/simulate.cu each implement it from
 * that text.  In short, with Philox4x32-10 (Salmon et al. 2011) keyed by the
 * seed, U(x) = (x + 1/2) 2^-32 for a 32-bit word x, and every fp64 operation
 * below rounded once, in the order written (built with -ffp-contract=off):
 *
 *   per curve c   B0 = philox(0, 0, c, 0): sigma, r, epoch fraction, alpha
 *                 B1 = philox(0, 1, c, 0): transit yes/no
 *                 Bk = philox(k, 2, c, 0), k = 0..63: (p, L/p) redrawn until the
 *                      duration L = (L/p) p lies in its own range (Table 2 gives
 *                      ranges for p, L and L/p and no joint law: reading R21)
 *                 depth d = alpha sigma / sqrt(n L / p)            (Eq. 2 solved for d)
 *                 trapezoid: duration L at half depth, short base / long base = r
 *                       => long base 2L/(1+r), short base r times that
 *   per sample i  philox(i, 0, c, 1) -> u1 (52 bits), u2 (32 bits);
 *                 z = sqrt(-2 ln u1) cos(2 pi u2)                  (Box-Muller)
 *                 t = t_start + i cadence
 *                 flux = (1 + sigma z) - d shape(t),   stored as fp32
 *
 * ln and cos are the short series written out below (not libm), so that the
 * CUDA path can reproduce them operation by operation; they are pinned against
 * libm in tests/test_oracle_sim.py.
 *
 * Pins (tests/test_oracle_sim.py): the Random123 known-answer vectors of
 * philox4x32-10; ln / cos against libm to a few ulp; moments and a
 * Kolmogorov-Smirnov test of z; Eq. 2 on hand-worked numbers (n L/p = 3600);
 * the noiseless trapezoid's area d L per transit, its floor 1 - d and its
 * half-depth width L; every drawn parameter inside Table 2's ranges; the
 * measured SNR of the injected transit.
 */
#include <math.h>
#include <stdint.h>
#include <string.h>

#define GPFC_REF_OK 0
#define GPFC_REF_ERR_INVALID_ARG 1

#define GPFC_REF_LC_CENTERED 1   /* store flux - 1 (fp32 subtraction after the fp32 rounding) */
#define GPFC_REF_LC_NO_NOISE 2   /* leave the Gaussian term out (the transit model alone)     */

typedef struct {
    double period_lo, period_hi;       /* p,     Table 2: (0.3, 1.0) d            */
    double duration_lo, duration_hi;   /* L,     Table 2: (0.03, 0.09) d          */
    double ratio_lo, ratio_hi;         /* L / p, Table 2: (0.04, 0.12)            */
    double sigma_lo, sigma_hi;         /* sigma, Table 2: (0.0001, 0.0005)        */
    double snr_lo, snr_hi;             /* alpha: [6, 10]            */
    double transit_fraction;           /* share of the curves that carry a transit */
    double cadence, t_start;           /* t_i = t_start + i cadence               */
    int32_t flags;
    int32_t reserved;
} gpfc_ref_lc_params;

/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): ten rounds of
 *   (c0, c1, c2, c3) <- (hi(M1 c2) ^ c1 ^ k0, lo(M1 c2), hi(M0 c0) ^ c3 ^ k1, lo(M0 c0))
 * with the key bumped by the Weyl constants after every round. */
void gpfc_ref_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

static void philox_at(uint64_t seed, uint32_t w0, uint32_t w1, uint32_t w2, uint32_t w3,
                      uint32_t out[4])
{
    uint32_t ctr[4] = {w0, w1, w2, w3};
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    gpfc_ref_philox4x32_10(ctr, key, out);
}

/* U(x) = (x + 1/2) 2^-32 in (0, 1): exact in fp64 */
double gpfc_ref_u32_to_unit(uint32_t x)
{
    return ((double)x + 0.5) * (1.0 / 4294967296.0);
}

/* 52-bit uniform from two words: ((x0 2^20 + (x1 >> 12)) + 1/2) 2^-52: exact in fp64 */
double gpfc_ref_u52_to_unit(uint32_t x0, uint32_t x1)
{
    double hi = (double)x0 * 1048576.0 + (double)(x1 >> 12);
    return (hi + 0.5) * (1.0 / 4503599627370496.0);
}

/* ln u for a normal positive u: u = m 2^e with m in [sqrt(1/2), sqrt(2)),
 * s = (m - 1)/(m + 1), ln m = 2 s (1 + s^2/3 + s^4/5 + ... + s^22/23) (|s| < 0.1716:
 * the first term left out is below 2e-19), ln u = e ln 2 + ln m. */
double gpfc_ref_ln(double u)
{
    uint64_t bits;
    memcpy(&bits, &u, 8);
    int e = (int)((bits >> 52) & 0x7ff) - 1022;
    bits = (bits & 0x000fffffffffffffull) | 0x3fe0000000000000ull;
    double m;
    memcpy(&m, &bits, 8);                 /* m in [1/2, 1) */
    if (m < 0.70710678118654752) {
        m = m * 2.0;
        e = e - 1;
    }
    double s = (m - 1.0) / (m + 1.0);
    double z = s * s;
    double P = 1.0 / 23.0;
    P = P * z + 1.0 / 21.0;
    P = P * z + 1.0 / 19.0;
    P = P * z + 1.0 / 17.0;
    P = P * z + 1.0 / 15.0;
    P = P * z + 1.0 / 13.0;
    P = P * z + 1.0 / 11.0;
    P = P * z + 1.0 / 9.0;
    P = P * z + 1.0 / 7.0;
    P = P * z + 1.0 / 5.0;
    P = P * z + 1.0 / 3.0;
    P = P * z + 1.0;
    double t1 = (double)e * 0.69314718055994531;
    double t2 = 2.0 * (s * P);
    return t1 + t2;
}

/* cos(2 pi v) for v in [0, 1): w = 8 v = k + f (octant k, exact), the angle inside the
 * octant measured from the nearer axis is theta = g pi/4 with g = f (k even) or 1 - f
 * (k odd), and the value is +-sin(theta) or +-cos(theta) by Taylor series to theta^15 /
 * theta^16 (theta <= pi/4: truncation below 5e-17). */
double gpfc_ref_cos2pi(double v)
{
    double w = v * 8.0;
    double kf = floor(w);
    int k = (int)kf & 7;
    double f = w - kf;
    double g = (k & 1) ? (1.0 - f) : f;
    double th = g * 0.78539816339744831;
    double z = th * th;
    double val;
    if (((k + 1) >> 1) & 1) {             /* octants 1, 2, 5, 6: sine */
        double S = -1.0 / 1307674368000.0;
        S = S * z + 1.0 / 6227020800.0;
        S = S * z - 1.0 / 39916800.0;
        S = S * z + 1.0 / 362880.0;
        S = S * z - 1.0 / 5040.0;
        S = S * z + 1.0 / 120.0;
        S = S * z - 1.0 / 6.0;
        S = S * z + 1.0;
        val = th * S;
    } else {                              /* octants 0, 3, 4, 7: cosine */
        double C = 1.0 / 20922789888000.0;
        C = C * z - 1.0 / 87178291200.0;
        C = C * z + 1.0 / 479001600.0;
        C = C * z - 1.0 / 3628800.0;
        C = C * z + 1.0 / 40320.0;
        C = C * z - 1.0 / 720.0;
        C = C * z + 1.0 / 24.0;
        C = C * z - 0.5;
        C = C * z + 1.0;
        val = C;
    }
    /* sign: cos(2 pi v) is negative in octants 2..5 */
    return (k >= 2 && k <= 5) ? -val : val;
}

/* standard normal of sample i of curve c (Box-Muller, one value per counter) */
double gpfc_ref_normal(uint64_t seed, uint32_t curve, uint32_t i)
{
    uint32_t x[4];
    philox_at(seed, i, 0u, curve, 1u, x);
    double u1 = gpfc_ref_u52_to_unit(x[0], x[1]);
    double u2 = gpfc_ref_u32_to_unit(x[2]);
    double t = -2.0 * gpfc_ref_ln(u1);
    return sqrt(t) * gpfc_ref_cos2pi(u2);
}

typedef struct {
    double p, L, sigma, depth, r, tc, alpha, has_transit;
    double half14, half23, ramp;
} curve_params;

static double lerp_u(double lo, double hi, uint32_t x)
{
    return lo + (hi - lo) * gpfc_ref_u32_to_unit(x);
}

/* the parameters of curve c (Table 2; reading R21 for the joint law) */
static void draw_curve(uint64_t seed, uint32_t c, int64_t n, const gpfc_ref_lc_params *prm,
                       curve_params *cp)
{
    uint32_t b[4];
    philox_at(seed, 0u, 0u, c, 0u, b);
    cp->sigma = lerp_u(prm->sigma_lo, prm->sigma_hi, b[0]);
    cp->r = gpfc_ref_u32_to_unit(b[1]);
    double efrac = gpfc_ref_u32_to_unit(b[2]);
    cp->alpha = lerp_u(prm->snr_lo, prm->snr_hi, b[3]);
    philox_at(seed, 0u, 1u, c, 0u, b);
    cp->has_transit = (gpfc_ref_u32_to_unit(b[0]) < prm->transit_fraction) ? 1.0 : 0.0;
    double p = 0.0, L = 0.0;
    for (uint32_t k = 0; k < 64; ++k) {
        philox_at(seed, k, 2u, c, 0u, b);
        p = lerp_u(prm->period_lo, prm->period_hi, b[0]);
        double ratio = lerp_u(prm->ratio_lo, prm->ratio_hi, b[1]);
        L = ratio * p;
        if (L >= prm->duration_lo && L <= prm->duration_hi) break;
        if (k == 63) {                    /* never seen with Table 2's ranges: clamp */
            if (L < prm->duration_lo) L = prm->duration_lo;
            if (L > prm->duration_hi) L = prm->duration_hi;
        }
    }
    cp->p = p;
    cp->L = L;
    cp->tc = efrac * p;
    /* Eq. 2 solved for the depth: d = alpha sigma / sqrt(n L / p) */
    double npts = ((double)n * L) / p;
    cp->depth = (cp->has_transit != 0.0) ? (cp->alpha * cp->sigma) / sqrt(npts) : 0.0;
    /* trapezoid: (long + short)/2 = L, short = r long */
    double t14 = (2.0 * L) / (1.0 + cp->r);
    double t23 = cp->r * t14;
    cp->half14 = 0.5 * t14;
    cp->half23 = 0.5 * t23;
    cp->ramp = cp->half14 - cp->half23;
}

/* trapezoid of unit depth at time t: 1 on the short base, 0 outside the long base */
static double shape_at(double t, const curve_params *cp)
{
    double y = (t - cp->tc) / cp->p;
    y = y - floor(y + 0.5);               /* in [-1/2, 1/2): phase from the nearest mid-transit */
    double x = fabs(y) * cp->p;
    if (x <= cp->half23) return 1.0;
    if (x >= cp->half14) return 0.0;
    return (cp->half14 - x) / cp->ramp;
}

int gpfc_ref_lc_params_default(gpfc_ref_lc_params *prm)
{
    if (!prm) return GPFC_REF_ERR_INVALID_ARG;
    memset(prm, 0, sizeof(*prm));
    prm->period_lo = 0.3;    prm->period_hi = 1.0;       /* Table 2 */
    prm->duration_lo = 0.03; prm->duration_hi = 0.09;
    prm->ratio_lo = 0.04;    prm->ratio_hi = 0.12;
    prm->sigma_lo = 0.0001;  prm->sigma_hi = 0.0005;
    prm->snr_lo = 6.0;       prm->snr_hi = 10.0;
    prm->transit_fraction = 0.5;                         /* half and half */
    prm->cadence = 0.020433; prm->t_start = 0.0;         /* Kepler long cadence, reading R16 */
    prm->flags = 0;
    return GPFC_REF_OK;
}

/*
 * times  [ncurves][n] fp64 or NULL, flux [ncurves][n] fp32,
 * params_out [ncurves][8] fp64 or NULL: {p, L, sigma, depth (0 without a transit), r,
 * mid-transit epoch tc, alpha, 1.0 / 0.0 = carries a transit}.
 */
int gpfc_ref_make_light_curves(uint64_t seed, int64_t ncurves, int64_t n,
                               const gpfc_ref_lc_params *prm, double *times, float *flux,
                               double *params_out)
{
    if (ncurves < 0 || n < 0 || !prm) return GPFC_REF_ERR_INVALID_ARG;
    if (ncurves > 0 && n > 0 && !flux) return GPFC_REF_ERR_INVALID_ARG;
    if (ncurves > 4294967295ll || n > 4294967295ll) return GPFC_REF_ERR_INVALID_ARG;
    if (!(prm->period_lo > 0.0) || !(prm->period_hi >= prm->period_lo) ||
        !(prm->duration_lo > 0.0) || !(prm->duration_hi >= prm->duration_lo) ||
        !(prm->ratio_lo > 0.0) || !(prm->ratio_hi >= prm->ratio_lo) ||
        !(prm->sigma_lo >= 0.0) || !(prm->sigma_hi >= prm->sigma_lo) ||
        !(prm->snr_hi >= prm->snr_lo) || !(prm->cadence > 0.0))
        return GPFC_REF_ERR_INVALID_ARG;
    for (int64_t c = 0; c < ncurves; ++c) {
        curve_params cp;
        draw_curve(seed, (uint32_t)c, n, prm, &cp);
        if (params_out) {
            double *o = params_out + c * 8;
            o[0] = cp.p; o[1] = cp.L; o[2] = cp.sigma; o[3] = cp.depth;
            o[4] = cp.r; o[5] = cp.tc; o[6] = cp.alpha; o[7] = cp.has_transit;
        }
        for (int64_t i = 0; i < n; ++i) {
            double t = prm->t_start + (double)i * prm->cadence;
            double f = 1.0;
            if (!(prm->flags & GPFC_REF_LC_NO_NOISE))
                f = f + cp.sigma * gpfc_ref_normal(seed, (uint32_t)c, (uint32_t)i);
            if (cp.has_transit != 0.0) f = f - cp.depth * shape_at(t, &cp);
            float f32 = (float)f;
            if (prm->flags & GPFC_REF_LC_CENTERED) f32 = f32 - 1.0f;
            if (times) times[c * n + i] = t;
            flux[c * n + i] = f32;
        }
    }
    return GPFC_REF_OK;
}
