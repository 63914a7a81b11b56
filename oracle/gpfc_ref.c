/*
 * gpfc_ref.c -- CPU ORACLE for the GPFC fold + noise-normalisation hot path.
 *
 * THIS FILE IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, the smoke
 * check in __graft_entry__.py and bench.py's cpu_baseline / --impl reference
 * legs may build, load or call it.  It shares no code, header, table or
 * helper with the CUDA path under paper_2312_02063_b200/csrc/ and neither
 * includes the other.
 *
 * What it is: the plain definition of what the path computes, written out in
 * the paper's order, in fp64, one sample at a time, with no blocking, fusion
 * or reordering.  Source of every step (PAPER.md = arXiv 2312.02063):
 *
 *   Eq. 1, PAPER.md:53-57   N_sample = N_o T / L, 100,000 periods uniformly
 *                           sampled in [0.2, 1.0] d          -> n_sample, grid
 *   Sec. 2.3, PAPER.md:87(1), :111 "First"   modular residual of each
 *                           timestamp by the folding period  -> phase
 *   Sec. 2.3, "Secondly", Fig. 4(b) :152  map the residual
 *                           to equally spaced bins           -> bin index
 *   Sec. 2.3, "Thirdly"   per-bin count and flux sum
 *   Sec. 2.3, "Lastly"    bin mean = sum / count
 *   Sec. 2.3, PAPER.md:111 "Fourthly", :105   equal-count merge of the
 *                           intermediary bins to the final bins (NEXT row)
 *   Sec. 2.1, PAPER.md:63   scale each folded result to a standard deviation
 *                           of 1.0 while maintaining its mean -> normalise
 *
 * Readings taken where the paper is silent are the ones listed in DESIGN.md
 * ("Readings of the paper"), numbered R1..; they are quoted at the point of
 * use below.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): the hand-built dyadic
 * vectors and paper values under tests/golden/, exact-rational brute force,
 * invariants (count conservation, sum conservation, period-shift and
 * permutation invariance, nb -> nb/2 pair merge), collapse closed forms, the
 * noiseless-box closed form, sqrt(N) noise attenuation, and
 * mean/std invariants plus a numpy cross-check for the normalisation.
 * gpfc_ref_two_tier_merge ("Fourthly"): pinned by hand-worked
 * merges with a fractional number of points per output bin, fine bins cut by
 * one and by three boundaries and empty fine bins (tests/golden/
 * hand_vectors.json "two_tier_merge"), the paper's own 65,536 / 256 = 256
 * points per bin, an independent piecewise-linear
 * interpolation of the cumulative flux in cumulative count, count/sum
 * conservation and the sort-based fold on tie-free inputs.  The pro-rata split
 * of a boundary bin is reading R18 (the paper does not say how a split bin's
 * flux is shared).
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fno-fast-math -shared -fPIC
 * (no FMA contraction, so every operation below rounds once, as written).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define GPFC_REF_OK 0
#define GPFC_REF_ERR_INVALID_ARG 1

/* mode_flags: bit 0 = spacing (0 uniform in frequency, 1 uniform in period),
 * bit 1 = endpoint handling (0 inclusive: divisor Np-1, 2 exclusive: divisor Np). */
#define GPFC_REF_GRID_UNIFORM_PERIOD 1
#define GPFC_REF_GRID_ENDPOINT_EXCLUSIVE 2

/* Eq. 1: N_sample = N_o * T / L. */
double gpfc_ref_n_sample(double n_o, double t_window, double l_width)
{
    return n_o * t_window / l_width;
}

/*
 * Trial-period grid ("uniformly sample 100,000 periods within
 * [0.2, 1.0] days"; BASELINE configs: uniform in frequency).
 * R11/R12: both spacings; endpoints inclusive by default (divisor D = Np-1),
 * exclusive with the flag (D = Np); multiply before divide; index ascending in
 * frequency (period descending) in frequency mode, ascending in period in
 * period mode; Np == 1 gives the start point (pmax in frequency mode, pmin in
 * period mode).
 */
int gpfc_ref_make_period_grid(double pmin, double pmax, int64_t nperiods,
                              int mode_flags, double *periods_out)
{
    if (nperiods < 0 || !(pmin > 0.0) || !(pmax >= pmin) || !isfinite(pmax))
        return GPFC_REF_ERR_INVALID_ARG;
    if (nperiods == 0)
        return GPFC_REF_OK;
    if (!periods_out)
        return GPFC_REF_ERR_INVALID_ARG;
    int64_t d = (mode_flags & GPFC_REF_GRID_ENDPOINT_EXCLUSIVE) ? nperiods : nperiods - 1;
    if (d < 1)
        d = 1;
    double dd = (double)d;
    if (mode_flags & GPFC_REF_GRID_UNIFORM_PERIOD) {
        double span = pmax - pmin;
        for (int64_t j = 0; j < nperiods; ++j) {
            double num = span * (double)j;
            double step = num / dd;
            periods_out[j] = pmin + step;
        }
    } else {
        double fmin = 1.0 / pmax;
        double fmax = 1.0 / pmin;
        double span = fmax - fmin;
        for (int64_t j = 0; j < nperiods; ++j) {
            double num = span * (double)j;
            double step = num / dd;
            double f = fmin + step;
            periods_out[j] = 1.0 / f;
        }
    }
    return GPFC_REF_OK;
}

/*
 * Steps 1-2 for one sample ("First", "Secondly"):
 *   u   = t - t0                     R3: t0 subtracted first, one rounding
 *   x   = u / P                      R2: IEEE division, one rounding
 *   phi = x - floor(x)               in [0, 1]; equals 1.0 only when a tiny
 *                                    negative x rounds up in x + 1
 *   k   = trunc(phi * nb)            R4: half-open bins [k/nb, (k+1)/nb)
 *   k   = nb-1 if k >= nb            R4: phi == 1.0 belongs to the last bin
 * R20: if u / P is not finite (a denormal-small P) the sample has no phase: -1, and the
 * fold skips it like a non-finite sample (R13).
 */
static int64_t bin_of(double t, double t0, double period, int nb)
{
    double u = t - t0;
    double x = u / period;
    if (!isfinite(x))
        return -1;   /* R20: the quotient overflows (period far below |u| / DBL_MAX): skip */
    double phi = x - floor(x);
    double scaled = phi * (double)nb;
    int64_t k = (int64_t)scaled;
    if (k >= nb)
        k = nb - 1;
    return k;
}

int gpfc_ref_bin_index(const double *times, int64_t n, double period, int nb,
                       double t0, int32_t *bins_out)
{
    if (n < 0 || nb < 1 || (n > 0 && (!times || !bins_out)))
        return GPFC_REF_ERR_INVALID_ARG;
    for (int64_t i = 0; i < n; ++i) {
        if (!isfinite(times[i]) || !(isfinite(period) && period > 0.0))
            bins_out[i] = -1;
        else
            bins_out[i] = (int32_t)bin_of(times[i], t0, period, nb);
    }
    return GPFC_REF_OK;
}

/*
 * Steps 1-3: for every trial period, per-bin flux sum and
 * count.  R5: sums accumulate in fp64 in sample order; out_sum is the fp32
 * rounding of that, out_sum64 (optional) keeps it.  R13: a sample with a
 * non-finite time or flux is skipped.  A period that is not finite and
 * positive yields an all-zero row.  Output [nperiods][nbins] row-major.
 */
int gpfc_ref_fold(const double *times, const float *flux, int64_t n,
                  const double *periods, int64_t nperiods, int nbins, double t0,
                  float *out_sum, uint32_t *out_count, double *out_sum64)
{
    if (n < 0 || nperiods < 0 || nbins < 1)
        return GPFC_REF_ERR_INVALID_ARG;
    if (n > 0 && (!times || !flux))
        return GPFC_REF_ERR_INVALID_ARG;
    if (nperiods > 0 && !periods)
        return GPFC_REF_ERR_INVALID_ARG;
    double *s = (double *)malloc(sizeof(double) * (size_t)nbins);
    uint32_t *c = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)nbins);
    if (!s || !c) {
        free(s);
        free(c);
        return GPFC_REF_ERR_INVALID_ARG;
    }
    for (int64_t j = 0; j < nperiods; ++j) {
        double period = periods[j];
        for (int k = 0; k < nbins; ++k) {
            s[k] = 0.0;
            c[k] = 0;
        }
        if (isfinite(period) && period > 0.0) {
            for (int64_t i = 0; i < n; ++i) {
                if (!isfinite(times[i]) || !isfinite(flux[i]))
                    continue;
                int64_t k = bin_of(times[i], t0, period, nbins);
                if (k < 0)
                    continue;
                s[k] += (double)flux[i];
                c[k] += 1;
            }
        }
        for (int k = 0; k < nbins; ++k) {
            size_t o = (size_t)j * (size_t)nbins + (size_t)k;
            if (out_sum)
                out_sum[o] = (float)s[k];
            if (out_count)
                out_count[o] = c[k];
            if (out_sum64)
                out_sum64[o] = s[k];
        }
    }
    free(s);
    free(c);
    return GPFC_REF_OK;
}

/*
 * Step 5 + noise normalisation of one profile (PAPER.md:111 "Lastly"; :63
 * "scaling the folded flux values to a standard deviation of 1.0, while
 * maintaining the mean of the folded results").
 *   m[k] = sum[k] / count[k]                    for non-empty bins
 *   mu   = (1/K) sum_k m[k]                     K = number of non-empty bins
 *   s    = sqrt((1/K) sum_k (m[k] - mu)^2)      R7: population std (ddof 0),
 *                                               unweighted, R9: signal included
 *   out[k] = mu + (m[k] - mu) / s               R8
 *   R6: an empty bin is left out of mu and s and gets the value mu.
 *   R10: K == 0 -> all zeros; K < 2 or s == 0 -> mu everywhere.
 */
static void normalize_profile(const double *sum, const uint32_t *count, int nb,
                              double *out)
{
    int64_t kk = 0;
    double acc = 0.0;
    for (int k = 0; k < nb; ++k) {
        if (count[k] > 0) {
            double m = sum[k] / (double)count[k];
            acc += m;
            kk += 1;
        }
    }
    if (kk == 0) {
        for (int k = 0; k < nb; ++k)
            out[k] = 0.0;
        return;
    }
    double mu = acc / (double)kk;
    double vacc = 0.0;
    for (int k = 0; k < nb; ++k) {
        if (count[k] > 0) {
            double m = sum[k] / (double)count[k];
            double d = m - mu;
            vacc += d * d;
        }
    }
    double var = vacc / (double)kk;
    double s = sqrt(var);
    if (kk < 2 || !(s > 0.0)) {
        for (int k = 0; k < nb; ++k)
            out[k] = mu;
        return;
    }
    for (int k = 0; k < nb; ++k) {
        if (count[k] > 0) {
            double m = sum[k] / (double)count[k];
            double d = m - mu;
            out[k] = mu + d / s;
        } else {
            out[k] = mu;
        }
    }
}

static int normalize_any(const float *sum32, const double *sum64,
                         const uint32_t *count, int64_t nprofiles, int nbins,
                         float *out_norm, double *out_norm64)
{
    if (nprofiles < 0 || nbins < 1)
        return GPFC_REF_ERR_INVALID_ARG;
    if (nprofiles > 0 && (!(sum32 || sum64) || !count))
        return GPFC_REF_ERR_INVALID_ARG;
    double *s = (double *)malloc(sizeof(double) * (size_t)nbins);
    double *o = (double *)malloc(sizeof(double) * (size_t)nbins);
    if (!s || !o) {
        free(s);
        free(o);
        return GPFC_REF_ERR_INVALID_ARG;
    }
    for (int64_t p = 0; p < nprofiles; ++p) {
        size_t base = (size_t)p * (size_t)nbins;
        for (int k = 0; k < nbins; ++k)
            s[k] = sum64 ? sum64[base + k] : (double)sum32[base + k];
        normalize_profile(s, count + base, nbins, o);
        for (int k = 0; k < nbins; ++k) {
            if (out_norm)
                out_norm[base + k] = (float)o[k];
            if (out_norm64)
                out_norm64[base + k] = o[k];
        }
    }
    free(s);
    free(o);
    return GPFC_REF_OK;
}

/* Normalise profiles given as fp32 sums + counts (the library's gpfc_normalize
 * inputs). */
int gpfc_ref_normalize(const float *sum, const uint32_t *count, int64_t nprofiles,
                       int nbins, float *out_norm, double *out_norm64)
{
    return normalize_any(sum, NULL, count, nprofiles, nbins, out_norm, out_norm64);
}

/* Same, from the fold's fp64 sums (what the fused fold + normalise computes). */
int gpfc_ref_normalize_f64(const double *sum64, const uint32_t *count,
                           int64_t nprofiles, int nbins, float *out_norm,
                           double *out_norm64)
{
    return normalize_any(NULL, sum64, count, nprofiles, nbins, out_norm, out_norm64);
}

/*
 * Batched fold (+ optional normalisation) over ncurves curves stored back to
 * back: curve c is samples offsets[c] .. offsets[c+1]-1, folded with t0[c]
 * (0.0 when t0 is NULL) over the shared period grid.  Outputs
 * [ncurves][nperiods][nbins]; any may be NULL.  The normalised profile is
 * computed from the fp64 sums (not from their fp32 roundings).
 */
int gpfc_ref_fold_batch(const double *times, const float *flux,
                        const int64_t *offsets, int64_t ncurves,
                        const double *periods, int64_t nperiods, int nbins,
                        const double *t0, float *out_sum, uint32_t *out_count,
                        float *out_norm, double *out_sum64, double *out_norm64)
{
    if (ncurves < 0 || nperiods < 0 || nbins < 1)
        return GPFC_REF_ERR_INVALID_ARG;
    if (ncurves > 0 && !offsets)
        return GPFC_REF_ERR_INVALID_ARG;
    size_t slab = (size_t)nperiods * (size_t)nbins;
    int need_norm = (out_norm || out_norm64);
    double *s64 = NULL;
    uint32_t *cnt = NULL;
    if (slab > 0) {
        s64 = (double *)malloc(sizeof(double) * slab);
        cnt = (uint32_t *)malloc(sizeof(uint32_t) * slab);
        if (!s64 || !cnt) {
            free(s64);
            free(cnt);
            return GPFC_REF_ERR_INVALID_ARG;
        }
    }
    int rc = GPFC_REF_OK;
    for (int64_t c = 0; c < ncurves && rc == GPFC_REF_OK; ++c) {
        int64_t lo = offsets[c], hi = offsets[c + 1];
        if (hi < lo) {
            rc = GPFC_REF_ERR_INVALID_ARG;
            break;
        }
        size_t o = (size_t)c * slab;
        rc = gpfc_ref_fold(times + lo, flux + lo, hi - lo, periods, nperiods, nbins,
                           t0 ? t0[c] : 0.0, out_sum ? out_sum + o : NULL, cnt, s64);
        if (rc != GPFC_REF_OK)
            break;
        if (out_count && slab)
            memcpy(out_count + o, cnt, sizeof(uint32_t) * slab);
        if (out_sum64 && slab)
            memcpy(out_sum64 + o, s64, sizeof(double) * slab);
        if (need_norm)
            rc = gpfc_ref_normalize_f64(s64, cnt, nperiods, nbins,
                                        out_norm ? out_norm + o : NULL,
                                        out_norm64 ? out_norm64 + o : NULL);
    }
    free(s64);
    free(cnt);
    return rc;
}

/*
 * Step 4 of PAPER.md:111 --
 * "scan the [fine] bins from left to right, combine the adjacent bins, and
 * split bins on the boundary as needed, to generate a final layout of [nb2]
 * bins ... each ... containing the same number of flux data points".
 * R18 (paper silent on how a split bin's flux is shared): a fine bin's points
 * are taken to carry its mean flux each, so a split takes flux pro rata by
 * count; i.e. the cumulative sum is linear in cumulative count inside a fine
 * bin.  Output bin b holds exactly N/nb2 points (N = total count, fractional
 * allowed): out_sum[b] = Scum((b+1) N / nb2) - Scum(b N / nb2), and
 * out_mean[b] = out_sum[b] / (N / nb2).  N == 0 gives zeros.
 */
int gpfc_ref_two_tier_merge(const double *fine_sum, const uint32_t *fine_count,
                            int nb1, int nb2, double *out_sum, double *out_mean)
{
    if (nb1 < 1 || nb2 < 1 || !fine_sum || !fine_count)
        return GPFC_REF_ERR_INVALID_ARG;
    double total = 0.0;
    for (int k = 0; k < nb1; ++k)
        total += (double)fine_count[k];
    if (!(total > 0.0)) {
        for (int b = 0; b < nb2; ++b) {
            if (out_sum)
                out_sum[b] = 0.0;
            if (out_mean)
                out_mean[b] = 0.0;
        }
        return GPFC_REF_OK;
    }
    double per = total / (double)nb2;
    int k = 0;            /* current fine bin */
    double c_before = 0.0; /* points in fine bins < k */
    double s_before = 0.0; /* flux in fine bins < k */
    double s_prev = 0.0;   /* Scum at the previous boundary */
    for (int b = 0; b < nb2; ++b) {
        double target = (b == nb2 - 1) ? total : per * (double)(b + 1);
        /* advance to the fine bin that contains cumulative count `target` */
        while (k < nb1 - 1 && c_before + (double)fine_count[k] < target) {
            c_before += (double)fine_count[k];
            s_before += fine_sum[k];
            ++k;
        }
        double ck = (double)fine_count[k];
        double frac = (ck > 0.0) ? (target - c_before) / ck : 0.0;
        if (frac > 1.0)
            frac = 1.0;
        if (frac < 0.0)
            frac = 0.0;
        double s_here = s_before + frac * fine_sum[k];
        double sb = s_here - s_prev;
        s_prev = s_here;
        if (out_sum)
            out_sum[b] = sb;
        if (out_mean)
            out_mean[b] = sb / per;
    }
    return GPFC_REF_OK;
}
