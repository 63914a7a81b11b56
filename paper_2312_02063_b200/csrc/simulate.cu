// Synthetic light curves on the device: white Gaussian noise around 1 plus a periodic
// trapezoidal transit whose depth follows from a requested SNR (PAPER.md 2.6: Eq. 2 :162,
// Table 2 :176-180, trapezoid :170, Fig. 7 :188).  include/gpfc.h ("Generator specification")
// fixes every operation; this file follows that text with round-to-nearest intrinsics, so
// nothing can be contracted into an FMA.
//
// Two kernels: sim_params_kernel (one thread per curve: the Table 2 draws, Eq. 2, the
// trapezoid's bases) and sim_samples_kernel (one thread per sample, four samples per thread:
// Philox4x32-10, Box-Muller, the transit model; coalesced 8-byte and 4-byte stores).  The
// sample kernel is bound by its fp64 arithmetic (~150 fp64 operations and 70 integer
// multiplies per sample against 12 bytes written), DESIGN.md 6.6.
#include "common.cuh"

namespace gpfc {

namespace {

constexpr int SIM_THREADS = 256;
constexpr int SIM_PER_THREAD = 4;
constexpr int SIM_CHUNK = SIM_THREADS * SIM_PER_THREAD;

// per-curve constants of the sample kernel
struct SimCurve {
    double p, tc, sigma, depth, half14, half23, ramp;
    int has_transit;
    int pad;
};

struct SimRanges {
    double period_lo, period_hi, duration_lo, duration_hi, ratio_lo, ratio_hi;
    double sigma_lo, sigma_hi, snr_lo, snr_hi, transit_fraction, cadence, t_start;
    int flags;
};

struct Words {
    unsigned x0, x1, x2, x3;
};

// Philox4x32-10: ten rounds, the key bumped by the Weyl constants after each
__device__ __forceinline__ Words philox10(unsigned c0, unsigned c1, unsigned c2, unsigned c3,
                                          unsigned k0, unsigned k1)
{
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const unsigned hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const unsigned hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const unsigned n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0;
        c1 = lo1;
        c2 = n2;
        c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return Words{c0, c1, c2, c3};
}

__device__ __forceinline__ double unit32(unsigned x)
{
    return __dmul_rn(__dadd_rn((double)x, 0.5), 1.0 / 4294967296.0);
}

__device__ __forceinline__ double unit52(unsigned x0, unsigned x1)
{
    const double hi = __dadd_rn(__dmul_rn((double)x0, 1048576.0), (double)(x1 >> 12));
    return __dmul_rn(__dadd_rn(hi, 0.5), 1.0 / 4503599627370496.0);
}

__device__ __forceinline__ double between(double lo, double hi, unsigned x)
{
    return __dadd_rn(lo, __dmul_rn(__dsub_rn(hi, lo), unit32(x)));
}

// ln u, u normal and positive: u = m 2^e, m in [sqrt(1/2), sqrt(2)); atanh series to s^23
__device__ __forceinline__ double sim_ln(double u)
{
    unsigned long long bits = (unsigned long long)__double_as_longlong(u);
    int e = (int)((bits >> 52) & 0x7ffull) - 1022;
    bits = (bits & 0x000fffffffffffffull) | 0x3fe0000000000000ull;
    double m = __longlong_as_double((long long)bits);
    if (m < 0.70710678118654752) {
        m = __dmul_rn(m, 2.0);
        e -= 1;
    }
    const double s = __ddiv_rn(__dsub_rn(m, 1.0), __dadd_rn(m, 1.0));
    const double z = __dmul_rn(s, s);
    double P = 1.0 / 23.0;
    P = __dadd_rn(__dmul_rn(P, z), 1.0 / 21.0);
    P = __dadd_rn(__dmul_rn(P, z), 1.0 / 19.0);
    P = __dadd_rn(__dmul_rn(P, z), 1.0 / 17.0);
    P = __dadd_rn(__dmul_rn(P, z), 1.0 / 15.0);
    P = __dadd_rn(__dmul_rn(P, z), 1.0 / 13.0);
    P = __dadd_rn(__dmul_rn(P, z), 1.0 / 11.0);
    P = __dadd_rn(__dmul_rn(P, z), 1.0 / 9.0);
    P = __dadd_rn(__dmul_rn(P, z), 1.0 / 7.0);
    P = __dadd_rn(__dmul_rn(P, z), 1.0 / 5.0);
    P = __dadd_rn(__dmul_rn(P, z), 1.0 / 3.0);
    P = __dadd_rn(__dmul_rn(P, z), 1.0);
    const double t1 = __dmul_rn((double)e, 0.69314718055994531);
    const double t2 = __dmul_rn(2.0, __dmul_rn(s, P));
    return __dadd_rn(t1, t2);
}

// cos(2 pi v), v in [0, 1): octant k of 8 v, angle from the nearer axis, Taylor series
__device__ __forceinline__ double sim_cos2pi(double v)
{
    const double w = __dmul_rn(v, 8.0);
    const double kf = floor(w);
    const int k = (int)kf & 7;
    const double f = __dsub_rn(w, kf);
    const double g = (k & 1) ? __dsub_rn(1.0, f) : f;
    const double th = __dmul_rn(g, 0.78539816339744831);
    const double z = __dmul_rn(th, th);
    double val;
    if (((k + 1) >> 1) & 1) {
        double S = -1.0 / 1307674368000.0;
        S = __dadd_rn(__dmul_rn(S, z), 1.0 / 6227020800.0);
        S = __dsub_rn(__dmul_rn(S, z), 1.0 / 39916800.0);
        S = __dadd_rn(__dmul_rn(S, z), 1.0 / 362880.0);
        S = __dsub_rn(__dmul_rn(S, z), 1.0 / 5040.0);
        S = __dadd_rn(__dmul_rn(S, z), 1.0 / 120.0);
        S = __dsub_rn(__dmul_rn(S, z), 1.0 / 6.0);
        S = __dadd_rn(__dmul_rn(S, z), 1.0);
        val = __dmul_rn(th, S);
    } else {
        double C = 1.0 / 20922789888000.0;
        C = __dsub_rn(__dmul_rn(C, z), 1.0 / 87178291200.0);
        C = __dadd_rn(__dmul_rn(C, z), 1.0 / 479001600.0);
        C = __dsub_rn(__dmul_rn(C, z), 1.0 / 3628800.0);
        C = __dadd_rn(__dmul_rn(C, z), 1.0 / 40320.0);
        C = __dsub_rn(__dmul_rn(C, z), 1.0 / 720.0);
        C = __dadd_rn(__dmul_rn(C, z), 1.0 / 24.0);
        C = __dsub_rn(__dmul_rn(C, z), 0.5);
        C = __dadd_rn(__dmul_rn(C, z), 1.0);
        val = C;
    }
    return (k >= 2 && k <= 5) ? -val : val;
}

__global__ void sim_params_kernel(unsigned k0, unsigned k1, long long ncurves, long long n,
                                  SimRanges r, SimCurve *curves, double *params_out)
{
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncurves) return;
    const unsigned cw = (unsigned)c;
    Words b = philox10(0u, 0u, cw, 0u, k0, k1);
    const double sigma = between(r.sigma_lo, r.sigma_hi, b.x0);
    const double ratio_r = unit32(b.x1);
    const double efrac = unit32(b.x2);
    const double alpha = between(r.snr_lo, r.snr_hi, b.x3);
    b = philox10(0u, 1u, cw, 0u, k0, k1);
    const bool has = unit32(b.x0) < r.transit_fraction;
    double p = 0.0, L = 0.0;
    for (unsigned k = 0; k < 64u; ++k) {
        b = philox10(k, 2u, cw, 0u, k0, k1);
        p = between(r.period_lo, r.period_hi, b.x0);
        L = __dmul_rn(between(r.ratio_lo, r.ratio_hi, b.x1), p);
        if (L >= r.duration_lo && L <= r.duration_hi) break;
        if (k == 63u) L = fmin(fmax(L, r.duration_lo), r.duration_hi);
    }
    const double npts = __ddiv_rn(__dmul_rn((double)n, L), p);
    const double depth = has ? __ddiv_rn(__dmul_rn(alpha, sigma), __dsqrt_rn(npts)) : 0.0;
    const double t14 = __ddiv_rn(__dmul_rn(2.0, L), __dadd_rn(1.0, ratio_r));
    const double t23 = __dmul_rn(ratio_r, t14);
    SimCurve s;
    s.p = p;
    s.tc = __dmul_rn(efrac, p);
    s.sigma = sigma;
    s.depth = depth;
    s.half14 = __dmul_rn(0.5, t14);
    s.half23 = __dmul_rn(0.5, t23);
    s.ramp = __dsub_rn(s.half14, s.half23);
    s.has_transit = has ? 1 : 0;
    s.pad = 0;
    curves[c] = s;
    if (params_out) {
        double *o = params_out + c * 8;
        o[0] = p;
        o[1] = L;
        o[2] = sigma;
        o[3] = depth;
        o[4] = ratio_r;
        o[5] = s.tc;
        o[6] = alpha;
        o[7] = has ? 1.0 : 0.0;
    }
}

__global__ void __launch_bounds__(SIM_THREADS)
sim_samples_kernel(unsigned k0, unsigned k1, long long ncurves, long long n, long long nchunks,
                   SimRanges r, const SimCurve *__restrict__ curves, double *__restrict__ times,
                   float *__restrict__ flux, long long *__restrict__ offsets)
{
    const long long nitems = ncurves * nchunks;
    const bool noise = !(r.flags & GPFC_LC_NO_NOISE), centred = (r.flags & GPFC_LC_CENTERED) != 0;
    if (offsets) {
        for (long long c = (long long)blockIdx.x * SIM_THREADS + threadIdx.x; c <= ncurves;
             c += (long long)gridDim.x * SIM_THREADS)
            offsets[c] = c * n;
    }
    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        const long long c = item / nchunks;
        const long long i0 = (item - c * nchunks) * SIM_CHUNK;
        const SimCurve s = curves[c];
#pragma unroll
        for (int k = 0; k < SIM_PER_THREAD; ++k) {
            const long long i = i0 + k * SIM_THREADS + threadIdx.x;
            if (i >= n) break;
            const double t = __dadd_rn(r.t_start, __dmul_rn((double)i, r.cadence));
            double f = 1.0;
            if (noise) {
                const Words x = philox10((unsigned)i, 0u, (unsigned)c, 1u, k0, k1);
                const double u1 = unit52(x.x0, x.x1), u2 = unit32(x.x2);
                const double rad = __dsqrt_rn(__dmul_rn(-2.0, sim_ln(u1)));
                const double z = __dmul_rn(rad, sim_cos2pi(u2));
                f = __dadd_rn(f, __dmul_rn(s.sigma, z));
            }
            if (s.has_transit) {
                double y = __ddiv_rn(__dsub_rn(t, s.tc), s.p);
                y = __dsub_rn(y, floor(__dadd_rn(y, 0.5)));
                const double x = __dmul_rn(fabs(y), s.p);
                double shape;
                if (x <= s.half23)
                    shape = 1.0;
                else if (x >= s.half14)
                    shape = 0.0;
                else
                    shape = __ddiv_rn(__dsub_rn(s.half14, x), s.ramp);
                f = __dsub_rn(f, __dmul_rn(s.depth, shape));
            }
            float f32 = __double2float_rn(f);
            if (centred) f32 = __fsub_rn(f32, 1.0f);
            if (times) times[c * n + i] = t;
            flux[c * n + i] = f32;
        }
    }
}

}  // namespace

size_t simulate_scratch_bytes(long long ncurves) { return (size_t)ncurves * sizeof(SimCurve); }

cudaError_t launch_simulate(unsigned long long seed, long long ncurves, long long n,
                            const gpfc_lc_params &prm, double *times, float *flux,
                            long long *offsets, double *params_out, void *scratch, int sms,
                            cudaStream_t st)
{
    SimRanges r;
    r.period_lo = prm.period_lo;
    r.period_hi = prm.period_hi;
    r.duration_lo = prm.duration_lo;
    r.duration_hi = prm.duration_hi;
    r.ratio_lo = prm.ratio_lo;
    r.ratio_hi = prm.ratio_hi;
    r.sigma_lo = prm.sigma_lo;
    r.sigma_hi = prm.sigma_hi;
    r.snr_lo = prm.snr_lo;
    r.snr_hi = prm.snr_hi;
    r.transit_fraction = prm.transit_fraction;
    r.cadence = prm.cadence;
    r.t_start = prm.t_start;
    r.flags = prm.flags;
    const unsigned k0 = (unsigned)seed, k1 = (unsigned)(seed >> 32);
    SimCurve *curves = static_cast<SimCurve *>(scratch);
    sim_params_kernel<<<(unsigned)((ncurves + 127) / 128), 128, 0, st>>>(k0, k1, ncurves, n, r, curves,
                                                                          params_out);
    note_launch();
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const long long nchunks = (n + SIM_CHUNK - 1) / SIM_CHUNK;
    const long long nitems = ncurves * (nchunks > 0 ? nchunks : 1);
    const long long cap = (long long)sms * 8;
    const long long grid = nitems < cap ? (nitems > 0 ? nitems : 1) : cap;
    sim_samples_kernel<<<(unsigned)grid, SIM_THREADS, 0, st>>>(k0, k1, ncurves, n, nchunks, r, curves,
                                                                times, flux, offsets);
    note_launch();
    return cudaGetLastError();
}

}  // namespace gpfc
