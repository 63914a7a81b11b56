// Prepass of the fold: per-curve sample conditioning and per-period reciprocals.
//
// Per curve (one CTA): drop samples with a non-finite time or flux (gpfc.h data
// conventions), form u = t - t0 in fp64 (one rounding, as the formula says), pick
// the curve's fixed-point exponent s and write q = rint((flux - center) * 2^s).
//
// Accumulation: shared-memory atomics are native only for 32-bit
// integers on sm_100a, so flux is summed in int32 fixed point.  s is the largest
// exponent with  sum_i |q_i| < 2^31  (L1 norm of the curve), hence no bin can
// overflow under any binning, and integer addition makes the sums exact and
// order-independent.  Flux that is already a multiple of 2^-s (fp32 flux near
// 1.0 minus an fp32 median is a multiple of 2^-24, and s >= 24 for the paper's
// noise levels) is represented without any rounding.  If the flux is far from
// centred (L1 norm dominated by its mean) the fp32-rounded mean is removed
// first and added back, times the bin count, at write-out.
#include "common.cuh"

namespace gpfc {

namespace {

constexpr int PREP_THREADS = 1024;
constexpr int PREP_K = 4;            // consecutive samples per thread in the compaction pass

struct BlockRed {
    double v[32];
};

__device__ double block_sum(double x, BlockRed &sm)
{
    int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    x = warp_sum(x);
    __syncthreads();
    if (lane == 0) sm.v[warp] = x;
    __syncthreads();
    double t = (lane < (int)(blockDim.x >> 5)) ? sm.v[lane] : 0.0;
    t = warp_sum(t);
    return t;   // same value in every thread (fixed tree: deterministic)
}

__device__ double block_min(double x, BlockRed &sm)
{
    int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x = fmin(x, __shfl_xor_sync(0xffffffffu, x, o));
    __syncthreads();
    if (lane == 0) sm.v[warp] = x;
    __syncthreads();
    double t = (lane < (int)(blockDim.x >> 5)) ? sm.v[lane] : CUDART_INF;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t = fmin(t, __shfl_xor_sync(0xffffffffu, t, o));
    return t;
}

__device__ __forceinline__ bool finite_d(double x) { return fabs(x) < CUDART_INF; }
__device__ __forceinline__ bool finite_f(float x) { return fabsf(x) < CUDART_INF_F; }

// One anchor tile of GPFC_TILE compacted samples (a whole warp): anchor a = min u of the tile,
// records {v = rint((u - a) 2^S), q}, TileInfo {a, 2^-S}.  Returns the tile's span.
__device__ __forceinline__ double prep_tile(const Scratch &s, long long start, long long rec0,
                                            long long tile0, int t, int n_valid, int lane)
{
    const int base = t * GPFC_TILE;
    double uu[GPFC_TILE / 32];
    double lo = CUDART_INF, hi = -CUDART_INF;
#pragma unroll
    for (int k = 0; k < GPFC_TILE / 32; ++k) {
        int i = base + k * 32 + lane;
        uu[k] = (i < n_valid) ? s.u[start + i] : CUDART_NAN;
        if (i < n_valid) {
            lo = fmin(lo, uu[k]);
            hi = fmax(hi, uu[k]);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    const double span = __dsub_ru(hi, lo);
    int e = 0;
    (void)frexp(span, &e);                 // span < 2^e
    int S = 32 - e;                        // span * 2^S < 2^32
    if (S > 40) S = 40;
    if (S < -900) S = -900;
    if (span * ldexp(1.0, S) > 4294967294.0) S -= 1;   // rint() below never reaches 2^32
    const double scale = ldexp(1.0, S);
#pragma unroll
    for (int k = 0; k < GPFC_TILE / 32; ++k) {
        int i = base + k * 32 + lane;
        if (i < n_valid) {
            double w = rint(__dmul_rn(__dsub_rn(uu[k], lo), scale));
            if (w > 4294967295.0) w = 4294967295.0;
            s.rec[rec0 + i] = make_int2((int)(unsigned)w, s.q[start + i]);
        }
    }
    if (lane == 0) {
        TileInfo ti;
        ti.a = lo;
        ti.inv_scale = ldexp(1.0, -S);
        s.tiles[tile0 + t] = ti;
    }
    return span;
}

__global__ void __launch_bounds__(PREP_THREADS)
prep_curves_kernel(const double *__restrict__ times, const float *__restrict__ flux,
                   const int64_t *__restrict__ offsets, const double *__restrict__ t0v,
                   double t0_scalar, Scratch s)
{
    __shared__ BlockRed red;
    __shared__ int warp_tot[2][32];
    __shared__ double warp_span[32];
    const long long c = blockIdx.x;
    const long long start = offsets[c];
    const long long n = offsets[c + 1] - start;
    const double t0 = t0v ? t0v[c] : t0_scalar;
    const double *t = times + start;
    const float *f = flux + start;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // pass 1: L1 norm, sum, count, range of u over the valid samples
    double a0 = 0.0, sm = 0.0, cnt = 0.0, cnt0 = 0.0, umin = CUDART_INF, nmax = CUDART_INF;
#pragma unroll 4
    for (long long i = tid; i < n; i += PREP_THREADS) {
        double ti = t[i];
        float fi = f[i];
        if (finite_d(ti) && finite_f(fi)) {
            double u = __dsub_rn(ti, t0);
            a0 += fabs((double)fi);
            sm += (double)fi;
            cnt += 1.0;
            if (u == 0.0) cnt0 += 1.0;
            umin = fmin(umin, u);
            nmax = fmin(nmax, -u);
        }
    }
    a0 = block_sum(a0, red);
    sm = block_sum(sm, red);
    cnt = block_sum(cnt, red);
    cnt0 = block_sum(cnt0, red);
    // samples at u == 0 (CurveMeta::n_zero) leave the sample arrays when there are few of them
    const bool divert = cnt0 > 0.0 && cnt0 <= 255.0;
    umin = block_min(umin, red);
    double umax = -block_min(nmax, red);

    // pass 2: L1 norm about the fp32-rounded mean; centre only if it buys >= 2 bits
    double center = 0.0, a = a0;
    if (cnt > 0.0) {
        float cf = (float)(sm / cnt);
        double a1 = 0.0;
#pragma unroll 4
        for (long long i = tid; i < n; i += PREP_THREADS) {
            double ti = t[i];
            float fi = f[i];
            if (finite_d(ti) && finite_f(fi)) a1 += fabs((double)fi - (double)cf);
        }
        a1 = block_sum(a1, red);
        if (finite_f(cf) && a1 * 4.0 < a0) {
            center = (double)cf;
            a = a1;
        }
    }
    // largest s with a * 2^s + n/2 < 2^31 (each |q_i| <= |f_i| 2^s + 1/2)
    int shift = 0;
    if (a > 0.0) {
        double room = 2147483647.0 - 0.5 * cnt - 1.0;
        int e;
        double mant = frexp(room / a, &e);   // room / a = mant * 2^e, mant in [0.5, 1)
        (void)mant;
        shift = e - 1;                        // 2^shift <= room / a
        // every finite fp32 curve fits: a <= n 2^128 and a >= 2^-149
        if (shift > 200) shift = 200;
        if (shift < -200) shift = -200;
    }
    const double scale = ldexp(1.0, shift);

    // pass 3: ordered compaction + conversion.  Every thread takes PREP_K consecutive samples;
    // one barrier per PREP_THREADS * PREP_K samples (the warp totals are double-buffered by
    // iteration parity, every thread keeps the running base itself).
    double qsum = 0.0, qzero = 0.0;
    int run_base = 0;
    int it = 0;
    for (long long b = 0; b < n; b += (long long)PREP_THREADS * PREP_K, ++it) {
        const long long i0 = b + (long long)tid * PREP_K;
        bool ok[PREP_K];
        double u[PREP_K];
        int q[PREP_K];
        int c = 0;
#pragma unroll
        for (int k = 0; k < PREP_K; ++k) {
            const long long i = i0 + k;
            ok[k] = false;
            u[k] = 0.0;
            q[k] = 0;
            if (i < n) {
                double ti = t[i];
                float fi = f[i];
                ok[k] = finite_d(ti) && finite_f(fi);
                if (ok[k]) {
                    u[k] = __dsub_rn(ti, t0);
                    q[k] = (int)llrint(((double)fi - center) * scale);
                    if (divert && u[k] == 0.0) {
                        qzero += (double)q[k];
                        qsum += (double)q[k];
                        ok[k] = false;
                    }
                }
            }
            c += ok[k] ? 1 : 0;
        }
        int inc = c;                                  // inclusive scan inside the warp
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += v;
        }
        if (lane == 31) warp_tot[it & 1][warp] = inc;
        __syncthreads();
        const int wt = warp_tot[it & 1][lane];        // lane w: total of warp w
        int winc = wt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += v;
        }
        const int wbase = __shfl_sync(0xffffffffu, winc, warp) - __shfl_sync(0xffffffffu, wt, warp);
        const int total = __shfl_sync(0xffffffffu, winc, 31);
        long long o = start + run_base + wbase + inc - c;
#pragma unroll
        for (int k = 0; k < PREP_K; ++k)
            if (ok[k]) {
                s.u[o] = u[k];
                s.q[o] = q[k];
                qsum += (double)q[k];
                ++o;
            }
        run_base += total;
    }
    __syncthreads();   // the compacted u / q of this CTA are visible to all of its warps
    // pass 4: anchor tiles of GPFC_TILE compacted samples: anchor a = min u of the tile,
    // record {v = u - a, q}.  (The compacted u / q were written by this CTA above.)
    const int n_valid = run_base;
    const long long tile0 = start / GPFC_TILE + c;   // disjoint per curve: ceil(n/T) <= n/T + 1
    const long long rec0 = (start + c + 1) & ~1LL;   // even, disjoint per curve
    qsum = block_sum(qsum, red);                     // exact: |sum q| < 2^31
    qzero = block_sum(qzero, red);
    double span_max = 0.0;
    for (int t = warp; t * GPFC_TILE < n_valid; t += PREP_THREADS / 32)
        span_max = fmax(span_max, prep_tile(s, start, rec0, tile0, t, n_valid, lane));
    if (lane == 0) warp_span[warp] = span_max;
    __syncthreads();
    if (tid == 0) {
        for (int w = 0; w < PREP_THREADS / 32; ++w) span_max = fmax(span_max, warp_span[w]);
        CurveMeta m;
        m.start = start;
        m.rec0 = rec0;
        m.pivot = (cnt > 0.0) ? __ddiv_rn(__dmul_rn(qsum, ldexp(1.0, -shift)), cnt) : 0.0;
        m.n_zero = divert ? (int)cnt0 : 0;
        m.q_zero = (int)qzero;
        m.tile0 = tile0;
        m.span_max = span_max;
        m.n_valid = run_base;
        m.shift = shift;
        m.center = center;
        m.inv_scale = ldexp(1.0, -shift);
        m.umin = (cnt > 0.0) ? umin : 0.0;
        m.umax = (cnt > 0.0) ? umax : 0.0;
        s.meta[c] = m;
    }
}

// ---- the same prepass split over PREP_NC CTAs per curve, for calls with few (long) curves:
// one SM pulls ~100 GB/s, so a single CTA needs ~130 us for a 70,000-sample curve (2-3 % of a
// config-1 / config-5 step).  Five small kernels, stream order is the only synchronisation;
// partial results go through Scratch::part.  Same arithmetic as prep_curves_kernel, with the
// partial sums combined in part order (deterministic).
struct PrepPart {
    double a0, sm, cnt, cnt0, umin, nmax, a1, qsum, qzero, span;
    double pad[6];
};
static_assert(sizeof(PrepPart) == PREP_PART_DOUBLES * sizeof(double), "Scratch::part stride");

struct PrepRange {
    long long start, n, lo, hi;
    double t0;
};

__device__ __forceinline__ PrepRange prep_range(const int64_t *offsets, const double *t0v, double t0_scalar,
                                                int nc)
{
    PrepRange r;
    const long long c = blockIdx.y;
    r.start = offsets[c];
    r.n = offsets[c + 1] - r.start;
    const long long chunk = (((r.n + nc - 1) / nc) + PREP_K - 1) / PREP_K * PREP_K;
    r.lo = min(r.n, (long long)blockIdx.x * chunk);
    r.hi = min(r.n, r.lo + chunk);
    r.t0 = t0v ? t0v[c] : t0_scalar;
    return r;
}

// totals of the curve from the per-part partials (every thread computes the same numbers)
struct PrepTotals {
    double a0, sm, cnt, cnt0, umin, umax, a1;
    double center, scale;
    int shift;
    bool divert;
};

__device__ PrepTotals prep_totals(const PrepPart *pp, int nc, bool with_a1)
{
    PrepTotals t;
    t.a0 = t.sm = t.cnt = t.cnt0 = t.a1 = 0.0;
    double umin = CUDART_INF, nmax = CUDART_INF;
    for (int k = 0; k < nc; ++k) {
        t.a0 += pp[k].a0;
        t.sm += pp[k].sm;
        t.cnt += pp[k].cnt;
        t.cnt0 += pp[k].cnt0;
        umin = fmin(umin, pp[k].umin);
        nmax = fmin(nmax, pp[k].nmax);
        if (with_a1) t.a1 += pp[k].a1;
    }
    t.umin = umin;
    t.umax = -nmax;
    t.divert = t.cnt0 > 0.0 && t.cnt0 <= 255.0;
    t.center = 0.0;
    t.shift = 0;
    t.scale = 1.0;
    if (with_a1) {
        double a = t.a0;
        if (t.cnt > 0.0) {
            const float cf = (float)(t.sm / t.cnt);
            if (finite_f(cf) && t.a1 * 4.0 < t.a0) {
                t.center = (double)cf;
                a = t.a1;
            }
        }
        if (a > 0.0) {
            const double room = 2147483647.0 - 0.5 * t.cnt - 1.0;
            int e;
            (void)frexp(room / a, &e);
            t.shift = e - 1;
            if (t.shift > 200) t.shift = 200;
            if (t.shift < -200) t.shift = -200;
        }
        t.scale = ldexp(1.0, t.shift);
    }
    return t;
}

__global__ void __launch_bounds__(PREP_THREADS)
prep_split1_kernel(const double *__restrict__ times, const float *__restrict__ flux,
                   const int64_t *__restrict__ offsets, const double *__restrict__ t0v,
                   double t0_scalar, int nc, PrepPart *part)
{
    __shared__ BlockRed red;
    const PrepRange r = prep_range(offsets, t0v, t0_scalar, nc);
    const double *t = times + r.start;
    const float *f = flux + r.start;
    const int tid = threadIdx.x;
    double a0 = 0.0, sm = 0.0, cnt = 0.0, cnt0 = 0.0, umin = CUDART_INF, nmax = CUDART_INF;
#pragma unroll 4
    for (long long i = r.lo + tid; i < r.hi; i += PREP_THREADS) {
        const double ti = t[i];
        const float fi = f[i];
        if (finite_d(ti) && finite_f(fi)) {
            const double u = __dsub_rn(ti, r.t0);
            a0 += fabs((double)fi);
            sm += (double)fi;
            cnt += 1.0;
            if (u == 0.0) cnt0 += 1.0;
            umin = fmin(umin, u);
            nmax = fmin(nmax, -u);
        }
    }
    a0 = block_sum(a0, red);
    sm = block_sum(sm, red);
    cnt = block_sum(cnt, red);
    cnt0 = block_sum(cnt0, red);
    umin = block_min(umin, red);
    nmax = block_min(nmax, red);
    if (tid == 0) {
        PrepPart &o = part[(size_t)blockIdx.y * nc + blockIdx.x];
        o.a0 = a0;
        o.sm = sm;
        o.cnt = cnt;
        o.cnt0 = cnt0;
        o.umin = umin;
        o.nmax = nmax;
        o.a1 = o.qsum = o.qzero = o.span = 0.0;
    }
}

__global__ void __launch_bounds__(PREP_THREADS)
prep_split2_kernel(const double *__restrict__ times, const float *__restrict__ flux,
                   const int64_t *__restrict__ offsets, const double *__restrict__ t0v,
                   double t0_scalar, int nc, PrepPart *part)
{
    __shared__ BlockRed red;
    const PrepRange r = prep_range(offsets, t0v, t0_scalar, nc);
    PrepPart *pp = part + (size_t)blockIdx.y * nc;
    const PrepTotals tot = prep_totals(pp, nc, false);
    const double *t = times + r.start;
    const float *f = flux + r.start;
    const int tid = threadIdx.x;
    double a1 = 0.0;
    if (tot.cnt > 0.0) {
        const float cf = (float)(tot.sm / tot.cnt);
#pragma unroll 4
        for (long long i = r.lo + tid; i < r.hi; i += PREP_THREADS) {
            const double ti = t[i];
            const float fi = f[i];
            if (finite_d(ti) && finite_f(fi)) a1 += fabs((double)fi - (double)cf);
        }
    }
    a1 = block_sum(a1, red);
    if (tid == 0) pp[blockIdx.x].a1 = a1;
}

__global__ void __launch_bounds__(PREP_THREADS)
prep_split3_kernel(const double *__restrict__ times, const float *__restrict__ flux,
                   const int64_t *__restrict__ offsets, const double *__restrict__ t0v,
                   double t0_scalar, int nc, PrepPart *part, Scratch s)
{
    __shared__ BlockRed red;
    __shared__ int warp_tot[2][32];
    const PrepRange r = prep_range(offsets, t0v, t0_scalar, nc);
    PrepPart *pp = part + (size_t)blockIdx.y * nc;
    const PrepTotals tot = prep_totals(pp, nc, true);
    const double *t = times + r.start;
    const float *f = flux + r.start;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // valid samples that stay in the arrays in front of this part
    double before = 0.0;
    for (int k = 0; k < (int)blockIdx.x; ++k) before += pp[k].cnt - (tot.divert ? pp[k].cnt0 : 0.0);
    int run_base = (int)before;
    double qsum = 0.0, qzero = 0.0;
    int it = 0;
    for (long long b = r.lo; b < r.hi; b += (long long)PREP_THREADS * PREP_K, ++it) {
        const long long i0 = b + (long long)tid * PREP_K;
        bool ok[PREP_K];
        double u[PREP_K];
        int q[PREP_K];
        int c = 0;
#pragma unroll
        for (int k = 0; k < PREP_K; ++k) {
            const long long i = i0 + k;
            ok[k] = false;
            u[k] = 0.0;
            q[k] = 0;
            if (i < r.hi) {
                const double ti = t[i];
                const float fi = f[i];
                ok[k] = finite_d(ti) && finite_f(fi);
                if (ok[k]) {
                    u[k] = __dsub_rn(ti, r.t0);
                    q[k] = (int)llrint(((double)fi - tot.center) * tot.scale);
                    if (tot.divert && u[k] == 0.0) {
                        qzero += (double)q[k];
                        qsum += (double)q[k];
                        ok[k] = false;
                    }
                }
            }
            c += ok[k] ? 1 : 0;
        }
        int inc = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += v;
        }
        if (lane == 31) warp_tot[it & 1][warp] = inc;
        __syncthreads();
        const int wt = warp_tot[it & 1][lane];
        int winc = wt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += v;
        }
        const int wbase = __shfl_sync(0xffffffffu, winc, warp) - __shfl_sync(0xffffffffu, wt, warp);
        const int total = __shfl_sync(0xffffffffu, winc, 31);
        long long o = r.start + run_base + wbase + inc - c;
#pragma unroll
        for (int k = 0; k < PREP_K; ++k)
            if (ok[k]) {
                s.u[o] = u[k];
                s.q[o] = q[k];
                qsum += (double)q[k];
                ++o;
            }
        run_base += total;
    }
    qsum = block_sum(qsum, red);
    qzero = block_sum(qzero, red);
    if (tid == 0) {
        pp[blockIdx.x].qsum = qsum;
        pp[blockIdx.x].qzero = qzero;
    }
}

// anchor tiles: the warps of all parts of a curve share its tiles
__global__ void __launch_bounds__(PREP_THREADS)
prep_split4_kernel(const int64_t *__restrict__ offsets, int nc, PrepPart *part, Scratch s)
{
    __shared__ double warp_span[32];
    const long long c = blockIdx.y;
    const long long start = offsets[c];
    PrepPart *pp = part + (size_t)c * nc;
    const PrepTotals tot = prep_totals(pp, nc, false);
    const int n_valid = (int)(tot.cnt - (tot.divert ? tot.cnt0 : 0.0));
    const long long tile0 = start / GPFC_TILE + c;
    const long long rec0 = (start + c + 1) & ~1LL;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double span_max = 0.0;
    for (int t = blockIdx.x * (PREP_THREADS / 32) + warp; t * GPFC_TILE < n_valid;
         t += nc * (PREP_THREADS / 32))
        span_max = fmax(span_max, prep_tile(s, start, rec0, tile0, t, n_valid, lane));
    if (lane == 0) warp_span[warp] = span_max;
    __syncthreads();
    if (tid == 0) {
        for (int w = 0; w < PREP_THREADS / 32; ++w) span_max = fmax(span_max, warp_span[w]);
        pp[blockIdx.x].span = span_max;
    }
}

__global__ void prep_split5_kernel(const int64_t *__restrict__ offsets, int nc, const PrepPart *part,
                                   Scratch s)
{
    const long long c = blockIdx.x;
    if (threadIdx.x != 0) return;
    const long long start = offsets[c];
    const PrepPart *pp = part + (size_t)c * nc;
    const PrepTotals tot = prep_totals(pp, nc, true);
    double qsum = 0.0, qzero = 0.0, span = 0.0;
    for (int k = 0; k < nc; ++k) {
        qsum += pp[k].qsum;          // exact: integers, |sum| < 2^31
        qzero += pp[k].qzero;
        span = fmax(span, pp[k].span);
    }
    CurveMeta m;
    m.start = start;
    m.rec0 = (start + c + 1) & ~1LL;
    m.tile0 = start / GPFC_TILE + c;
    m.pivot = (tot.cnt > 0.0) ? __ddiv_rn(__dmul_rn(qsum, ldexp(1.0, -tot.shift)), tot.cnt) : 0.0;
    m.n_zero = tot.divert ? (int)tot.cnt0 : 0;
    m.q_zero = (int)qzero;
    m.span_max = span;
    m.n_valid = (int)(tot.cnt - (tot.divert ? tot.cnt0 : 0.0));
    m.shift = tot.shift;
    m.center = tot.center;
    m.inv_scale = ldexp(1.0, -tot.shift);
    m.umin = (tot.cnt > 0.0) ? tot.umin : 0.0;
    m.umax = (tot.cnt > 0.0) ? tot.umax : 0.0;
    s.meta[c] = m;
}

// rp[j] = RN(1/P_j) * rows (exact scaling for power-of-two rows), NaN when the
// period is not finite and positive.  rows = fold_rows(nbins): the resolution the fold
// kernel works at (it merges adjacent rows at write-out when nbins is smaller).
__global__ void prep_periods_kernel(const double *__restrict__ periods, long long nperiods,
                                    int rows, double *__restrict__ rp)
{
    long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= nperiods) return;
    double p = periods[j];
    double r = CUDART_NAN;
    if (period_ok(p)) r = __dmul_rn(__drcp_rn(p), (double)rows);
    rp[j] = r;
}

}  // namespace

cudaError_t launch_prep(const double *times, const float *flux, const int64_t *offsets,
                        long long ncurves, const double *t0, double t0_scalar,
                        const double *periods, long long nperiods, int rows, Scratch s,
                        long long n_total, int sms, cudaStream_t st)
{
    if (ncurves > 0) {
        // few long curves: PREP_NC CTAs per curve (the host only knows the mean length)
        int nc = 1;
        if (s.part && ncurves * 2 <= sms) {
            const long long mean_n = n_total / ncurves;
            nc = (int)(sms / ncurves);
            if (nc > PREP_NC_MAX) nc = PREP_NC_MAX;
            if ((long long)nc * 2048 > mean_n) nc = (int)(mean_n / 2048);
        }
        if (nc >= 2) {
            PrepPart *part = reinterpret_cast<PrepPart *>(s.part);
            const dim3 grid((unsigned)nc, (unsigned)ncurves);
            prep_split1_kernel<<<grid, PREP_THREADS, 0, st>>>(times, flux, offsets, t0, t0_scalar, nc, part);
            prep_split2_kernel<<<grid, PREP_THREADS, 0, st>>>(times, flux, offsets, t0, t0_scalar, nc, part);
            prep_split3_kernel<<<grid, PREP_THREADS, 0, st>>>(times, flux, offsets, t0, t0_scalar, nc, part, s);
            prep_split4_kernel<<<grid, PREP_THREADS, 0, st>>>(offsets, nc, part, s);
            prep_split5_kernel<<<(unsigned)ncurves, 32, 0, st>>>(offsets, nc, part, s);
            note_launch(5);
        } else {
            prep_curves_kernel<<<(unsigned)ncurves, PREP_THREADS, 0, st>>>(times, flux, offsets, t0,
                                                                          t0_scalar, s);
            note_launch();
        }
    }
    if (nperiods > 0) {
        unsigned blocks = (unsigned)((nperiods + 255) / 256);
        prep_periods_kernel<<<blocks, 256, 0, st>>>(periods, nperiods, rows, s.rp);
        note_launch();
    }
    return cudaGetLastError();
}

}  // namespace gpfc
