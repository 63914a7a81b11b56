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

__global__ void __launch_bounds__(PREP_THREADS)
prep_curves_kernel(const double *__restrict__ times, const float *__restrict__ flux,
                   const int64_t *__restrict__ offsets, const double *__restrict__ t0v,
                   double t0_scalar, Scratch s)
{
    __shared__ BlockRed red;
    __shared__ int warp_tot[32];
    __shared__ int tile_base;
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

    // pass 3: ordered compaction + conversion
    if (tid == 0) tile_base = 0;
    __syncthreads();
    double qsum = 0.0, qzero = 0.0;
    for (long long b = 0; b < n; b += PREP_THREADS) {
        long long i = b + tid;
        bool ok = false;
        double u = 0.0;
        int q = 0;
        if (i < n) {
            double ti = t[i];
            float fi = f[i];
            ok = finite_d(ti) && finite_f(fi);
            if (ok) {
                u = __dsub_rn(ti, t0);
                q = (int)llrint(((double)fi - center) * scale);
                if (divert && u == 0.0) {
                    qzero += (double)q;
                    qsum += (double)q;
                    ok = false;
                }
            }
        }
        unsigned bal = __ballot_sync(0xffffffffu, ok);
        int wpos = __popc(bal & ((1u << lane) - 1u));
        if (lane == 0) warp_tot[warp] = __popc(bal);
        __syncthreads();
        int wbase = 0;
        for (int w = 0; w < warp; ++w) wbase += warp_tot[w];
        int base = tile_base;
        if (ok) {
            long long o = start + base + wbase + wpos;
            s.u[o] = u;
            s.q[o] = q;
            qsum += (double)q;
        }
        __syncthreads();
        if (tid == PREP_THREADS - 1) tile_base = base + wbase + __popc(bal);
        __syncthreads();
    }
    // pass 4: anchor tiles of GPFC_TILE compacted samples: anchor a = min u of the tile,
    // record {v = u - a, q}.  (The compacted u / q were written by this CTA above.)
    const int n_valid = tile_base;
    const long long tile0 = start / GPFC_TILE + c;   // disjoint per curve: ceil(n/T) <= n/T + 1
    const long long rec0 = (start + c + 1) & ~1LL;   // even, disjoint per curve
    qsum = block_sum(qsum, red);                     // exact: |sum q| < 2^31
    qzero = block_sum(qzero, red);
    double span_max = 0.0;
    for (int t = warp; t * GPFC_TILE < n_valid; t += PREP_THREADS / 32) {
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
        span_max = fmax(span_max, span);
    }
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
        m.n_valid = tile_base;
        m.shift = shift;
        m.center = center;
        m.inv_scale = ldexp(1.0, -shift);
        m.umin = (cnt > 0.0) ? umin : 0.0;
        m.umax = (cnt > 0.0) ? umax : 0.0;
        s.meta[c] = m;
    }
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
                        cudaStream_t st)
{
    if (ncurves > 0) {
        prep_curves_kernel<<<(unsigned)ncurves, PREP_THREADS, 0, st>>>(times, flux, offsets, t0,
                                                                      t0_scalar, s);
        note_launch();
    }
    if (nperiods > 0) {
        unsigned blocks = (unsigned)((nperiods + 255) / 256);
        prep_periods_kernel<<<blocks, 256, 0, st>>>(periods, nperiods, rows, s.rp);
        note_launch();
    }
    return cudaGetLastError();
}

}  // namespace gpfc
