// Shared declarations of the CUDA path of libgpfc (sm_100a).  Not used by, and
// not using, anything under oracle/.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

#include "../../include/gpfc.h"

namespace gpfc {

// Samples are handled in anchor tiles of GPFC_TILE consecutive (compacted) samples of a
// curve: the prepass stores, per tile, the smallest u (the anchor a) and a power-of-two
// scale 2^-S with (max u - a) * 2^S < 2^32, and per sample the 8-byte record
// {iv = rint((u - a) * 2^S) (uint32), q (int32)}: |iv * 2^-S - (u - a)| <= 2^-(S+1).
constexpr int GPFC_TILE = 128;

// split prepass (prep.cu): at most PREP_NC_MAX CTAs per curve, used when ncurves * 2 <= SMs
constexpr int PREP_NC_MAX = 32;
constexpr int PREP_PART_DOUBLES = 16;
constexpr size_t PREP_PART_BYTES = (size_t)160 * PREP_PART_DOUBLES * sizeof(double);   // <= 160 CTAs in all

struct TileInfo {
    double a;          // min of u over the tile
    double inv_scale;  // 2^-S
};

// Per-curve table written by the prepass (prep.cu) and read by the fold.
struct CurveMeta {
    long long start;   // first compacted sample of this curve in the u / q scratch arrays
    long long rec0;    // first record of this curve in rec (even: 16-byte aligned)
    long long tile0;   // first entry of this curve in the tile table
    int n_valid;       // samples with finite time and flux (compacted to the front)
    int shift;         // fixed-point exponent s: q = rint((flux - center) * 2^s)
    double center;     // per-curve constant removed before quantisation (0 for centred input)
    double inv_scale;  // 2^-s
    double umin;       // min / max of u = t - t0 over the valid samples
    double umax;
    double span_max;   // largest tile span of the curve
    double pivot;      // mean of the centred, quantised flux: (sum q) 2^-s / n_valid
    // Samples with u == 0 exactly (t == t0: the first sample of a curve whose times start at
    // t0) have phase 0 and bin 0 at EVERY period, and would sit in the guard band of every
    // (tile, period).  The prepass keeps up to 255 of them out of the sample arrays; the fold
    // epilogues add them to bin 0: n_zero points with fixed-point flux sum q_zero.
    int n_zero;
    int q_zero;
};

// Scratch carved out of the workspace for one gpfc_fold_batch call.
struct Scratch {
    double *u;         // [n_total]  t - t0, valid samples compacted per curve
    int *q;            // [n_total]  fixed-point flux
    int2 *rec;         // [n_total + ncurves + 2]  {iv, q} (see GPFC_TILE)
    TileInfo *tiles;   // [n_total / GPFC_TILE + ncurves + 1]
    CurveMeta *meta;   // [ncurves]
    double *part;      // [PREP_PART_BYTES / 8] partial results of the split prepass (prep.cu), or NULL
    double *rp;        // [nperiods] RN(1/P) * rows, NaN for a period that is not finite-positive;
                       // rows = fold_rows(nbins): 256 for nbins in {32..256}, 1024 for {512, 1024},
                       // else nbins
};

struct FoldArgs {
    const double *u;
    const int *q;
    const int2 *rec;
    const TileInfo *tiles;
    const CurveMeta *meta;
    const double *rp;
    const double *periods;
    long long ncurves;
    long long nperiods;
    int nbins;
    float *out_sum;
    uint32_t *out_count;
    float *out_norm;
    int vec_ok;                   // every non-NULL output above is 16-byte aligned (vector stores)
    // fused equal-count merge (fold_pk.cu): nb2 > 0 replaces the three outputs above
    int nb2;
    float *out_mean2;             // [curve][period][nb2]
    float *out_norm2;             // [curve][period][nb2]
    unsigned *side;               // fold_pk.cu: 32-bit count overflow area, 32768 words per CTA, or NULL
    // Non-NULL (the unfused two-tier route, api.cu): out_sum holds the sums of flux - center
    // (small numbers: their fp32 rounding no longer costs the 6e-8 of an uncentred flux near 1)
    // and the curve's center goes to center_out[curve] for the merge kernel to add back.
    double *center_out;
    unsigned long long *stats;    // device counters (DeviceInfo::stats), or NULL
};

// Per-device state, initialised on first use of a device by any thread (api.cu): kernel
// attributes (opt-in dynamic shared memory) are per device, so is the SM count.  Nothing here
// synchronises a stream or the host.
struct DeviceInfo {
    int num_sms;
    unsigned long long *stats;    // device counters: [0] work items folded with the exact formula
                                  // for every point-period, [1] guard-band re-checks (lane x tile),
                                  // [2] work items folded twice (packed 16-bit count overflow)
};
cudaError_t device_info(const DeviceInfo **out);
void note_launch(int n = 1);      // per-thread kernel-launch counter (gpfc_profile_read)

// ---- exact bin of one sample (-1 = skip the sample, reading R20): the formula of include/gpfc.h, every operation
// rounded once (intrinsics, so nothing can be contracted into an FMA).
// PAPER.md:111 "First", "Secondly".
__device__ __forceinline__ int exact_bin(double u, double period, int nbins)
{
    double x = __ddiv_rn(u, period);
    if (!(fabs(x) < CUDART_INF)) return -1;   // R20: u / P overflows -> the sample is skipped
    double phi = __dsub_rn(x, floor(x));
    double scaled = __dmul_rn(phi, (double)nbins);
    long long k = (long long)scaled;   // truncation; scaled >= 0
    if (k >= nbins) k = nbins - 1;
    return (int)k;
}

__device__ __forceinline__ bool period_ok(double p)
{
    return (p > 0.0) && (p < CUDART_INF);   // false for NaN, <= 0, +inf
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ int warp_sum_int(int v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// One folded profile held in shared memory as nbins 8-byte slots
// {int32 fixed-point sum, uint32 count}.  A whole warp converts it, writes the
// requested outputs and leaves the slots zeroed.
//   out_sum[k]   = (float)(Q * 2^-s + count * center)
//   out_norm[k]  = mu + (m[k] - mu) / s, fp64, population std over
//                  the non-empty bins; empty bins -> mu; K = 0 -> 0; K < 2 or s = 0 -> mu
__device__ __forceinline__ void emit_profile(unsigned long long *slots, int nbins, int lane,
                                             double inv_scale, double center, bool zero_row,
                                             float *out_sum, uint32_t *out_count,
                                             float *out_norm)
{
    double acc = 0.0;
    int kk = 0;
    double *mslots = reinterpret_cast<double *>(slots);
    for (int k = lane; k < nbins; k += 32) {
        unsigned long long s = slots[k];
        int qsum = (int)(unsigned)(s & 0xffffffffull);
        unsigned cnt = (unsigned)(s >> 32);
        if (zero_row) {
            qsum = 0;
            cnt = 0;
        }
        double sf = __dadd_rn(__dmul_rn((double)qsum, inv_scale),
                              __dmul_rn((double)cnt, center));
        if (out_sum) out_sum[k] = (float)sf;
        if (out_count) out_count[k] = cnt;
        if (out_norm) {
            double m = CUDART_NAN;
            if (cnt > 0) {
                m = __ddiv_rn(sf, (double)cnt);
                acc += m;
                kk += 1;
            }
            mslots[k] = m;
        } else {
            slots[k] = 0ull;
        }
    }
    if (!out_norm) return;
    __syncwarp();
    acc = warp_sum(acc);
    kk = warp_sum_int(kk);
    double mu = (kk > 0) ? __ddiv_rn(acc, (double)kk) : 0.0;
    double vacc = 0.0;
    for (int k = lane; k < nbins; k += 32) {
        double m = mslots[k];
        if (m == m) {
            double d = __dsub_rn(m, mu);
            vacc += __dmul_rn(d, d);
        }
    }
    vacc = warp_sum(vacc);
    double sd = (kk > 0) ? sqrt(__ddiv_rn(vacc, (double)kk)) : 0.0;
    bool flat = (kk < 2) || !(sd > 0.0);
    for (int k = lane; k < nbins; k += 32) {
        double m = mslots[k];
        double o = mu;
        if (!flat && m == m) o = __dadd_rn(mu, __ddiv_rn(__dsub_rn(m, mu), sd));
        out_norm[k] = (float)o;
        slots[k] = 0ull;
    }
}

// launchers (defined in the .cu files).  Every launch_* counts its kernels with note_launch().
cudaError_t launch_prep(const double *times, const float *flux, const int64_t *offsets,
                        long long ncurves, const double *t0, double t0_scalar,
                        const double *periods, long long nperiods, int rows, Scratch s,
                        long long n_total, int sms, cudaStream_t st);
int fold_rows(int nbins);         // fold.cu: resolution the fold kernel for `nbins` works at
cudaError_t launch_fold(const FoldArgs &a, cudaStream_t st);
cudaError_t launch_fold_lp(const FoldArgs &a, cudaStream_t st, int sms);   // fold_lp.cu: nbins 32..256
cudaError_t launch_fold_pk(const FoldArgs &a, cudaStream_t st, int sms);   // fold_pk.cu: nbins 512..4096
cudaError_t launch_fold_generic(const FoldArgs &a, cudaStream_t st, int sms);   // fold.cu: any nbins
bool fold_lp_handles(int nbins);
bool fold_lp_pow2(int nbins);
bool fold_pk_handles(int nbins);
int fold_pk_rows(int nbins);
bool fold_pk_can_merge(int nbins, int nb2);      // the fused equal-count merge fits in shared memory
size_t fold_pk_side_bytes(int sms);
long long fold_pk_flush_samples();               // curves longer than this need FoldArgs::side
cudaError_t fold_lp_init_device();
cudaError_t fold_pk_init_device();
cudaError_t merge_init_device();
cudaError_t launch_normalize(const float *sum, const uint32_t *count, long long nprofiles,
                             int nbins, float *out, cudaStream_t st);
cudaError_t launch_merge(const float *sum, const uint32_t *count, long long nprofiles, int nb1,
                         int nb2, float *out_mean, float *out_norm, const double *offset,
                         cudaStream_t st);
cudaError_t launch_grid(double pmin, double pmax, long long nperiods, int mode_flags,
                        double *out, cudaStream_t st);
cudaError_t measure_peaks(double *out_host, cudaStream_t st);
size_t simulate_scratch_bytes(long long ncurves);                                 // simulate.cu
cudaError_t launch_simulate(unsigned long long seed, long long ncurves, long long n,
                            const gpfc_lc_params &prm, double *times, float *flux,
                            long long *offsets, double *params_out, void *scratch, int sms,
                            cudaStream_t st);

}  // namespace gpfc
