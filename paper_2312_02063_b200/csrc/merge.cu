// Step 4 of the paper's fold ("Fourthly", Fig. 4(c)): merge the nb1
// equal-width intermediary bins of a folded profile into nb2 final bins that each hold the
// same number of points, scanning left to right and splitting a bin on a boundary pro rata
// by count (reading R18).  With N = total count and cumulative count / sum
// C(k), S(k) after fine bin k, output bin b ends at target_b = (N / nb2) (b + 1) (= N for
// the last bin) inside the first fine bin k with C(k) >= target_b:
//     Scum_b  = S(k-1) + ((target_b - C(k-1)) / count[k]) * sum[k]
//     out_sum[b] = Scum_b - Scum_{b-1},  out_mean[b] = out_sum[b] / (N / nb2)
// One warp per profile: lane l owns nb1/32 consecutive fine bins, a warp scan gives the
// cumulative count and sum at the start of its chunk, and the lane emits the boundaries that
// fall inside its bins.  fp64 throughout, every operation rounded once (no FMA).
// Optionally the merged profile is noise-normalised in the same pass.
#include "common.cuh"

namespace gpfc {

namespace {

constexpr int MERGE_THREADS = 256;   // fewer when nb2 is large (8 (nb2 + 1) bytes per warp)

__global__ void __launch_bounds__(MERGE_THREADS)
merge_equal_count_kernel(const float *__restrict__ sum, const uint32_t *__restrict__ count,
                         long long nprofiles, int nb1, int nb2, float *__restrict__ out_mean,
                         float *__restrict__ out_norm)
{
    extern __shared__ __align__(16) unsigned char merge_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double *scum = reinterpret_cast<double *>(merge_smem) + (size_t)warp * (nb2 + 1);
    const int chunk = (nb1 + 31) / 32;
    const int nwarps = blockDim.x >> 5;
    for (long long prof = (long long)blockIdx.x * nwarps + warp; prof < nprofiles;
         prof += (long long)gridDim.x * nwarps) {
        const float *s = sum + prof * nb1;
        const uint32_t *c = count + prof * nb1;
        const int k0 = min(nb1, lane * chunk), k1 = min(nb1, k0 + chunk);
        // chunk totals -> exclusive warp scan
        double cs = 0.0, ss = 0.0;
        for (int k = k0; k < k1; ++k) {
            cs += (double)c[k];
            ss += (double)s[k];
        }
        double cpre = cs, spre = ss;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            double a = __shfl_up_sync(0xffffffffu, cpre, o);
            double b = __shfl_up_sync(0xffffffffu, spre, o);
            if (lane >= o) {
                cpre += a;
                spre += b;
            }
        }
        const double total = __shfl_sync(0xffffffffu, cpre, 31);
        double cb = cpre - cs, sb = spre - ss;      // cumulative count / sum before fine bin k0
        __syncwarp();
        if (!(total > 0.0)) {
            for (int b = lane; b < nb2; b += 32) {
                if (out_mean) out_mean[prof * nb2 + b] = 0.f;
                if (out_norm) out_norm[prof * nb2 + b] = 0.f;
            }
            continue;
        }
        const double per = __ddiv_rn(total, (double)nb2);
        // first boundary whose target lies beyond the points before this chunk
        int b = (int)floor(__ddiv_rn(cb, per)) - 1;
        if (b < 0) b = 0;
        while (b < nb2 && !(((b == nb2 - 1) ? total : __dmul_rn(per, (double)(b + 1))) > cb)) ++b;
        if (lane == 0) b = 0;
        for (int k = k0; k < k1; ++k) {
            const double ck = (double)c[k], sk = (double)s[k];
            const double ca = cb + ck;
            const bool last = (k == nb1 - 1);
            while (b < nb2) {
                const double target = (b == nb2 - 1) ? total : __dmul_rn(per, (double)(b + 1));
                if (!last && ca < target) break;            // boundary lies in a later bin
                double frac = (ck > 0.0) ? __ddiv_rn(__dsub_rn(target, cb), ck) : 0.0;
                frac = fmin(fmax(frac, 0.0), 1.0);
                scum[b + 1] = __dadd_rn(sb, __dmul_rn(frac, sk));
                ++b;
            }
            cb = ca;
            sb += sk;
        }
        if (lane == 0) scum[0] = 0.0;
        __syncwarp();
        // differences, means, optional normalisation (mean kept, population std 1)
        double acc = 0.0;
        for (int bb = lane; bb < nb2; bb += 32) {
            const double m = __ddiv_rn(__dsub_rn(scum[bb + 1], scum[bb]), per);
            if (out_mean) out_mean[prof * nb2 + bb] = (float)m;
            acc += m;
        }
        if (out_norm) {
            acc = warp_sum(acc);
            const double mu = __ddiv_rn(acc, (double)nb2);
            double vacc = 0.0;
            for (int bb = lane; bb < nb2; bb += 32) {
                const double d = __dsub_rn(__ddiv_rn(__dsub_rn(scum[bb + 1], scum[bb]), per), mu);
                vacc += __dmul_rn(d, d);
            }
            vacc = warp_sum(vacc);
            const double sd = sqrt(__ddiv_rn(vacc, (double)nb2));
            const bool flat = (nb2 < 2) || !(sd > 0.0);
            for (int bb = lane; bb < nb2; bb += 32) {
                const double m = __ddiv_rn(__dsub_rn(scum[bb + 1], scum[bb]), per);
                const double o = flat ? mu : __dadd_rn(mu, __ddiv_rn(__dsub_rn(m, mu), sd));
                out_norm[prof * nb2 + bb] = (float)o;
            }
        }
        __syncwarp();
    }
}

}  // namespace

cudaError_t launch_merge(const float *sum, const uint32_t *count, long long nprofiles, int nb1,
                         int nb2, float *out_mean, float *out_norm, cudaStream_t st)
{
    if (nprofiles <= 0) return cudaSuccess;
    int warps = MERGE_THREADS / 32;
    while (warps > 1 && (size_t)warps * (nb2 + 1) * sizeof(double) > 96 * 1024) warps >>= 1;
    long long blocks = (nprofiles + warps - 1) / warps;
    if (blocks > 148LL * 16) blocks = 148LL * 16;
    size_t smem = (size_t)warps * (nb2 + 1) * sizeof(double);
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(merge_equal_count_kernel,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    merge_equal_count_kernel<<<(unsigned)blocks, warps * 32, smem, st>>>(
        sum, count, nprofiles, nb1, nb2, out_mean, out_norm);
    return cudaGetLastError();
}

}  // namespace gpfc
