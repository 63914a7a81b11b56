// Step 4 of the paper's fold ("Fourthly", Fig. 4(c)): merge the nb1
// equal-width intermediary bins of a folded profile into nb2 final bins that each hold the
// same number of points, scanning left to right and splitting a bin on a boundary pro rata
// by count (reading R18).  With N = total count and cumulative count / sum
// C(k), S(k) after fine bin k, output bin b ends at target_b = (N / nb2) (b + 1) (= N for
// the last bin) inside the first fine bin k with C(k) >= target_b:
//     Scum_b  = S(k-1) + ((target_b - C(k-1)) / count[k]) * sum[k]
//     out_sum[b] = Scum_b - Scum_{b-1},  out_mean[b] = out_sum[b] / (N / nb2)
// One warp per profile: the profile is staged in shared memory with coalesced loads (padded
// by one word per lane chunk, so the per-lane walks below are bank-conflict-free); lane l owns
// nb1/32 consecutive fine bins, a warp scan gives the cumulative count and sum at the start of
// its chunk, and the lane emits the boundaries that fall inside its bins.  fp64 throughout, every operation rounded once (no FMA).
// Optionally the merged profile is noise-normalised in the same pass.
#include "common.cuh"

namespace gpfc {

namespace {

constexpr int MERGE_THREADS = 512;   // fewer when nb2 is large (8 (nb2 + 1) bytes per warp)
constexpr int MERGE_SEG = 512;       // fine bins staged per pass (per warp: 4.3 KB)

__global__ void __launch_bounds__(MERGE_THREADS)
merge_equal_count_kernel(const float *__restrict__ sum, const uint32_t *__restrict__ count,
                         long long nprofiles, int nb1, int nb2, float *__restrict__ out_mean,
                         float *__restrict__ out_norm, const double *__restrict__ offset)
{
    // a constant the sums were taken relative to (the unfused route of gpfc_fold_two_tier passes
    // the curve's center): every output bin holds exactly N / nb2 points, so its mean shifts by it
    const double off = offset ? *offset : 0.0;
    extern __shared__ __align__(16) unsigned char merge_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nwarps = blockDim.x >> 5;
    const int seg = min(nb1, MERGE_SEG);
    const int chunk = (seg + 31) / 32;                    // bins per lane and segment
    const int pad = (chunk & 1) ? 0 : 1;                  // lane stride chunk + pad is odd
    const unsigned magic = (chunk > 1) ? (unsigned)((4294967296ull + chunk - 1) / chunk) : 0u;
    const int padded = seg + 32;
    double *scum = reinterpret_cast<double *>(merge_smem) + (size_t)warp * (nb2 + 1);
    float *fs = reinterpret_cast<float *>(reinterpret_cast<double *>(merge_smem) +
                                          (size_t)nwarps * (nb2 + 1)) + (size_t)warp * 2 * padded;
    uint32_t *fc = reinterpret_cast<uint32_t *>(fs + padded);
    for (long long prof = (long long)blockIdx.x * nwarps + warp; prof < nprofiles;
         prof += (long long)gridDim.x * nwarps) {
        const float *gs = sum + prof * nb1;
        const uint32_t *gc = count + prof * nb1;
        // total number of points of the profile
        unsigned tot_i = 0;
        for (int kb = 0; kb < nb1; kb += 256) {
            unsigned v[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int k = kb + j * 32 + lane;
                v[j] = (k < nb1) ? gc[k] : 0u;
            }
#pragma unroll
            for (int j = 0; j < 8; ++j) tot_i += v[j];
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) tot_i += __shfl_xor_sync(0xffffffffu, tot_i, o);
        const double total = (double)tot_i;
        if (tot_i == 0u) {
            for (int b = lane; b < nb2; b += 32) {
                if (out_mean) out_mean[prof * nb2 + b] = 0.f;
                if (out_norm) out_norm[prof * nb2 + b] = 0.f;
            }
            continue;
        }
        const double per = __ddiv_rn(total, (double)nb2);
        unsigned cum_c = 0;        // points before the current segment
        double cum_s = 0.0;        // flux before the current segment
        for (int s0 = 0; s0 < nb1; s0 += seg) {
            const int sn = min(seg, nb1 - s0);
            __syncwarp();
            // stage the segment: 8 independent coalesced loads in flight per array
            for (int kb = 0; kb < sn; kb += 256) {
                float vs[8];
                uint32_t vc[8];
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int k = kb + j * 32 + lane;
                    vs[j] = (k < sn) ? gs[s0 + k] : 0.f;
                    vc[j] = (k < sn) ? gc[s0 + k] : 0u;
                }
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int k = kb + j * 32 + lane;
                    if (k < sn) {
                        const int q = (chunk > 1) ? (int)__umulhi((unsigned)k, magic) : k;   // k / chunk
                        fs[k + pad * q] = vs[j];
                        fc[k + pad * q] = vc[j];
                    }
                }
            }
            __syncwarp();
            const int k0 = min(sn, lane * chunk), k1 = min(sn, k0 + chunk);
            const float *s = fs + pad * lane;            // s[k] for k in [k0, k1)
            const uint32_t *c = fc + pad * lane;
            // chunk totals -> exclusive warp scan
            unsigned cs = 0;
            double ss = 0.0;
            for (int k = k0; k < k1; ++k) {
                cs += c[k];
                ss += (double)s[k];
            }
            unsigned cpre = cs;
            double spre = ss;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                unsigned a = __shfl_up_sync(0xffffffffu, cpre, o);
                double b = __shfl_up_sync(0xffffffffu, spre, o);
                if (lane >= o) {
                    cpre += a;
                    spre += b;
                }
            }
            const unsigned seg_c = __shfl_sync(0xffffffffu, cpre, 31);
            const double seg_s = __shfl_sync(0xffffffffu, spre, 31);
            unsigned cbi = cum_c + (cpre - cs);           // points before fine bin s0 + k0
            double sb = cum_s + (spre - ss);              // flux before it
            // first boundary whose target lies beyond the points before this chunk
            const double cbd0 = (double)cbi;
            int b = (int)floor(__ddiv_rn(cbd0, per)) - 1;
            if (b < 0) b = 0;
            while (b < nb2 && !(((b == nb2 - 1) ? total : __dmul_rn(per, (double)(b + 1))) > cbd0)) ++b;
            if (cbi == 0u) b = 0;
            // walk this lane's bins.  Counts are integers, so "C(k) >= target" is the integer
            // test C(k) > thr with thr = ceil(target) - 1; fp64 only when a boundary is emitted.
            double target = (b < nb2) ? ((b == nb2 - 1) ? total : __dmul_rn(per, (double)(b + 1))) : 0.0;
            unsigned thr = (b < nb2) ? (unsigned)ceil(target) - 1u : 0xffffffffu;
            for (int k = k0; k < k1; ++k) {
                const unsigned cki = c[k];
                const double sk = (double)s[k];
                const unsigned cai = cbi + cki;
                const bool last = (s0 + k == nb1 - 1);
                if (b < nb2 && (last || cai > thr)) {
                    const double ck = (double)cki, cbd = (double)cbi;
                    do {
                        double frac = (cki > 0u) ? __ddiv_rn(__dsub_rn(target, cbd), ck) : 0.0;
                        frac = fmin(fmax(frac, 0.0), 1.0);
                        scum[b + 1] = __dadd_rn(sb, __dmul_rn(frac, sk));
                        ++b;
                        if (b < nb2) {
                            target = (b == nb2 - 1) ? total : __dmul_rn(per, (double)(b + 1));
                            thr = (unsigned)ceil(target) - 1u;
                        }
                    } while (b < nb2 && (last || cai > thr));
                }
                cbi = cai;
                sb += sk;
            }
            cum_c += seg_c;
            cum_s += seg_s;
        }
        if (lane == 0) scum[0] = 0.0;
        __syncwarp();
        // differences, means, optional normalisation (mean kept, population std 1)
        double acc = 0.0;
        for (int bb = lane; bb < nb2; bb += 32) {
            const double m = __ddiv_rn(__dsub_rn(scum[bb + 1], scum[bb]), per);
            if (out_mean) out_mean[prof * nb2 + bb] = (float)__dadd_rn(m, off);
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
                const double o = flat ? __dadd_rn(mu, off)
                                      : __dadd_rn(__dadd_rn(mu, off), __ddiv_rn(__dsub_rn(m, mu), sd));
                out_norm[prof * nb2 + bb] = (float)o;
            }
        }
        __syncwarp();
    }
}

}  // namespace

cudaError_t merge_init_device()
{
    return cudaFuncSetAttribute(merge_equal_count_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                200 * 1024);
}

cudaError_t launch_merge(const float *sum, const uint32_t *count, long long nprofiles, int nb1,
                         int nb2, float *out_mean, float *out_norm, const double *offset,
                         cudaStream_t st)
{
    if (nprofiles <= 0) return cudaSuccess;
    int warps = MERGE_THREADS / 32;
    const int seg = nb1 < MERGE_SEG ? nb1 : MERGE_SEG;
    const size_t per_warp = (size_t)(nb2 + 1) * sizeof(double) + (size_t)2 * (seg + 32) * 4;
    while (warps > 1 && (size_t)warps * per_warp > 200 * 1024) --warps;
    long long blocks = (nprofiles + warps - 1) / warps;
    if (blocks > 148LL * 16) blocks = 148LL * 16;
    size_t smem = (size_t)warps * per_warp;
    merge_equal_count_kernel<<<(unsigned)blocks, warps * 32, smem, st>>>(
        sum, count, nprofiles, nb1, nb2, out_mean, out_norm, offset);
    note_launch();
    return cudaGetLastError();
}

}  // namespace gpfc
