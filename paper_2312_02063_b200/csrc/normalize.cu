// Stand-alone noise normalisation ("Lastly" + :63): one warp per
// profile, fp64 arithmetic, two-pass mean / population std over the non-empty
// bins.  Streams 8 B in and 4 B out per bin; the re-reads of a profile (<= 32 KB)
// hit L1/L2.
#include "common.cuh"

namespace gpfc {

namespace {

constexpr int NORM_THREADS = 256;

__global__ void __launch_bounds__(NORM_THREADS)
normalize_kernel(const float *__restrict__ sum, const uint32_t *__restrict__ count,
                 long long nprofiles, int nb, float *__restrict__ out)
{
    const int lane = threadIdx.x & 31;
    const long long wpb = NORM_THREADS / 32;
    for (long long prof = (long long)blockIdx.x * wpb + (threadIdx.x >> 5); prof < nprofiles;
         prof += (long long)gridDim.x * wpb) {
        const float *s = sum + prof * nb;
        const uint32_t *c = count + prof * nb;
        float *o = out + prof * nb;
        double acc = 0.0;
        int kk = 0;
        for (int k = lane; k < nb; k += 32) {
            uint32_t ck = c[k];
            if (ck > 0) {
                acc += __ddiv_rn((double)s[k], (double)ck);
                kk += 1;
            }
        }
        acc = warp_sum(acc);
        kk = warp_sum_int(kk);
        double mu = (kk > 0) ? __ddiv_rn(acc, (double)kk) : 0.0;
        double vacc = 0.0;
        for (int k = lane; k < nb; k += 32) {
            uint32_t ck = c[k];
            if (ck > 0) {
                double d = __dsub_rn(__ddiv_rn((double)s[k], (double)ck), mu);
                vacc += __dmul_rn(d, d);
            }
        }
        vacc = warp_sum(vacc);
        double sd = (kk > 0) ? sqrt(__ddiv_rn(vacc, (double)kk)) : 0.0;
        bool flat = (kk < 2) || !(sd > 0.0);
        for (int k = lane; k < nb; k += 32) {
            uint32_t ck = c[k];
            double v = mu;
            if (!flat && ck > 0) {
                double d = __dsub_rn(__ddiv_rn((double)s[k], (double)ck), mu);
                v = __dadd_rn(mu, __ddiv_rn(d, sd));
            }
            o[k] = (float)v;
        }
    }
}

}  // namespace

cudaError_t launch_normalize(const float *sum, const uint32_t *count, long long nprofiles,
                             int nbins, float *out, cudaStream_t st)
{
    if (nprofiles <= 0) return cudaSuccess;
    long long wpb = NORM_THREADS / 32;
    long long blocks = (nprofiles + wpb - 1) / wpb;
    if (blocks > 148LL * 32) blocks = 148LL * 32;
    normalize_kernel<<<(unsigned)blocks, NORM_THREADS, 0, st>>>(sum, count, nprofiles, nbins, out);
    note_launch();
    return cudaGetLastError();
}

}  // namespace gpfc
