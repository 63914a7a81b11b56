// Dispatch of the fold (PAPER.md:111 steps 1-3 and 5; noise normalisation :63 fused into the
// epilogues) and the generic kernel.  The tuned kernels live in fold_lp.cu (any nbins up to 256,
// lane = period) and fold_pk.cu (nbins 512 ... 4096, powers of two, packed counts, optional
// fused equal-count merge); every other nbins in [257, 4096] takes fold_generic_kernel below: one CTA per
// (curve, period), the exact formula (true division) for every point-period.  It is the
// correctness path for bin counts that are not a power of two, not a tuned one; launches of
// it are counted (gpfc_profile_read) so that a caller can see when it was taken.
#include "common.cuh"

namespace gpfc {

namespace {

// Generic kernel: any nbins in [1, 4096], exact formula for every point-period,
// one CTA per (curve, period), CTA-shared histogram of 8-byte slots.
constexpr int GEN_THREADS = 256;

__global__ void __launch_bounds__(GEN_THREADS)
fold_generic_kernel(FoldArgs a, long long nitems)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    unsigned long long *R = reinterpret_cast<unsigned long long *>(smem_raw);
    const int nb = a.nbins;
    const int tid = threadIdx.x;
    for (int i = tid; i < nb; i += GEN_THREADS) R[i] = 0ull;
    __syncthreads();
    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        const long long curve = item / a.nperiods;
        const long long j = item - curve * a.nperiods;
        const CurveMeta m = a.meta[curve];
        const double per = a.periods[j];
        if (period_ok(per)) {
            const double *__restrict__ u = a.u + m.start;
            const int *__restrict__ q = a.q + m.start;
            for (int i = tid; i < m.n_valid; i += GEN_THREADS) {
                int ke = exact_bin(u[i], per, nb);
                if (ke < 0) continue;
                unsigned *slot = reinterpret_cast<unsigned *>(R + ke);
                atomicAdd(slot, (unsigned)q[i]);
                atomicAdd(slot + 1, 1u);
            }
        }
        __syncthreads();
        if (tid == 0 && m.n_zero > 0 && period_ok(per)) {
            // the samples at u == 0 (CurveMeta::n_zero) are not in the sample arrays: bin 0
            unsigned *slot = reinterpret_cast<unsigned *>(R);
            slot[0] += (unsigned)m.q_zero;
            slot[1] += (unsigned)m.n_zero;
        }
        __syncthreads();
        if (tid < 32) {
            const long long row = (curve * a.nperiods + j) * (long long)nb;
            if (a.center_out && j == 0 && tid == 0) a.center_out[curve] = m.center;
            // centred sums (FoldArgs::center_out) come without a normalised profile (api.cu)
            emit_profile(R, nb, tid, m.inv_scale, a.center_out ? 0.0 : m.center, false,
                         a.out_sum ? a.out_sum + row : nullptr,
                         a.out_count ? a.out_count + row : nullptr,
                         a.out_norm ? a.out_norm + row : nullptr);
        }
        __syncthreads();
    }
}

}  // namespace

int fold_rows(int nbins)
{
    if (fold_lp_handles(nbins)) return fold_lp_pow2(nbins) ? 256 : 1;
    if (fold_pk_handles(nbins)) return fold_pk_rows(nbins);
    return nbins;
}

cudaError_t launch_fold(const FoldArgs &a, cudaStream_t st)
{
    if (a.ncurves <= 0 || a.nperiods <= 0) return cudaSuccess;
    const DeviceInfo *di = nullptr;
    cudaError_t e = device_info(&di);
    if (e != cudaSuccess) return e;
    if (fold_lp_handles(a.nbins)) return launch_fold_lp(a, st, di->num_sms);
    if (fold_pk_handles(a.nbins)) return launch_fold_pk(a, st, di->num_sms);
    return launch_fold_generic(a, st, di->num_sms);
}

cudaError_t launch_fold_generic(const FoldArgs &a, cudaStream_t st, int sms)
{
    if (a.ncurves <= 0 || a.nperiods <= 0) return cudaSuccess;
    long long nitems = a.ncurves * a.nperiods;
    long long cap = (long long)sms * 8;
    long long grid = nitems < cap ? nitems : cap;
    fold_generic_kernel<<<(unsigned)grid, GEN_THREADS, (size_t)a.nbins * 8, st>>>(a, nitems);
    note_launch();
    return cudaGetLastError();
}

}  // namespace gpfc
