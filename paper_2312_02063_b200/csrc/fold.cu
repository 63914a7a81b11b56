// The fold kernels (PAPER.md:111 steps 1-3 and 5; noise normalisation :63 fused
// into the epilogue).  See DESIGN.md "Kernel design".
//
// fold_cols_kernel (power-of-two nbins, 32..4096): one persistent CTA per SM.  A
// work item is (curve, group of PB consecutive trial periods).  All warps of the
// CTA stream through the curve's conditioned samples (u, q) -- each lane keeps KS
// samples in registers and reuses them for the PB periods -- and update a
// shared-memory histogram laid out [period][sum|count][bin][COLS] with native
// 32-bit shared atomics (ATOMS.ADD / ATOMS.POPC.INC).  With COLS = 32 every lane
// owns a bank, so each atomic instruction is one conflict-free wavefront; the
// atomics only arbitrate between warps.  No global atomics anywhere.
//
// Phase math per point-period: y = u * rp (DMUL), m = RD(y + 1.5*2^(20+NBLOG))
// (DADD.RM): the low word of m holds floor(y) mod nbins in its top NBLOG bits and
// g = 32 - NBLOG fraction bits below.  The fast bin can differ from the exact
// formula (true division, include/gpfc.h) only if y is within 2^-g of an integer,
// i.e. only if those g bits are all 0 or all 1; a running unsigned-min over
// (lo + 1) << NBLOG detects that for a whole register tile, and the rare tile
// that trips it is re-checked sample by sample against the exact formula and
// corrected with compensating atomics.  Proof of the bound: DESIGN.md "Exact bins".
//
// Epilogue: ATOMS.EXCH reads and clears the columns in one pass (each lane owns
// one bin and walks the columns diagonally, conflict-free), the per-bin totals go
// to 8-byte slots, and one warp per period converts / normalises / stores the
// profile with coalesced writes while the other warps already fold the next item.
#include "common.cuh"

namespace gpfc {

namespace {

constexpr int FOLD_THREADS = 1024;
constexpr int FOLD_WARPS = FOLD_THREADS / 32;

template <int NBLOG, int COLSLOG, int PB>
struct Cfg {
    static constexpr int NB = 1 << NBLOG;
    static constexpr int COLS = 1 << COLSLOG;
    static constexpr int HW = NB * COLS;                 // words per (period, array)
    static constexpr int CHUNKS = NB / 32;
    static constexpr int WANT = (2 * FOLD_WARPS + PB * CHUNKS - 1) / (PB * CHUNKS);
    static constexpr int CSPLIT = WANT <= 1 ? 1 : (WANT <= 2 ? 2 : (WANT <= 4 ? 4 : 8));
    static constexpr int CS = CSPLIT > COLS ? COLS : CSPLIT;
    static constexpr size_t SMEM = (size_t)PB * 2 * HW * 4 + (size_t)PB * NB * 8 + 16;
};

template <int NBLOG, int COLSLOG, int PB, int KS>
__global__ void __launch_bounds__(FOLD_THREADS, 1)
fold_cols_kernel(FoldArgs a, long long ngroups, long long nitems)
{
    using C = Cfg<NBLOG, COLSLOG, PB>;
    constexpr int NB = C::NB, COLS = C::COLS, HW = C::HW;
    constexpr int TILE = 32 * KS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    int *H = reinterpret_cast<int *>(smem_raw);                       // [PB][2][HW]
    unsigned long long *R = reinterpret_cast<unsigned long long *>(H + PB * 2 * HW);  // [PB][NB]
    int *ctr = reinterpret_cast<int *>(R + PB * NB);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int col = lane & (COLS - 1);
    for (int i = tid; i < PB * 2 * HW; i += FOLD_THREADS) H[i] = 0;
    for (int i = tid; i < PB * NB; i += FOLD_THREADS) R[i] = 0ull;
    if (tid == 0) *ctr = 0;
    __syncthreads();

    // 1.5 * 2^(52 - g), g = 32 - NBLOG
    const double MAGIC = 6755399441055744.0 / (double)(1ull << (32 - NBLOG));
    const double YLIM = (double)(1ull << (18 + NBLOG));

    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        const long long curve = item / ngroups;
        const long long p0 = (item - curve * ngroups) * PB;
        const int np = (int)((a.nperiods - p0) < PB ? (a.nperiods - p0) : PB);
        const CurveMeta m = a.meta[curve];
        const int n = m.n_valid;
        const double *__restrict__ u = a.u + m.start;
        const int *__restrict__ q = a.q + m.start;
        const int ntiles = (n + TILE - 1) / TILE;

        double r[PB];
        bool fast = (np == PB) && (m.umin >= 0.0);
#pragma unroll
        for (int p = 0; p < PB; ++p) {
            r[p] = (p < np) ? a.rp[p0 + p] : 0.0;
            fast = fast && (r[p] * m.umax < YLIM);     // false for NaN
        }

        if (fast) {
            for (;;) {
                int tile = 0;
                if (lane == 0) tile = atomicAdd(ctr, 1);
                tile = __shfl_sync(0xffffffffu, tile, 0);
                if (tile >= ntiles) break;
                const int base = tile * TILE;
                double uu[KS];
                int qq[KS];
                bool ok[KS];
                const bool full = (base + TILE <= n);
#pragma unroll
                for (int k = 0; k < KS; ++k) {
                    int idx = base + k * 32 + lane;
                    ok[k] = full || (idx < n);
                    uu[k] = ok[k] ? u[idx] : 0.5;
                    qq[k] = ok[k] ? q[idx] : 0;
                }
                unsigned gmin = 0xffffffffu;
                if (full) {
#pragma unroll
                    for (int p = 0; p < PB; ++p) {
#pragma unroll
                        for (int k = 0; k < KS; ++k) {
                            double y = __dmul_rn(uu[k], r[p]);
                            double mm = __dadd_rd(y, MAGIC);
                            unsigned lo = (unsigned)__double2loint(mm);
                            unsigned bin = lo >> (32 - NBLOG);
                            gmin = min(gmin, lo * (unsigned)NB + (unsigned)NB);
                            int *hs = H + p * 2 * HW + bin * COLS + col;
                            atomicAdd(hs, qq[k]);
                            atomicAdd(reinterpret_cast<unsigned *>(hs + HW), 1u);
                        }
                    }
                } else {
#pragma unroll
                    for (int p = 0; p < PB; ++p) {
#pragma unroll
                        for (int k = 0; k < KS; ++k) {
                            double y = __dmul_rn(uu[k], r[p]);
                            double mm = __dadd_rd(y, MAGIC);
                            unsigned lo = (unsigned)__double2loint(mm);
                            unsigned bin = lo >> (32 - NBLOG);
                            if (ok[k]) {
                                gmin = min(gmin, lo * (unsigned)NB + (unsigned)NB);
                                int *hs = H + p * 2 * HW + bin * COLS + col;
                                atomicAdd(hs, qq[k]);
                                atomicAdd(reinterpret_cast<unsigned *>(hs + HW), 1u);
                            }
                        }
                    }
                }
                if (gmin <= (unsigned)NB) {
                    // rare: some y sat within 2^-g of an integer.  Re-check against the
                    // exact formula and move the sample if the fast bin was wrong.
#pragma unroll
                    for (int p = 0; p < PB; ++p) {
#pragma unroll
                        for (int k = 0; k < KS; ++k) {
                            double y = __dmul_rn(uu[k], r[p]);
                            double mm = __dadd_rd(y, MAGIC);
                            unsigned lo = (unsigned)__double2loint(mm);
                            if (ok[k] && (lo * (unsigned)NB + (unsigned)NB) <= (unsigned)NB) {
                                int kf = (int)(lo >> (32 - NBLOG));
                                int ke = exact_bin(uu[k], a.periods[p0 + p], NB);
                                if (ke != kf) {
                                    int *hf = H + p * 2 * HW + kf * COLS + col;
                                    atomicAdd(hf, -qq[k]);
                                    atomicSub(reinterpret_cast<unsigned *>(hf + HW), 1u);
                                    if (ke >= 0) {
                                        int *he = H + p * 2 * HW + ke * COLS + col;
                                        atomicAdd(he, qq[k]);
                                        atomicAdd(reinterpret_cast<unsigned *>(he + HW), 1u);
                                    }
                                }
                            }
                        }
                    }
                }
            }
        } else {
            // exact path: negative u, a period outside the fast range, an invalid
            // period (row stays zero) or a ragged last group.
            double per[PB];
#pragma unroll
            for (int p = 0; p < PB; ++p) per[p] = (p < np) ? a.periods[p0 + p] : 0.0;
            for (;;) {
                int tile = 0;
                if (lane == 0) tile = atomicAdd(ctr, 1);
                tile = __shfl_sync(0xffffffffu, tile, 0);
                if (tile >= ntiles) break;
                const int base = tile * TILE;
#pragma unroll
                for (int k = 0; k < KS; ++k) {
                    int idx = base + k * 32 + lane;
                    if (idx < n) {
                        double ui = u[idx];
                        int qi = q[idx];
#pragma unroll
                        for (int p = 0; p < PB; ++p) {
                            if (period_ok(per[p])) {
                                int ke = exact_bin(ui, per[p], NB);
                                if (ke < 0) continue;
                                int *he = H + p * 2 * HW + ke * COLS + col;
                                atomicAdd(he, qi);
                                atomicAdd(reinterpret_cast<unsigned *>(he + HW), 1u);
                            }
                        }
                    }
                }
            }
        }
        __syncthreads();   // A: every update of this item is in H

        // E1: read-and-clear the columns; lane owns bin, walks the columns diagonally
        constexpr int CS = C::CS;
        constexpr int CPP = COLS / CS;       // columns per part
        constexpr int UNITS = PB * C::CHUNKS * CS;
        for (int unit = warp; unit < UNITS; unit += FOLD_WARPS) {
            const int part = unit % CS;
            const int chunk = (unit / CS) % C::CHUNKS;
            const int p = unit / (CS * C::CHUNKS);
            const int bin = chunk * 32 + lane;
            int *hs = H + p * 2 * HW + bin * COLS;
            int s = 0;
            unsigned c = 0;
#pragma unroll 8
            for (int k = 0; k < CPP; ++k) {
                int cc = (lane + k + part * CPP) & (COLS - 1);
                s += atomicExch(hs + cc, 0);
                c += atomicExch(reinterpret_cast<unsigned *>(hs + HW + cc), 0u);
            }
            unsigned *slot = reinterpret_cast<unsigned *>(R + p * NB + bin);
            if (CS == 1) {
                slot[0] = (unsigned)s;
                slot[1] = c;
            } else {
                atomicAdd(slot, (unsigned)s);
                atomicAdd(slot + 1, c);
            }
        }
        if (tid == 0) *ctr = 0;
        __syncthreads();   // B: totals are in R, H is zero again, tile counter reset

        // E2: one warp per period converts / normalises / stores; the rest move on
        if (warp < np) {
            const long long row = (curve * a.nperiods + p0 + warp) * (long long)NB;
            emit_profile(R + warp * NB, NB, lane, m.inv_scale, m.center, false,
                         a.out_sum ? a.out_sum + row : nullptr,
                         a.out_count ? a.out_count + row : nullptr,
                         a.out_norm ? a.out_norm + row : nullptr);
        }
    }
}

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
        if (m.n_valid < a.n_min || m.n_valid > a.n_max) continue;   // another launch owns it
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
        if (tid < 32) {
            const long long row = (curve * a.nperiods + j) * (long long)nb;
            emit_profile(R, nb, tid, m.inv_scale, m.center, false,
                         a.out_sum ? a.out_sum + row : nullptr,
                         a.out_count ? a.out_count + row : nullptr,
                         a.out_norm ? a.out_norm + row : nullptr);
        }
        __syncthreads();
    }
}

template <int NBLOG, int COLSLOG, int PB, int KS>
cudaError_t launch_cols(const FoldArgs &a, cudaStream_t st)
{
    using C = Cfg<NBLOG, COLSLOG, PB>;
    auto kern = fold_cols_kernel<NBLOG, COLSLOG, PB, KS>;
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)C::SMEM);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    long long ngroups = (a.nperiods + PB - 1) / PB;
    long long nitems = ngroups * a.ncurves;
    long long grid = nitems < num_sms() ? nitems : num_sms();
    kern<<<(unsigned)grid, FOLD_THREADS, C::SMEM, st>>>(a, ngroups, nitems);
    return cudaGetLastError();
}

}  // namespace

int num_sms()
{
    static int g_num_sms = 0;
    if (g_num_sms == 0) {
        int dev = 0, n = 0;
        if (cudaGetDevice(&dev) == cudaSuccess &&
            cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n > 0)
            g_num_sms = n;
        else
            return 148;
    }
    return g_num_sms;
}

cudaError_t launch_fold(const FoldArgs &a, cudaStream_t st)
{
    if (a.ncurves <= 0 || a.nperiods <= 0) return cudaSuccess;
    if (fold_lp_handles(a.nbins)) return launch_fold_lp(a, st);
    switch (a.nbins) {
        case 2048: return launch_cols<11, 3, 1, 4>(a, st);
        case 4096: return launch_cols<12, 2, 1, 4>(a, st);
        default: break;
    }
    return launch_fold_generic(a, st);
}

cudaError_t launch_fold_generic(const FoldArgs &a, cudaStream_t st)
{
    if (a.ncurves <= 0 || a.nperiods <= 0) return cudaSuccess;
    long long nitems = a.ncurves * a.nperiods;
    long long cap = (long long)num_sms() * 8;
    long long grid = nitems < cap ? nitems : cap;
    fold_generic_kernel<<<(unsigned)grid, GEN_THREADS, (size_t)a.nbins * 8, st>>>(a, nitems);
    return cudaGetLastError();
}

}  // namespace gpfc
