// fold_lp_kernel: the "lane = period" fold for power-of-two nbins in [32, 256]
// (PAPER.md:111 steps 1-3 and 5, noise normalisation :63 fused into the epilogue).
// DESIGN.md "Kernel design" has the full derivation; in short:
//
// * One persistent CTA per SM.  A work item is (curve, group of 32*R consecutive trial
//   periods).  Lane l of EVERY warp owns the R periods p0 + r*32 + l; the warps split
//   the curve's samples (anchor tiles of GPFC_TILE samples, handed out dynamically).
// * The histograms of the group live in shared memory as [r][row 0..255][sum|count][lane]
//   32-bit words: a warp-wide update touches 32 different banks whatever the bins are
//   (bank = lane), so every ATOMS is one conflict-free wavefront; the atomics only
//   arbitrate between warps.  No replication, hence no column reduction afterwards, and
//   32*R periods share every sample load.  No global atomics anywhere.
// * Samples are staged per warp in shared memory with coalesced 16-byte loads and read
//   back with one broadcast LDS.128 per sample {v, q}.
// * Phase math per point-period is ONE fp64 instruction: m = RD(v * rp + C) (DFMA.RM),
//   v = u - a the sample's offset from its tile anchor, rp = 256 * RN(1/P),
//   C = 2^20 + delta + ((a * rp) mod 256) set up once per (tile, period).  ulp(m) = 2^-32:
//   the low word of m is the fraction of the row coordinate, bits 0..7 of the high word
//   are the row.  One PRMT builds the shared-memory address (row * 256 + lane * 4), one
//   VIMNMX keeps the smallest fraction seen: 5 instructions per point-period with the two
//   atomics.
// * Exactness: the row can differ from the exact formula (true division, gpfc.h) only
//   if the fraction is below D = 2 * delta (DESIGN.md "Exact bins" derives delta from the
//   rounding errors); a tile whose running minimum trips that is re-checked sample by
//   sample against the exact formula and corrected with compensating atomics.
// * nbins < 256 folds at 256 rows and merges 256 / nbins adjacent rows at write-out
//   (exact: floor(phi * 256) >> k == floor(phi * (256 >> k))).
// * Epilogue: lane l walks ITS periods' rows (conflict-free), so mean / std need no
//   cross-lane reduction; every lane writes 32-byte sectors (8 bins) of its own rows.
#include "common.cuh"

namespace gpfc {

namespace {

constexpr int LP_THREADS = 512;
constexpr int LP_WARPS = LP_THREADS / 32;
constexpr int LP_R = 3;                       // periods per lane
constexpr int LP_GROUP = 32 * LP_R;           // periods per work item
constexpr int LP_ROWS = 256;                  // rows per period (fold resolution)
constexpr int LP_GRAN = 64;                   // samples per staging granule
constexpr int LP_PARTS = 4;                   // bin ranges per period in the statistics sweeps
constexpr unsigned LP_SMEM_BASE = 0x400;      // shared-window address of dynamic shared memory

constexpr int LP_HIST_BYTES = LP_R * LP_ROWS * 256;           // 196,608
constexpr int LP_STAGE_OFF = LP_HIST_BYTES;                   // int4 [LP_WARPS][LP_GRAN]
constexpr int LP_STAGE_BYTES = LP_WARPS * LP_GRAN * 16;
constexpr int LP_PART_OFF = LP_STAGE_OFF + LP_STAGE_BYTES;    // double [LP_PARTS][LP_GROUP]
constexpr int LP_PARTK_OFF = LP_PART_OFF + LP_PARTS * LP_GROUP * 8;   // int [LP_PARTS][LP_GROUP]
constexpr int LP_MU_OFF = LP_PARTK_OFF + LP_PARTS * LP_GROUP * 4;     // double [LP_GROUP]
constexpr int LP_ISD_OFF = LP_MU_OFF + LP_GROUP * 8;                  // double [LP_GROUP]
constexpr int LP_KK_OFF = LP_ISD_OFF + LP_GROUP * 8;                  // int [LP_GROUP]
constexpr int LP_CTR_OFF = LP_KK_OFF + LP_GROUP * 4;
constexpr int LP_SMEM_BYTES = LP_CTR_OFF + 16;
static_assert(LP_SMEM_BYTES <= 227 * 1024, "shared memory budget");
static_assert(LP_R * LP_PARTS <= LP_WARPS, "statistics sweep needs R * PARTS warps");

// shared-memory reductions with an immediate offset: ATOMS.ADD / ATOMS.POPC.INC
template <int IMM>
__device__ __forceinline__ void red_add(unsigned addr, int v)
{
    asm volatile("red.shared.add.u32 [%0+%2], %1;" ::"r"(addr), "r"(v), "n"(IMM) : "memory");
}
template <int IMM>
__device__ __forceinline__ void red_inc(unsigned addr)
{
    asm volatile("red.shared.add.u32 [%0+%1], 1;" ::"r"(addr), "n"(IMM) : "memory");
}

// word index of (r, row, array, lane) in the histogram
__device__ __forceinline__ int hidx(int r, int row, int arr, int lane)
{
    return r * (LP_ROWS * 64) + row * 64 + arr * 32 + lane;
}

// one point-period of the fast path for period slot r (compile-time)
template <int r>
__device__ __forceinline__ void pp_update(double v, int q, double rp, double C, unsigned lane4,
                                          unsigned &gmin)
{
    double m = __fma_rd(v, rp, C);
    unsigned lo = (unsigned)__double2loint(m), hi = (unsigned)__double2hiint(m);
    unsigned addr = __byte_perm(lane4, hi, 0x3240);      // (row << 8) | (lane << 2)
    gmin = min(gmin, lo);
    red_add<(int)LP_SMEM_BASE + r * 65536>(addr, q);
    red_inc<(int)LP_SMEM_BASE + r * 65536 + 128>(addr);
}

template <int r0>
struct ForR {
    __device__ __forceinline__ static void run(double v, int q, const double (&rp)[LP_R],
                                               const double (&C)[LP_R], unsigned lane4,
                                               unsigned &gmin)
    {
        pp_update<r0>(v, q, rp[r0], C[r0], lane4, gmin);
        ForR<r0 + 1>::run(v, q, rp, C, lane4, gmin);
    }
};
template <>
struct ForR<LP_R> {
    __device__ __forceinline__ static void run(double, int, const double (&)[LP_R],
                                               const double (&)[LP_R], unsigned, unsigned &) {}
};

__global__ void __launch_bounds__(LP_THREADS, 1)
fold_lp_kernel(FoldArgs a, long long ngroups, long long nitems, unsigned *probe)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    if (probe) {   // report where dynamic shared memory starts (host checks LP_SMEM_BASE once)
        if (threadIdx.x == 0 && blockIdx.x == 0) *probe = (unsigned)__cvta_generic_to_shared(smem);
        return;
    }
    unsigned *H = reinterpret_cast<unsigned *>(smem);
    int4 *stage_all = reinterpret_cast<int4 *>(smem + LP_STAGE_OFF);
    double *part_s = reinterpret_cast<double *>(smem + LP_PART_OFF);
    int *part_k = reinterpret_cast<int *>(smem + LP_PARTK_OFF);
    double *st_mu = reinterpret_cast<double *>(smem + LP_MU_OFF);
    double *st_isd = reinterpret_cast<double *>(smem + LP_ISD_OFF);
    int *st_kk = reinterpret_cast<int *>(smem + LP_KK_OFF);
    int *ctr = reinterpret_cast<int *>(smem + LP_CTR_OFF);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned lane4 = (unsigned)lane << 2;
    int4 *stage = stage_all + warp * LP_GRAN;
    for (int i = tid; i < LP_HIST_BYTES / 4; i += LP_THREADS) H[i] = 0u;
    if (tid == 0) *ctr = 0;
    __syncthreads();

    const int nb = a.nbins;                      // 32, 64, 128 or 256
    const int mshift = 8 - (31 - __clz(nb));     // rows merged per bin = 1 << mshift
    const int M = 1 << mshift;
    const double M2 = 1729382256910270464.0;     // 1.5 * 2^60: ulp = 256

    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        const long long curve = item / ngroups;
        const long long p0 = (item - curve * ngroups) * LP_GROUP;
        const CurveMeta cm = a.meta[curve];
        const int n = cm.n_valid;
        const int ntiles = (n + GPFC_TILE - 1) / GPFC_TILE;

        // this lane's periods
        double rp[LP_R];
        bool valid[LP_R];
        double rpmax = 0.0;
#pragma unroll
        for (int r = 0; r < LP_R; ++r) {
            long long j = p0 + r * 32 + lane;
            double x = (j < a.nperiods) ? a.rp[j] : CUDART_NAN;
            valid[r] = (x == x);
            rp[r] = valid[r] ? x : 256.0;          // dummy period: its columns are never written out
            if (valid[r]) rpmax = fmax(rpmax, x);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) rpmax = fmax(rpmax, __shfl_xor_sync(0xffffffffu, rpmax, o));

        // guard band, in units of 2^-32 row:
        //   E <= 4 * 2^-53 * max|u| * rpmax + 2^-33 + 2^-46  ->  eunits = 4 U rpmax 2^-21 + 1
        //   delta >= E + 1 unit, D = 2 delta  ->  D >= 2 eunits + 2
        const double U = fmax(fabs(cm.umin), fabs(cm.umax));
        const double need = 2.0 * (4.0 * U * rpmax * (1.0 / 2097152.0) + 1.0) + 2.0;
        unsigned D = 16u;
        while ((double)D < need && D < 32768u) D <<= 1;
        const bool fast = (need <= 16384.0) && (cm.span_max * rpmax + 512.0 < 1048576.0);
        const double K = 1048576.0 + (double)(D >> 1) * (1.0 / 4294967296.0);

        if (fast) {
            for (;;) {
                int t = 0;
                if (lane == 0) t = atomicAdd(ctr, 1);
                t = __shfl_sync(0xffffffffu, t, 0);
                if (t >= ntiles) break;
                const int base = t * GPFC_TILE;
                const int cnt = min(GPFC_TILE, n - base);
                const TileInfo ti = a.tiles[cm.tile0 + t];
                double C[LP_R];
#pragma unroll
                for (int r = 0; r < LP_R; ++r) {
                    double w = __fma_rd(ti.a, rp[r], M2);       // M2 + 256 * floor(a rp / 256)
                    double z = __dsub_rn(w, M2);
                    double c1 = __fma_rn(ti.a, rp[r], -z);      // (a rp) mod 256, error <= 2^-46
                    C[r] = __dadd_rn(c1, K);
                }
                const int4 *src = a.rec + cm.start + base;
                unsigned gmin = 0xffffffffu;
                int4 n0 = make_int4(0, 0, 0, 0), n1 = n0;
                if (lane < cnt) n0 = __ldg(src + lane);
                if (lane + 32 < cnt) n1 = __ldg(src + lane + 32);
                for (int g0 = 0; g0 < cnt; g0 += LP_GRAN) {
                    const int gc = min(LP_GRAN, cnt - g0);
                    __syncwarp();
                    stage[lane] = n0;
                    stage[lane + 32] = n1;
                    __syncwarp();
                    if (g0 + LP_GRAN + lane < cnt) n0 = __ldg(src + g0 + LP_GRAN + lane);
                    if (g0 + LP_GRAN + lane + 32 < cnt) n1 = __ldg(src + g0 + LP_GRAN + lane + 32);
                    if (gc == LP_GRAN) {
#pragma unroll 1
                        for (int s = 0; s < LP_GRAN; s += 4) {
                            int4 rc[4];
#pragma unroll
                            for (int k = 0; k < 4; ++k) rc[k] = stage[s + k];
#pragma unroll
                            for (int k = 0; k < 4; ++k)
                                ForR<0>::run(__hiloint2double(rc[k].y, rc[k].x), rc[k].z, rp, C,
                                             lane4, gmin);
                        }
                    } else {
#pragma unroll 1
                        for (int s = 0; s < gc; ++s) {
                            int4 rc = stage[s];
                            ForR<0>::run(__hiloint2double(rc.y, rc.x), rc.z, rp, C, lane4, gmin);
                        }
                    }
                }
                if (__any_sync(0xffffffffu, gmin < D)) {
                    // rare: some row coordinate sat within the guard band of an integer.
                    // Re-check those samples against the exact formula; move the ones that
                    // the fast path put in the wrong row.
                    if (gmin < D) {
                        const double *us = a.u + cm.start + base;
#pragma unroll
                        for (int r = 0; r < LP_R; ++r) {
                            if (!valid[r]) continue;
                            const double per = a.periods[p0 + r * 32 + lane];
#pragma unroll 1
                            for (int s = 0; s < cnt; ++s) {
                                int4 rc = __ldg(src + s);
                                double m = __fma_rd(__hiloint2double(rc.y, rc.x), rp[r], C[r]);
                                if ((unsigned)__double2loint(m) < D) {
                                    int kf = __double2hiint(m) & (LP_ROWS - 1);
                                    int ke = exact_bin(us[s], per, LP_ROWS);
                                    if (ke != kf) {
                                        atomicAdd(&H[hidx(r, kf, 0, lane)], (unsigned)(-rc.z));
                                        atomicSub(&H[hidx(r, kf, 1, lane)], 1u);
                                        atomicAdd(&H[hidx(r, ke, 0, lane)], (unsigned)rc.z);
                                        atomicAdd(&H[hidx(r, ke, 1, lane)], 1u);
                                    }
                                }
                            }
                        }
                    }
                }
            }
        } else {
            // exact path: a period far outside the fast range or a tile spanning a huge gap
            double per[LP_R];
#pragma unroll
            for (int r = 0; r < LP_R; ++r)
                per[r] = valid[r] ? a.periods[p0 + r * 32 + lane] : 1.0;
            for (;;) {
                int t = 0;
                if (lane == 0) t = atomicAdd(ctr, 1);
                t = __shfl_sync(0xffffffffu, t, 0);
                if (t >= ntiles) break;
                const int base = t * GPFC_TILE;
                const int cnt = min(GPFC_TILE, n - base);
                const double *us = a.u + cm.start + base;
                const int *qs = a.q + cm.start + base;
#pragma unroll 1
                for (int s = 0; s < cnt; ++s) {
                    const double ui = us[s];
                    const int qi = qs[s];
#pragma unroll
                    for (int r = 0; r < LP_R; ++r) {
                        if (valid[r]) {
                            int ke = exact_bin(ui, per[r], LP_ROWS);
                            atomicAdd(&H[hidx(r, ke, 0, lane)], (unsigned)qi);
                            atomicAdd(&H[hidx(r, ke, 1, lane)], 1u);
                        }
                    }
                }
            }
        }
        __syncthreads();   // A: every update of this item is in H

        // ---- epilogue.  Lane l reads only its own columns: conflict-free, no cross-lane
        // reduction.  Bin b = rows b*M .. b*M + M-1.
        const double inv_scale = cm.inv_scale, center = cm.center;
        if (a.out_norm) {
            // sweep 1: number of non-empty bins and sum of bin means (of the centred flux)
            const int r = warp / LP_PARTS, part = warp % LP_PARTS;
            const int nbp = nb / LP_PARTS;
            if (warp < LP_R * LP_PARTS) {
                double s1 = 0.0;
                int kk = 0;
                for (int b = part * nbp; b < (part + 1) * nbp; ++b) {
                    int S = 0;
                    unsigned c = 0;
                    for (int j = 0; j < M; ++j) {
                        S += (int)H[hidx(r, b * M + j, 0, lane)];
                        c += H[hidx(r, b * M + j, 1, lane)];
                    }
                    if (c > 0) {
                        s1 += __ddiv_rn(__dmul_rn((double)S, inv_scale), (double)c);
                        kk += 1;
                    }
                }
                part_s[part * LP_GROUP + r * 32 + lane] = s1;
                part_k[part * LP_GROUP + r * 32 + lane] = kk;
            }
            __syncthreads();
            if (warp < LP_R) {
                double s1 = 0.0;
                int kk = 0;
                for (int p = 0; p < LP_PARTS; ++p) {
                    s1 += part_s[p * LP_GROUP + warp * 32 + lane];
                    kk += part_k[p * LP_GROUP + warp * 32 + lane];
                }
                st_mu[warp * 32 + lane] = (kk > 0) ? __ddiv_rn(s1, (double)kk) : 0.0;
                st_kk[warp * 32 + lane] = kk;
            }
            __syncthreads();
            // sweep 2: sum of squared deviations
            if (warp < LP_R * LP_PARTS) {
                const double mu = st_mu[r * 32 + lane];
                double s2 = 0.0;
                for (int b = part * nbp; b < (part + 1) * nbp; ++b) {
                    int S = 0;
                    unsigned c = 0;
                    for (int j = 0; j < M; ++j) {
                        S += (int)H[hidx(r, b * M + j, 0, lane)];
                        c += H[hidx(r, b * M + j, 1, lane)];
                    }
                    if (c > 0) {
                        double d = __dsub_rn(__ddiv_rn(__dmul_rn((double)S, inv_scale), (double)c), mu);
                        s2 += __dmul_rn(d, d);
                    }
                }
                part_s[part * LP_GROUP + r * 32 + lane] = s2;
            }
            __syncthreads();
            if (warp < LP_R) {
                double s2 = 0.0;
                for (int p = 0; p < LP_PARTS; ++p) s2 += part_s[p * LP_GROUP + warp * 32 + lane];
                const int kk = st_kk[warp * 32 + lane];
                const double sd = (kk > 0) ? sqrt(__ddiv_rn(s2, (double)kk)) : 0.0;
                const bool flat = (kk < 2) || !(sd > 0.0);
                st_isd[warp * 32 + lane] = flat ? 0.0 : __ddiv_rn(1.0, sd);
            }
            __syncthreads();
        }
        // sweep 3: convert, write 8 bins (one 32-byte sector per array) at a time, clear rows
        {
            const int octs = nb >> 3;
            for (int unit = warp; unit < LP_R * octs; unit += LP_WARPS) {
                const int r = unit / octs, oct = unit - r * octs;
                const long long j = p0 + r * 32 + lane;
                const bool live = j < a.nperiods;
                bool ok = false;
                if (live) {
                    const double x = a.rp[j];
                    ok = (x == x);
                }
                const double mu = a.out_norm ? st_mu[r * 32 + lane] : 0.0;
                const double isd = a.out_norm ? st_isd[r * 32 + lane] : 0.0;
                const int kk = a.out_norm ? st_kk[r * 32 + lane] : 0;
                float fs[8], fn[8];
                unsigned fc[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int b = oct * 8 + e;
                    int S = 0;
                    unsigned c = 0;
                    for (int jj = 0; jj < M; ++jj) {
                        const int i0 = hidx(r, b * M + jj, 0, lane);
                        S += (int)H[i0];
                        c += H[i0 + 32];
                        H[i0] = 0u;
                        H[i0 + 32] = 0u;
                    }
                    if (!ok) {
                        S = 0;
                        c = 0;
                    }
                    const double sq = __dmul_rn((double)S, inv_scale);
                    fs[e] = (float)__dadd_rn(sq, __dmul_rn((double)c, center));
                    fc[e] = c;
                    double o = 0.0;
                    if (ok && kk > 0) {
                        o = __dadd_rn(mu, center);
                        if (c > 0 && isd > 0.0)
                            o = __dadd_rn(o, __dmul_rn(__dsub_rn(__ddiv_rn(sq, (double)c), mu), isd));
                    }
                    fn[e] = (float)o;
                }
                if (live) {
                    const long long off = ((curve * a.nperiods + j) * nb) + oct * 8;
                    if (a.out_sum) {
                        float4 *o4 = reinterpret_cast<float4 *>(a.out_sum + off);
                        o4[0] = make_float4(fs[0], fs[1], fs[2], fs[3]);
                        o4[1] = make_float4(fs[4], fs[5], fs[6], fs[7]);
                    }
                    if (a.out_count) {
                        uint4 *o4 = reinterpret_cast<uint4 *>(a.out_count + off);
                        o4[0] = make_uint4(fc[0], fc[1], fc[2], fc[3]);
                        o4[1] = make_uint4(fc[4], fc[5], fc[6], fc[7]);
                    }
                    if (a.out_norm) {
                        float4 *o4 = reinterpret_cast<float4 *>(a.out_norm + off);
                        o4[0] = make_float4(fn[0], fn[1], fn[2], fn[3]);
                        o4[1] = make_float4(fn[4], fn[5], fn[6], fn[7]);
                    }
                }
            }
        }
        if (tid == 0) *ctr = 0;
        __syncthreads();   // B: H is zero again, tile counter reset
    }
}

}  // namespace

bool fold_lp_handles(int nbins)
{
    return nbins == 32 || nbins == 64 || nbins == 128 || nbins == 256;
}

cudaError_t launch_fold_lp(const FoldArgs &a, cudaStream_t st)
{
    static int state = 0;   // 0 = not initialised, 1 = ready, -1 = shared-memory base differs
    if (state == 0) {
        cudaError_t e = cudaFuncSetAttribute(fold_lp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             LP_SMEM_BYTES);
        if (e != cudaSuccess) return e;
        unsigned *d = nullptr, h = 0;
        e = cudaMalloc(reinterpret_cast<void **>(&d), sizeof(unsigned));
        if (e != cudaSuccess) return e;
        fold_lp_kernel<<<1, LP_THREADS, LP_SMEM_BYTES, st>>>(a, 0, 0, d);
        e = cudaMemcpyAsync(&h, d, sizeof(unsigned), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        cudaFree(d);
        if (e != cudaSuccess) return e;
        state = (h == LP_SMEM_BASE) ? 1 : -1;
    }
    if (state < 0) return cudaErrorInvalidConfiguration;   // never seen; reported, not worked around
    const long long ngroups = (a.nperiods + LP_GROUP - 1) / LP_GROUP;
    const long long nitems = ngroups * a.ncurves;
    const long long grid = nitems < num_sms() ? nitems : num_sms();
    fold_lp_kernel<<<(unsigned)grid, LP_THREADS, LP_SMEM_BYTES, st>>>(a, ngroups, nitems, nullptr);
    return cudaGetLastError();
}

}  // namespace gpfc
