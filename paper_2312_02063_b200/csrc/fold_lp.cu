// fold_lp_kernel: the "lane = period" fold for every nbins <= 256 (powers of two from 32 at 256
// rows, fold_lp_kernel<false>; anything else one row per bin, fold_lp_kernel<true>)
// (PAPER.md:111 steps 1-3 and 5, noise normalisation :63 fused into the epilogue).
// DESIGN.md 6.1 has the full derivation; in short:
//
// * One persistent CTA per SM.  A work item is (curve, group of 32*R consecutive trial
//   periods).  Lane l of EVERY warp owns the R periods p0 + r*32 + l; the warps split
//   the curve's samples (anchor tiles of GPFC_TILE samples, handed out dynamically).
// * The histograms of the group live in shared memory as [r][row 0..255][sum|count][lane]
//   32-bit words: a warp-wide update touches 32 different banks whatever the bins are
//   (bank = lane), so every ATOMS is one conflict-free wavefront; the atomics only
//   arbitrate between warps.  No replication, hence no column reduction afterwards, and
//   32*R periods share every sample load.  No global atomics anywhere.
// * Samples are 8-byte records {iv, q} (iv = the sample's offset from its tile anchor in
//   32-bit fixed point), staged per warp in shared memory with coalesced 16-byte loads and
//   read back with one broadcast LDS.128 per TWO samples; one I2F.F64 per sample.
// * Phase math per point-period is ONE fp64 instruction: m = RD(v * rp + C) (DFMA.RM),
//   v = iv 2^-S ~ u - a, rp = 256 * RN(1/P),
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
// * The fold loop is unrolled 8x (32 samples per iteration); per sample the three ATOMS.ADD
//   come before the three ATOMS.POPC.INC (fewer replays in the atomic unit).
// * Epilogue: lane l walks ITS periods' rows (conflict-free), so mean / std need no
//   cross-lane reduction; every lane writes 32-byte sectors (8 bins) of its own rows.  Bin
//   means through a shared-memory table of correctly rounded reciprocals; deviations from the
//   curve mean kept as fp32 in units of the fixed-point quantum; second sweep in fp32.
#include "common.cuh"

namespace gpfc {

namespace {

constexpr int LP_R = 3;                       // periods per lane
constexpr int LP_ROWLOG = 8, LP_ROWS = 256;
constexpr int LP_THREADS = 768, LP_WARPS = LP_THREADS / 32;
constexpr int LP_GROUP = 32 * LP_R;           // periods per work item
constexpr int LP_WPR = LP_WARPS / LP_R;       // epilogue: warps per period slot
constexpr int LP_GRAN = 64;                   // samples per staging granule
#ifndef LP_UNROLL
#define LP_UNROLL 8
#endif
constexpr int LP_UNROLL_C = LP_UNROLL;        // iterations (4 samples each) unrolled in the fold loop

constexpr int LP_HIST_BYTES = 196608;         // [r][row][sum|count][lane] 32-bit words
// scratch after the histograms: sample staging during the fold, statistics partials in the
// epilogue (the two never live at the same time)
constexpr int LP_STAGE_OFF = LP_HIST_BYTES;                   // int2 [warps][LP_GRAN]
constexpr int LP_PS1_OFF = LP_HIST_BYTES;                     // double [LP_WPR][GROUP]
constexpr int LP_PS2_OFF = LP_PS1_OFF + LP_WPR * LP_GROUP * 8;
constexpr int LP_PKK_OFF = LP_PS2_OFF + LP_WPR * LP_GROUP * 8;   // int [LP_WPR][GROUP]
constexpr int LP_MU_OFF = LP_PKK_OFF + LP_WPR * LP_GROUP * 4;    // double [GROUP]
constexpr int LP_ISD_OFF = LP_MU_OFF + LP_GROUP * 8;             // double [GROUP]
constexpr int LP_KK_OFF = LP_ISD_OFF + LP_GROUP * 8;             // int [GROUP]
constexpr int LP_CTR_OFF = LP_KK_OFF + LP_GROUP * 4;
constexpr int LP_RT_N = 1024;                 // epilogue: RN(1 / c) for the counts c < LP_RT_N
constexpr int LP_RT_OFF = LP_CTR_OFF + 16;    // double [LP_RT_N], written once per CTA
constexpr int LP_SMEM_BYTES = LP_RT_OFF + LP_RT_N * 8;
static_assert(LP_SMEM_BYTES <= 227 * 1024, "shared memory budget");
static_assert(GPFC_TILE == 2 * LP_GRAN, "half-tile work units are one staging granule");
static_assert(LP_WARPS * LP_GRAN * 8 <= LP_MU_OFF - LP_STAGE_OFF, "staging fits in the scratch");
static_assert(LP_WARPS % LP_R == 0, "warps per period slot");

template <int N>
struct LpInt {
    static constexpr int value = N;
};
template <bool B>
struct LpBool {
    static constexpr bool value = B;
};

// shared-memory reductions with an immediate offset: ATOMS.ADD / ATOMS.POPC.INC [R + UR + imm].
// `addr` carries the shared-window address of the histogram (__cvta_generic_to_shared), which
// ptxas keeps in a uniform register: the window base is never assumed.
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

// word index of (r, row, array, lane) in the histogram [r][row][sum|count][lane]
__device__ __forceinline__ int hidx(int r, int row, int arr, int lane)
{
    return r * (64 * LP_ROWS) + row * 64 + arr * 32 + lane;
}

// generic (slow-path) update of one sample: move = +1 adds it to `row`, -1 removes it
__device__ __forceinline__ void hist_update(unsigned *H, int r, int row, int lane, int q, int move)
{
    atomicAdd(&H[hidx(r, row, 0, lane)], (unsigned)(move * q));
    atomicAdd(&H[hidx(r, row, 1, lane)], (unsigned)move);
}

// sq / c for a count c in [1, 2^32): reciprocal from an fp32 seed + two Newton steps
// (relative error < 2^-49), then one residual correction.  The result is exact whenever the
// quotient is representable (what the flat-profile test needs) and within 1 ulp otherwise.
__device__ __forceinline__ double div_by_count(double sq, unsigned c)
{
    const double cd = (double)c;
    double r = (double)__frcp_rn((float)c);
    r = __fma_rn(__fma_rn(-cd, r, 1.0), r, r);
    r = __fma_rn(__fma_rn(-cd, r, 1.0), r, r);
    const double q0 = __dmul_rn(sq, r);
    return __fma_rn(__fma_rn(-q0, cd, sq), r, q0);
}

// the same for a count beyond the epilogue's reciprocal table: rare, kept out of line
__device__ __noinline__ double div_by_count_slow(double sq, unsigned c)
{
    return div_by_count(sq, c);
}

// Shared-window address of dynamic shared memory on sm_100a (the first KB of the window is the
// driver's): with this value the histogram offsets are instruction immediates.  The kernel
// compares it with the real address and takes the register-base code path if they differ
// (one more integer add per point-period, same results), so nothing depends on it.
constexpr unsigned LP_WINDOW_BASE = 0x400;

// row address of one point-period: (row << 8) | (lane << 2) (+ the window base unless it is an
// immediate); keeps the smallest fraction seen in gmin
template <bool IMM, bool GEN>
__device__ __forceinline__ unsigned pp_addr(double v, double rp, double C, unsigned lane4,
                                            unsigned sbase, unsigned &gmin, unsigned nbu)
{
    double m = __fma_rd(v, rp, C);
    unsigned lo = (unsigned)__double2loint(m), hi = (unsigned)__double2hiint(m);
    if constexpr (GEN) {
        // any nbins <= 256: m counts cycles, lo = frac(u / P) 2^32; bin = floor(phi nbins) is
        // the high word of lo * nbins, the low word is the position inside the bin
        const unsigned long long pr = (unsigned long long)lo * nbu;
        lo = (unsigned)pr;
        hi = (unsigned)(pr >> 32);
    }
    gmin = min(gmin, lo);
    unsigned addr = __byte_perm(lane4, hi, 0x3240);      // (row << 8) | (lane << 2)
    if (!IMM) addr += sbase;
    return addr;
}

// one sample at the lane's periods: the sums first, then the counts (measured: the pair of
// atomics of one row back to back is ~1 % slower).  NR = period slots of the work item that hold
// periods: LP_R for the items of fold_lp_kernel, 1 for those of fold_lp_tail_kernel.
template <int NR, bool IMM, bool GEN>
__device__ __forceinline__ void sample_update(double v, int q, const double (&rp)[LP_R],
                                              const double (&C)[LP_R], unsigned lane4,
                                              unsigned sbase, unsigned (&gmin)[LP_R], unsigned nbu)
{
    static_assert(LP_R == 3 && (NR == 1 || NR == 3), "written out for one or three period slots");
    constexpr int B = IMM ? (int)LP_WINDOW_BASE : 0;
    const unsigned a0 = pp_addr<IMM, GEN>(v, rp[0], C[0], lane4, sbase, gmin[0], nbu);
    if constexpr (NR == 3) {
        const unsigned a1 = pp_addr<IMM, GEN>(v, rp[1], C[1], lane4, sbase, gmin[1], nbu);
        const unsigned a2 = pp_addr<IMM, GEN>(v, rp[2], C[2], lane4, sbase, gmin[2], nbu);
        red_add<B>(a0, q);
        red_add<B + 65536>(a1, q);
        red_add<B + 131072>(a2, q);
        red_inc<B + 128>(a0);
        red_inc<B + 65536 + 128>(a1);
        red_inc<B + 131072 + 128>(a2);
    } else {
        red_add<B>(a0, q);
        red_inc<B + 128>(a0);
    }
}

// NR = LP_R: work items 0 .. nitems - 1 are (curve, group of LP_GROUP periods).
// NR = 1 (fold_lp_tail_kernel): the groups from `first` on, cut into single period slots of 32
// periods, nitems = LP_R x groups; only slot 0 of the histogram, 8 of the 24 warps in the epilogue.
template <bool IMM, bool GEN, int NR>
__device__ __forceinline__ void fold_lp_body(const FoldArgs &a, long long ngroups, long long first,
                                             long long nitems, unsigned char *smem, unsigned sbase)
{
    unsigned *H = reinterpret_cast<unsigned *>(smem);
    double *ps1 = reinterpret_cast<double *>(smem + LP_PS1_OFF);
    double *ps2 = reinterpret_cast<double *>(smem + LP_PS2_OFF);
    int *pkk = reinterpret_cast<int *>(smem + LP_PKK_OFF);
    double *st_mu = reinterpret_cast<double *>(smem + LP_MU_OFF);
    double *st_isd = reinterpret_cast<double *>(smem + LP_ISD_OFF);
    int *st_kk = reinterpret_cast<int *>(smem + LP_KK_OFF);
    int *ctr = reinterpret_cast<int *>(smem + LP_CTR_OFF);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned lane4 = (unsigned)lane << 2;
    int4 *stage = reinterpret_cast<int4 *>(smem + LP_STAGE_OFF) + warp * (LP_GRAN / 2);
    for (int i = tid; i < LP_HIST_BYTES / 4; i += LP_THREADS) H[i] = 0u;
    if (tid == 0) *ctr = 0;
    double *rt = reinterpret_cast<double *>(smem + LP_RT_OFF);
    for (int i = tid; i < LP_RT_N; i += LP_THREADS) rt[i] = __ddiv_rn(1.0, (double)i);   // [0]: inf, never used
    __syncthreads();

    // !GEN: nb a power of two, 32 <= nb <= LP_ROWS, folded at LP_ROWS rows (rp = LP_ROWS / P).
    // GEN: any 1 <= nb <= LP_ROWS, one row per bin, the DFMA counts cycles (rp = 1 / P).
    const int nb = a.nbins;
    const unsigned nbu = (unsigned)nb;
    const int mshift = GEN ? 0 : LP_ROWLOG - (31 - __clz(nb));   // rows merged per bin = 1 << mshift
    const int M = 1 << mshift;
    const int xrows = GEN ? nb : LP_ROWS;        // bins of the exact formula at the kernel's resolution
    // 1.5 * 2^52 * (rows per cycle): ulp = LP_ROWS (or 1), so that w - M2 = rows floor(a rp / rows)
    const double M2 = GEN ? 6755399441055744.0 : 1729382256910270464.0;
    const bool want_norm = a.out_norm != nullptr;
    const bool vec = a.vec_ok != 0;

    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        long long curve, p0, pend;                                   // pend: end of the item's periods
        if constexpr (NR == LP_R) {
            curve = item / ngroups;
            p0 = (item - curve * ngroups) * LP_GROUP;
            pend = a.nperiods;
        } else {
            const long long grp = first + item / LP_R;
            curve = grp / ngroups;
            p0 = (grp - curve * ngroups) * LP_GROUP + 32 * (item % LP_R);
            pend = p0 + 32 * NR;
            if (pend > a.nperiods) pend = a.nperiods;
            if (pend <= p0) continue;                                // a slot past the last period
        }
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
            double x = (j < pend) ? a.rp[j] : CUDART_NAN;
            valid[r] = (x == x);
            rp[r] = valid[r] ? x : (double)LP_ROWS;   // dummy period: its columns are never written out
            if (valid[r]) rpmax = fmax(rpmax, x);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) rpmax = fmax(rpmax, __shfl_xor_sync(0xffffffffu, rpmax, o));

        // guard band, in units of 2^-32 row.  Per item:
        //   ebase = 4 * 2^-53 * max|u| * rpmax * 2^32 + 1     (roundings of u/P, 1/P, v, C)
        // per tile, the quantisation of v adds  eq = 2^-(S+1) * rpmax * 2^32;
        //   delta >= E + 1 unit, D = 2 delta  ->  D >= 2 (ebase + eq) + 2
        const double U = fmax(fabs(cm.umin), fabs(cm.umax));
        const double ebase = 4.0 * U * rpmax * (1.0 / 2097152.0) + 1.0;
        // worst tile of the curve: 2^-S <= 2 span_max 2^-32 (or 2^-40)
        const double eq_max = fmax(2.0 * cm.span_max, 1.0 / 256.0) * rpmax;
        const bool fast = (2.0 * (ebase + eq_max) + 2.0 <= 1048576.0) &&
                          (cm.span_max * rpmax + 2.0 * LP_ROWS < 1048576.0);

        if (fast) {
            // work units: whole anchor tiles first, then the last 2 * LP_WARPS tiles in halves
            // (one staging granule each), so that the warps reach the barrier closer together
            const int nfull = max(0, ntiles - 2 * LP_WARPS);
            const int nunits = nfull + 2 * (ntiles - nfull);
            for (;;) {
                int u = 0;
                if (lane == 0) u = atomicAdd(ctr, 1);
                u = __shfl_sync(0xffffffffu, u, 0);
                if (u >= nunits) break;
                const int t = (u < nfull) ? u : nfull + ((u - nfull) >> 1);
                const int half = (u < nfull) ? 0 : ((u - nfull) & 1);
                const int base = t * GPFC_TILE + half * LP_GRAN;
                const int cnt = min((u < nfull) ? GPFC_TILE : LP_GRAN, n - base);
                if (cnt <= 0) continue;
                const TileInfo ti = a.tiles[cm.tile0 + t];
                // D = smallest even integer >= need (>= 16); the quantisation of v is a rounding
                // to nearest: |iv 2^-S - v| <= 2^-(S+1)
                const double need = 2.0 * (ebase + 0.5 * ti.inv_scale * rpmax * 4294967296.0) + 2.0;
                unsigned D = ((unsigned)need + 2u) & ~1u;
                if (D < 16u) D = 16u;
                const double K = 1048576.0 + (double)(D >> 1) * (1.0 / 4294967296.0);
                double C[LP_R], rps[LP_R];
#pragma unroll
                for (int r = 0; r < LP_R; ++r) {
                    double w = __fma_rd(ti.a, rp[r], M2);       // M2 + ROWS * floor(a rp / ROWS)
                    double z = __dsub_rn(w, M2);
                    double c1 = __fma_rn(ti.a, rp[r], -z);      // (a rp) mod ROWS, error <= 2^-44
                    C[r] = __dadd_rn(c1, K);
                    rps[r] = __dmul_rn(rp[r], ti.inv_scale);    // exact (power of two)
                }
                const int2 *src = a.rec + cm.rec0 + base;      // 16-byte aligned
                const int4 *src4 = reinterpret_cast<const int4 *>(src);
                unsigned gmin[LP_R];
#pragma unroll
                for (int r = 0; r < LP_R; ++r) gmin[r] = 0xffffffffu;
                int4 nx = make_int4(0, 0, 0, 0);
                if (2 * lane < cnt) nx = __ldg(src4 + lane);
                for (int g0 = 0; g0 < cnt; g0 += LP_GRAN) {
                    const int gc = min(LP_GRAN, cnt - g0);
                    __syncwarp();
                    stage[lane] = nx;
                    __syncwarp();
                    if (g0 + LP_GRAN + 2 * lane < cnt) nx = __ldg(src4 + (g0 + LP_GRAN) / 2 + lane);
                    if (gc == LP_GRAN) {
#pragma unroll(LP_UNROLL_C)
                        for (int s = 0; s < LP_GRAN / 2; s += 2) {
                            const int4 ra = stage[s], rb = stage[s + 1];
                            sample_update<NR, IMM, GEN>((double)(unsigned)ra.x, ra.y, rps, C, lane4, sbase, gmin, nbu);
                            sample_update<NR, IMM, GEN>((double)(unsigned)ra.z, ra.w, rps, C, lane4, sbase, gmin, nbu);
                            sample_update<NR, IMM, GEN>((double)(unsigned)rb.x, rb.y, rps, C, lane4, sbase, gmin, nbu);
                            sample_update<NR, IMM, GEN>((double)(unsigned)rb.z, rb.w, rps, C, lane4, sbase, gmin, nbu);
                        }
                    } else {
                        const int2 *st2 = reinterpret_cast<const int2 *>(stage);
#pragma unroll 1
                        for (int s = 0; s < gc; ++s) {
                            const int2 rc = st2[s];
                            sample_update<NR, IMM, GEN>((double)(unsigned)rc.x, rc.y, rps, C, lane4, sbase, gmin, nbu);
                        }
                    }
                }
                unsigned gall = gmin[0];
#pragma unroll
                for (int r = 1; r < LP_R; ++r) gall = min(gall, gmin[r]);
                // GEN: the guard band is D units of 2^-32 cycle = D nb units of 2^-32 bin (< 2^28)
                const unsigned Dn = GEN ? D * nbu : D;
                if (__any_sync(0xffffffffu, gall < Dn)) {
                    // rare: some row coordinate sat within the guard band of an integer.
                    // Re-check those samples against the exact formula; move the ones that
                    // the fast path put in the wrong row.
                    const double *us = a.u + cm.start + base;
#pragma unroll
                    for (int r = 0; r < LP_R; ++r) {
                        if (gmin[r] >= Dn || !valid[r]) continue;
                        const double per = a.periods[p0 + r * 32 + lane];
                        if (a.stats) atomicAdd(a.stats + 1, 1ull);
#pragma unroll 4
                        for (int s = 0; s < cnt; ++s) {
                            const int2 rc = __ldg(src + s);
                            double m = __fma_rd((double)(unsigned)rc.x, rps[r], C[r]);
                            unsigned flo = (unsigned)__double2loint(m);
                            int kf = __double2hiint(m) & (LP_ROWS - 1);
                            if constexpr (GEN) {
                                const unsigned long long pr = (unsigned long long)flo * nbu;
                                flo = (unsigned)pr;
                                kf = (int)(pr >> 32);
                            }
                            if (flo < Dn) {
                                int ke = exact_bin(us[s], per, xrows);
                                if (ke != kf) {
                                    hist_update(H, r, kf, lane, rc.y, -1);
                                    if (ke >= 0) hist_update(H, r, ke, lane, rc.y, +1);
                                }
                            }
                        }
                    }
                }
            }
        } else {
            // exact path: a period far outside the fast range or a tile spanning a huge gap
            if (tid == 0 && a.stats) atomicAdd(a.stats + 0, 1ull);
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
                            int ke = exact_bin(ui, per[r], xrows);
                            if (ke >= 0) hist_update(H, r, ke, lane, qi, +1);
                        }
                    }
                }
            }
        }
        // the samples at u == 0 (CurveMeta::n_zero) are not in the sample arrays: bin 0 of every
        // period (atomics: other warps may still be folding)
        if (warp < NR && cm.n_zero > 0) {
            atomicAdd(&H[hidx(warp, 0, 0, lane)], (unsigned)cm.q_zero);
            atomicAdd(&H[hidx(warp, 0, 1, lane)], (unsigned)cm.n_zero);
        }
        __syncthreads();   // A: every update of this item is in H

        // ---- epilogue.  Lane l reads only its own columns: conflict-free, no cross-lane
        // reduction.  Bin b = rows b*M .. b*M + M-1; warp group g = warp / LP_WPR takes period
        // slot r = g, its LP_WPR warps split the octets of bins (one 32-byte sector per output
        // array and lane).
        const double inv_scale = cm.inv_scale, center = cm.center, pivot = cm.pivot;
        const double pivot_q = __dmul_rn(pivot, __ddiv_rn(1.0, inv_scale));   // in units of 2^-s: exact
        const double center_s = a.center_out ? 0.0 : center;       // FoldArgs::center_out: centred sums
        if (a.center_out && p0 == 0 && tid == 0) a.center_out[curve] = center;
        // GEN: the last octet may be partial; a period slot the item does not use was never
        // touched: nothing to write, nothing to clear
        const int octs = (warp / LP_WPR < NR) ? ((nb + 7) >> 3) : 0;
        const bool vec8 = vec && !(nb & 7);
        const int r = warp / LP_WPR, wr = warp - r * LP_WPR;
        const long long j = p0 + r * 32 + lane;
        const bool live = j < pend;
        bool ok = false;
#pragma unroll
        for (int rr = 0; rr < LP_R; ++rr)
            if (rr == r) ok = live && valid[rr];
        unsigned *Hr = H + r * (LP_ROWS * 64) + lane;
        {
            // sweep 1: sums and counts out; deviation d of the bin mean from the curve mean back
            // into the bin's first sum word as fp32 (NaN = empty), every other word cleared;
            // one-pass moments of d (exactly zero for a flat profile).
            double s1 = 0.0, s2 = 0.0;
            int kk = 0;
            // compiled per (rows per bin, sums / counts wanted or not): the common cases carry
            // no dead arithmetic and no run-time row loop
            auto sweep1 = [&](auto m_c, auto ws_c) {
            constexpr int MC = decltype(m_c)::value;           // rows per bin; 0: M, at run time
            constexpr bool WS = decltype(ws_c)::value;         // out_sum or out_count wanted
            const int MM = MC ? MC : M;
            for (int oct = wr; oct < octs; oct += LP_WPR) {
                float fs[8];
                unsigned fc[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    unsigned *h0 = Hr + (oct * 8 + e) * MM * 64;
                    int S = (int)h0[0];
                    unsigned c = h0[32];
#pragma unroll
                    for (int jj = 1; jj < MM; ++jj) {
                        S += (int)h0[jj * 64];
                        c += h0[jj * 64 + 32];
                        h0[jj * 64] = 0u;
                        h0[jj * 64 + 32] = 0u;
                    }
                    if (!ok) {
                        S = 0;
                        c = 0;
                    }
                    const double Sd = (double)S;
                    const double cd = (double)c;
                    if constexpr (WS) {
                        fs[e] = (float)__dadd_rn(__dmul_rn(Sd, inv_scale), __dmul_rn(cd, center_s));
                        fc[e] = c;
                    }
                    unsigned dw = 0u;
                    if (want_norm) {
                        // mean = S / c, in units of 2^-s (the fixed-point quantum: whatever the
                        // flux scale, the deviations are then of order 1 .. 2^31 and fit fp32),
                        // through the table of correctly rounded reciprocals: q0 = S r, one
                        // residual correction (exact whenever the quotient is representable,
                        // like div_by_count)
                        double m;
                        if (c < (unsigned)LP_RT_N) {
                            const double rc = rt[c];           // c == 0: inf, discarded below
                            const double q0 = __dmul_rn(Sd, rc);
                            m = __fma_rn(__fma_rn(-q0, cd, Sd), rc, q0);
                        } else {
                            m = div_by_count_slow(Sd, c);
                        }
                        const bool nz = c > 0u;
                        const double d = nz ? __dsub_rn(m, pivot_q) : 0.0;
                        s1 += d;
                        s2 += __dmul_rn(d, d);
                        kk += nz ? 1 : 0;
                        dw = nz ? __float_as_uint((float)d) : 0x7fc00000u;    // NaN: empty bin
                    }
                    h0[0] = dw;
                    h0[32] = 0u;
                }
                if constexpr (WS) {
                if (live) {
                    const long long off = ((curve * a.nperiods + j) * nb) + oct * 8;
                    if (vec8) {
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
                    } else {
                        // outputs that are only 4-byte aligned: scalar stores
#pragma unroll
                        for (int e = 0; e < 8; ++e) {
                            if (GEN && oct * 8 + e >= nb) break;
                            if (a.out_sum) a.out_sum[off + e] = fs[e];
                            if (a.out_count) a.out_count[off + e] = fc[e];
                        }
                    }
                }
                }
            }
            };
            const bool ws = a.out_sum != nullptr || a.out_count != nullptr;
            if (M == 1) {
                if (ws)
                    sweep1(LpInt<1>{}, LpBool<true>{});
                else
                    sweep1(LpInt<1>{}, LpBool<false>{});
            } else if (M == 2) {
                if (ws)
                    sweep1(LpInt<2>{}, LpBool<true>{});
                else
                    sweep1(LpInt<2>{}, LpBool<false>{});
            } else {
                sweep1(LpInt<0>{}, LpBool<true>{});
            }
            if (want_norm) {
                ps1[wr * LP_GROUP + r * 32 + lane] = s1;
                ps2[wr * LP_GROUP + r * 32 + lane] = s2;
                pkk[wr * LP_GROUP + r * 32 + lane] = kk;
            }
        }
        if (want_norm) {
            __syncthreads();
            if (warp < NR) {
                double s1 = 0.0, s2 = 0.0;
                int kk = 0;
                for (int w = 0; w < LP_WPR; ++w) {          // fixed order: deterministic
                    s1 += ps1[w * LP_GROUP + warp * 32 + lane];
                    s2 += ps2[w * LP_GROUP + warp * 32 + lane];
                    kk += pkk[w * LP_GROUP + warp * 32 + lane];
                }
                // mean and population std of the deviations, in units of 2^-s
                double dm = 0.0, isd = 0.0;
                if (kk > 0) {
                    dm = __ddiv_rn(s1, (double)kk);
                    const double var = __dsub_rn(__ddiv_rn(s2, (double)kk), __dmul_rn(dm, dm));
                    const double sd = (var > 0.0) ? sqrt(var) : 0.0;
                    if (kk >= 2 && sd > 0.0) isd = __ddiv_rn(1.0, sd);
                }
                st_mu[warp * 32 + lane] = dm;
                st_isd[warp * 32 + lane] = isd;
                st_kk[warp * 32 + lane] = kk;
            }
            __syncthreads();
            // sweep 2: out = base + (d - dm) / s from the fp32 deviations, in fp32 (d, dm and s in
            // units of 2^-s; (d - dm) / s is a z-score of a few units, base = mu + center: each
            // rounding is 6e-8 relative against the 1e-4 bar of the normalised profile); rows
            // cleared (same split as sweep 1)
            const double dm = st_mu[r * 32 + lane], isd = st_isd[r * 32 + lane];
            const double mu = __dadd_rn(pivot, __dmul_rn(dm, inv_scale));      // profile mean, flux units
            const float dmf = (float)dm, isdf = ok ? (float)isd : 0.f;
            const float basef = (ok && st_kk[r * 32 + lane] > 0) ? (float)__dadd_rn(mu, center) : 0.f;
            auto sweep2 = [&](auto m_c) {
            constexpr int MC = decltype(m_c)::value;           // rows per bin; 0: M, at run time
            const int MM = MC ? MC : M;
            for (int oct = wr; oct < octs; oct += LP_WPR) {
                float fn[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    unsigned *h0 = Hr + (oct * 8 + e) * MM * 64;
                    const float df = __uint_as_float(h0[0]);
                    h0[0] = 0u;
                    // NaN (empty bin) or s == 0: the profile mean
                    const float z = __fmaf_rn(__fsub_rn(df, dmf), isdf, basef);
                    fn[e] = (df == df && isdf > 0.f) ? z : basef;
                }
                if (live) {
                    float *on = a.out_norm + ((curve * a.nperiods + j) * nb) + oct * 8;
                    if (vec8) {
                        float4 *o4 = reinterpret_cast<float4 *>(on);
                        o4[0] = make_float4(fn[0], fn[1], fn[2], fn[3]);
                        o4[1] = make_float4(fn[4], fn[5], fn[6], fn[7]);
                    } else {
#pragma unroll
                        for (int e = 0; e < 8; ++e)
                            if (!GEN || oct * 8 + e < nb) on[e] = fn[e];
                    }
                }
            }
            };
            if (M == 1)
                sweep2(LpInt<1>{});
            else if (M == 2)
                sweep2(LpInt<2>{});
            else
                sweep2(LpInt<0>{});
        }
        if (tid == 0) *ctr = 0;
        __syncthreads();   // B: H is zero again, tile counter reset
    }
}

template <bool GEN>
__global__ void __launch_bounds__(LP_THREADS, 1)
fold_lp_kernel(FoldArgs a, long long ngroups, long long nitems)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    const unsigned sbase = (unsigned)__cvta_generic_to_shared(smem);
    if (sbase == LP_WINDOW_BASE)
        fold_lp_body<true, GEN, LP_R>(a, ngroups, 0, nitems, smem, sbase);
    else
        fold_lp_body<false, GEN, LP_R>(a, ngroups, 0, nitems, smem, sbase);
}

// the groups of a launch's last, partly filled wave, as single-slot items (launch_fold_lp)
template <bool GEN>
__global__ void __launch_bounds__(LP_THREADS, 1)
fold_lp_tail_kernel(FoldArgs a, long long ngroups, long long first, long long nitems)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    const unsigned sbase = (unsigned)__cvta_generic_to_shared(smem);
    if (sbase == LP_WINDOW_BASE)
        fold_lp_body<true, GEN, 1>(a, ngroups, first, nitems, smem, sbase);
    else
        fold_lp_body<false, GEN, 1>(a, ngroups, first, nitems, smem, sbase);
}

}  // namespace

bool fold_lp_handles(int nbins) { return nbins >= 1 && nbins <= LP_ROWS; }

// powers of two from 32 fold at 256 rows (masks instead of a multiply); anything else up to
// 256 bins takes the one-row-per-bin variant
bool fold_lp_pow2(int nbins) { return nbins == 32 || nbins == 64 || nbins == 128 || nbins == 256; }

cudaError_t fold_lp_init_device()
{
    cudaError_t e = cudaFuncSetAttribute(fold_lp_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         LP_SMEM_BYTES);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(fold_lp_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 LP_SMEM_BYTES);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(fold_lp_tail_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 LP_SMEM_BYTES);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(fold_lp_tail_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 LP_SMEM_BYTES);
    return e;
}

cudaError_t launch_fold_lp(const FoldArgs &a, cudaStream_t st, int sms)
{
    const long long ngroups = (a.nperiods + LP_GROUP - 1) / LP_GROUP;
    const long long n3 = ngroups * a.ncurves;
    // The CTAs take the items round robin, so the last wave of a launch holds n3 mod sms items
    // while the other SMs idle for a whole item (config 1: 12 of 148 in wave 15 of 15).  When
    // those groups, cut into single period slots, fit one wave, they go to fold_lp_tail_kernel
    // instead (a single-slot item takes ~0.4 of a full one); so does a call of fewer groups
    // than a third of the SMs.  The main kernel's code is the same with or without a tail.
    const long long rem = n3 % sms;
    const long long ntail = (rem > 0 && rem * LP_R <= sms) ? rem : 0;
    const long long nreg = n3 - ntail;
    const bool pow2 = fold_lp_pow2(a.nbins);
    if (nreg > 0) {
        const unsigned grid = (unsigned)(nreg < sms ? nreg : sms);
        if (pow2)
            fold_lp_kernel<false><<<grid, LP_THREADS, LP_SMEM_BYTES, st>>>(a, ngroups, nreg);
        else
            fold_lp_kernel<true><<<grid, LP_THREADS, LP_SMEM_BYTES, st>>>(a, ngroups, nreg);
        note_launch();
    }
    if (ntail > 0) {
        const unsigned grid = (unsigned)(ntail * LP_R);
        if (pow2)
            fold_lp_tail_kernel<false><<<grid, LP_THREADS, LP_SMEM_BYTES, st>>>(a, ngroups, nreg, ntail * LP_R);
        else
            fold_lp_tail_kernel<true><<<grid, LP_THREADS, LP_SMEM_BYTES, st>>>(a, ngroups, nreg, ntail * LP_R);
        note_launch();
    }
    return cudaGetLastError();
}

}  // namespace gpfc
