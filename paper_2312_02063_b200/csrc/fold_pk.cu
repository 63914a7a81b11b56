// fold_pk_kernel: the fold at 1024 / 2048 / 4096 rows (nbins 512 ... 4096), with the paper's
// equal-count merge optionally fused into the epilogue (PAPER.md:105, :111 steps 1-5, Fig. 4;
// noise normalisation :63).  DESIGN.md 6.2 has the derivation; in short:
//
// * One persistent CTA per SM, 24 warps.  A work item is (curve, group of PL consecutive trial
//   periods), PL = 32768 / ROWS (32, 16, 8).  The 32 lanes of EVERY warp are PL periods x SL
//   sample slots (SL = 32 / PL = 1, 2, 4): lane (slot, p) folds the samples of its slot at
//   period p0 + p.  The warps split the curve's samples in anchor tiles.
// * Histogram in shared memory: sums [row][PL] int32 (128 KB) and PACKED counts
//   [row mod ROWS/2][PL] (64 KB): the low half-word counts rows k and k + ROWS/2 together, the
//   high half-word counts row k + ROWS/2 alone.  The bank of a word is (row mod SL) * PL + p:
//   one conflict-free wavefront per warp-wide atomic when SL = 1; for SL > 1 two slots collide
//   when their rows agree mod SL (hardware replays, correctness is not affected).
//   A half-word cannot overflow while at most 65,535 samples have been added.  Longer curves
//   (the paper's Kepler curves have up to 70,000 epochs) are folded without
//   a flush first and checked (the low half-words of a period add up to n_valid iff none
//   wrapped); only if one did is the item folded again in segments of 65,408 samples with the
//   counts flushed to a 32-bit side array in global memory (one per CTA, L2-resident) between.
// * Phase math, guard band and exact re-check: as in fold_lp.cu (one DFMA.RM per point-period,
//   m = RD(v rp + C), row = bits of the high word, fraction = the low word; a tile whose
//   smallest fraction is inside the guard band is re-checked against the exact formula, by
//   the whole warp, 32 samples at a time for every flagged lane).  Fold loop unrolled 8x.
// * Epilogue, one of
//   (1) bins: sums / counts (/ normalised profile) of nbins = ROWS >> k bins, written per lane;
//   (1b) bins at ROWS = nbins = 1024 (config 3): the row vectors are permuted in place so that
//       a warp walks the bins of one period with lane = bin, and every store is a full line;
//   (2) merge: the nbins intermediary bins are merged left to right into nb2 bins of equal
//       count (boundary bins split pro rata, R18) straight from the exact integer
//       sums in shared memory -- the intermediary profile never reaches HBM -- then the mean
//       and the noise-normalised profile of the nb2 bins are written.
#include "common.cuh"

namespace gpfc {

namespace {

constexpr int PK_THREADS = 768;
constexpr int PK_WARPS = PK_THREADS / 32;
constexpr int PK_GRAN = 64;                       // samples per staging granule
constexpr int PK_CNT_OFF = 131072;                // byte offset of the packed counts
constexpr int PK_HIST_BYTES = 196608;
constexpr int PK_HIST_WORDS = PK_HIST_BYTES / 4;
constexpr int PK_CELLS = 32768;                   // ROWS * PL, every variant
constexpr int PK_SCR_OFF = PK_HIST_BYTES;         // scratch: staging | statistics partials | merge
constexpr int PK_SCR_BYTES = 35072;
constexpr int PK_CTR_OFF = PK_SCR_OFF + PK_SCR_BYTES;
constexpr int PK_SMEM_BYTES = PK_CTR_OFF + 16;
constexpr int PK_FLUSH_TILES = 511;               // 65,408 samples between count flushes
#ifndef PK_UNROLL
#define PK_UNROLL 8
#endif
constexpr int PK_UNROLL_C = PK_UNROLL;          // iterations (4 samples per lane each) unrolled in the fold loop
// scratch, fold phase: int2 stage[PK_WARPS][PK_GRAN]                       12,288 B
// scratch, bins epilogue: double ps1, ps2 [PK_WARPS][32]; int pkk [PK_WARPS][32];
//                         double mu[32], isd[32]; int kk[32]                16,000 B
constexpr int PK_PS1_OFF = PK_SCR_OFF;
constexpr int PK_PS2_OFF = PK_PS1_OFF + PK_WARPS * 32 * 8;
constexpr int PK_PKK_OFF = PK_PS2_OFF + PK_WARPS * 32 * 8;
constexpr int PK_MU_OFF = PK_PKK_OFF + PK_WARPS * 32 * 4;
constexpr int PK_ISD_OFF = PK_MU_OFF + 32 * 8;
constexpr int PK_KK_OFF = PK_ISD_OFF + 32 * 8;
// scratch, lane = bin epilogue (1024 rows): {1 / c, c} as doubles for the counts c < PK_RT_N,
// written once per CTA behind the other bins-epilogue scratch (the fold's staging and the
// statistics partials stay below it; the merge epilogue, which uses the whole scratch, never
// runs in the same launch)
constexpr int PK_RT_N = 256;
constexpr int PK_RT_OFF = PK_SCR_OFF + 16384;
static_assert(PK_KK_OFF + 32 * 4 <= PK_RT_OFF, "reciprocal table behind the bins-epilogue scratch");
static_assert(PK_RT_OFF + PK_RT_N * 16 <= PK_SCR_OFF + PK_SCR_BYTES, "reciprocal table fits");
// scratch, merge epilogue: cumulative count / integer flux in front of every mini-chunk
// (32 or 16 KB), warp totals [PK_WARPS][PL] (6 KB at most); the cumulative flux at the
// boundaries goes over the histogram: [nb2 + 1][PL] doubles, PL * nb2 <= PK_MG_MAX
constexpr int PK_MG_MAX = 2048;
static_assert((PK_MG_MAX + 32) * 8 <= PK_HIST_BYTES, "cumulative flux table fits over the histogram");
static_assert(PK_KK_OFF + 32 * 4 <= PK_SCR_OFF + PK_SCR_BYTES, "bins-epilogue scratch");
static_assert(PK_WARPS * PK_GRAN * 8 <= PK_SCR_BYTES, "staging scratch");
static_assert(PK_SMEM_BYTES <= 227 * 1024, "shared memory budget");
static_assert(GPFC_TILE == 2 * PK_GRAN, "half-tile work units are one staging granule");

template <bool B>
struct PkBool {
    static constexpr bool value = B;
};

template <int ROWLOG>
struct PkV {
    static constexpr int ROWS = 1 << ROWLOG, HALF = ROWS / 2;
    static constexpr int PLOG = 15 - ROWLOG, PL = 1 << PLOG;      // periods per work item
    static constexpr int SLOG = 5 - PLOG, SL = 1 << SLOG;         // sample slots per warp
    static constexpr int KSH = PLOG + 2;                          // log2 of the row stride in bytes
    static constexpr unsigned SMASK = 0x1ffffu & ~((1u << KSH) - 1u);
    static constexpr unsigned CMASK = 0x0ffffu & ~((1u << KSH) - 1u);
};

// shared-memory reduction with an immediate offset (ATOMS.ADD [R + UR + imm]: `addr` already
// holds the shared-window address of the histogram, which ptxas keeps in a uniform register)
template <int IMM>
__device__ __forceinline__ void pk_red_add(unsigned addr, int v)
{
    asm volatile("red.shared.add.u32 [%0+%2], %1;" ::"r"(addr), "r"(v), "n"(IMM) : "memory");
}

// a value the compiler cannot see through, so that (x & mask) | p4 stays ONE LOP3
__device__ __forceinline__ unsigned pk_opaque(unsigned x)
{
    unsigned y;
    asm volatile("mov.u32 %0, %1;" : "=r"(y) : "r"(x));
    return y;
}

// Shared-window address of dynamic shared memory on sm_100a (the first KB of the window is the
// driver's): with this value the histogram offsets are instruction immediates.  The kernel
// compares it with the real address and takes the register-base code path if they differ
// (two more integer adds per point-period, same results), so nothing depends on it.
constexpr unsigned PK_WINDOW_BASE = 0x400;

// one point-period: row from the DFMA, two shared-memory atomics
template <int ROWLOG, bool IMM>
__device__ __forceinline__ void pk_update(double v, int q, double rps, double C, unsigned p4,
                                          unsigned one, unsigned sbase, unsigned &gmin)
{
    using V = PkV<ROWLOG>;
    const double m = __fma_rd(v, rps, C);
    const unsigned lo = (unsigned)__double2loint(m), hi = (unsigned)__double2hiint(m);
    gmin = min(gmin, lo);
    const unsigned tt = hi << V::KSH;                      // row * (4 PL) (+ junk above bit 16)
    const unsigned saddr = (tt & V::SMASK) | p4;           // row * 4 PL + p * 4
    const unsigned caddr = (tt & V::CMASK) | p4;           // (row mod HALF) * 4 PL + p * 4
    const unsigned val = (tt & 0x10000u) | one;            // 1 + ((row >= HALF) << 16)
    if (IMM) {
        pk_red_add<(int)PK_WINDOW_BASE>(saddr, q);
        pk_red_add<(int)PK_WINDOW_BASE + PK_CNT_OFF>(caddr, (int)val);
    } else {
        pk_red_add<0>(saddr + sbase, q);
        pk_red_add<PK_CNT_OFF>(caddr + sbase, (int)val);
    }
}

// slow-path update of one sample: move = +1 adds it to `row`, -1 removes it
template <int ROWLOG>
__device__ __forceinline__ void pk_hist_update(unsigned *H, int row, int p, int q, int move)
{
    using V = PkV<ROWLOG>;
    atomicAdd(&H[row * V::PL + p], (unsigned)(move * q));
    atomicAdd(&H[PK_CNT_OFF / 4 + (row & (V::HALF - 1)) * V::PL + p],
              (unsigned)move * (1u + ((unsigned)(row >> (ROWLOG - 1)) << 16)));
}

// count of (row, p): packed half-words in shared memory + the flushed part, if any
template <int ROWLOG>
__device__ __forceinline__ unsigned pk_count(const unsigned *H, const unsigned *side, int row, int p)
{
    using V = PkV<ROWLOG>;
    const unsigned w = H[PK_CNT_OFF / 4 + (row & (V::HALF - 1)) * V::PL + p];
    unsigned c = (row >> (ROWLOG - 1)) ? (w >> 16) : ((w & 0xffffu) - (w >> 16));
    if (side) c += __ldcg(side + row * V::PL + p);
    return c;
}

// sq / c for a count c in [1, 2^32): reciprocal from an fp32 seed + two Newton steps, then
// one residual correction.  Exact whenever the quotient is representable, within 1 ulp
// otherwise (same routine as fold_lp.cu).
__device__ __forceinline__ double pk_div_by_count(double sq, unsigned c)
{
    const double cd = (double)c;
    double r = (double)__frcp_rn((float)c);
    r = __fma_rn(__fma_rn(-cd, r, 1.0), r, r);
    r = __fma_rn(__fma_rn(-cd, r, 1.0), r, r);
    const double q0 = __dmul_rn(sq, r);
    return __fma_rn(__fma_rn(-q0, cd, sq), r, q0);
}

template <int ROWLOG, bool IMM>
__device__ __forceinline__ void fold_pk_body(const FoldArgs &a, long long ngroups, long long nitems,
                                             unsigned char *smem, unsigned sbase)
{
    using V = PkV<ROWLOG>;
    constexpr int ROWS = V::ROWS, HALF = V::HALF, PL = V::PL, PLOG = V::PLOG, SL = V::SL;
    unsigned *H = reinterpret_cast<unsigned *>(smem);
    int *ctr = reinterpret_cast<int *>(smem + PK_CTR_OFF);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int p = lane & (PL - 1), slot = lane >> PLOG;
    const unsigned p4 = pk_opaque((unsigned)p << 2);
    const unsigned one = pk_opaque((unsigned)(a.nbins > 0));   // 1, not foldable
    int4 *stage4 = reinterpret_cast<int4 *>(smem + PK_SCR_OFF) + warp * (PK_GRAN / 2);
    for (int i = tid; i < PK_HIST_WORDS; i += PK_THREADS) H[i] = 0u;
    if (tid == 0) *ctr = 0;
    if (ROWLOG == 10 && a.nb2 == 0 && tid < PK_RT_N) {
        double2 *rt = reinterpret_cast<double2 *>(smem + PK_RT_OFF);
        rt[tid] = make_double2(__ddiv_rn(1.0, (double)tid), (double)tid);   // [0] is never read
    }
    __syncthreads();

    const int nb = a.nbins;                               // power of two, ROWS / 2 <= nb <= ROWS
    const int mshift = ROWLOG - (31 - __clz(nb));         // rows merged per bin = 1 << mshift
    const int M = 1 << mshift;
    const double M2 = 6755399441055744.0 * (double)ROWS;  // 1.5 * 2^(52 + ROWLOG): ulp = ROWS
    unsigned *side = a.side ? a.side + (size_t)blockIdx.x * PK_CELLS : nullptr;

    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        const long long curve = item / ngroups;
        const long long p0 = (item - curve * ngroups) * PL;
        const CurveMeta cm = a.meta[curve];
        const int n = cm.n_valid;
        const int ntiles = (n + GPFC_TILE - 1) / GPFC_TILE;

        // this lane's period
        const long long j = p0 + p;
        const bool live = j < a.nperiods;
        const double x = live ? a.rp[j] : CUDART_NAN;
        const bool valid = (x == x);
        const double rp = valid ? x : (double)ROWS;       // dummy: its column is never written out
        double rpmax = valid ? x : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) rpmax = fmax(rpmax, __shfl_xor_sync(0xffffffffu, rpmax, o));

        // guard band, units of 2^-32 row; see fold_lp.cu
        const double U = fmax(fabs(cm.umin), fabs(cm.umax));
        const double ebase = 4.0 * U * rpmax * (1.0 / 2097152.0) + 1.0;
        const double eq_max = fmax(2.0 * cm.span_max, 1.0 / 256.0) * rpmax;
        const bool fast = (2.0 * (ebase + eq_max) + 2.0 <= 1048576.0) &&
                          (cm.span_max * rpmax + 2.0 * ROWS < 1048576.0);
        if (!fast && tid == 0 && a.stats) atomicAdd(a.stats + 0, 1ull);
        const double per_exact = (valid && !fast) ? a.periods[j] : 1.0;

        // Count flushes.  A curve of more than PK_FLUSH_TILES tiles could overflow a packed
        // half-word, but only if more than 65,535 of its points share one pair of rows: the
        // first attempt folds it without flushes and checks afterwards (the low half-words of
        // a period add up to n_valid exactly iff none of them wrapped); if one did, the
        // histogram is cleared and the item is folded again in segments of at most
        // PK_FLUSH_TILES tiles with the counts flushed to the 32-bit side array in between.
        const unsigned *sd = nullptr;
        for (int attempt = 0;; ++attempt) {
        const int nseg = (fast && attempt == 0) ? 1 : (ntiles + PK_FLUSH_TILES - 1) / PK_FLUSH_TILES;
        const int tps = (nseg > 1) ? (ntiles + nseg - 1) / nseg : ntiles;
        for (int seg = 0; seg < nseg; ++seg) {
            const int t_lo = seg * tps;
            const int t_n = min(ntiles - t_lo, tps);
            if (fast) {
                // work units: whole anchor tiles first, the last 2 * PK_WARPS tiles in halves
                const int nfull = max(0, t_n - 2 * PK_WARPS);
                const int nunits = nfull + 2 * (t_n - nfull);
                for (;;) {
                    int u = 0;
                    if (lane == 0) u = atomicAdd(ctr, 1);
                    u = __shfl_sync(0xffffffffu, u, 0);
                    if (u >= nunits) break;
                    const int t = t_lo + ((u < nfull) ? u : nfull + ((u - nfull) >> 1));
                    const int half = (u < nfull) ? 0 : ((u - nfull) & 1);
                    const int base = t * GPFC_TILE + half * PK_GRAN;
                    const int cnt = min((u < nfull) ? GPFC_TILE : PK_GRAN, n - base);
                    if (cnt <= 0) continue;
                    const TileInfo ti = a.tiles[cm.tile0 + t];
                    const double need = 2.0 * (ebase + 0.5 * ti.inv_scale * rpmax * 4294967296.0) + 2.0;
                    unsigned D = ((unsigned)need + 2u) & ~1u;
                    if (D < 16u) D = 16u;
                    const double K = 1048576.0 + (double)(D >> 1) * (1.0 / 4294967296.0);
                    const double w = __fma_rd(ti.a, rp, M2);          // M2 + ROWS floor(a rp / ROWS)
                    const double z = __dsub_rn(w, M2);
                    const double c1 = __fma_rn(ti.a, rp, -z);         // (a rp) mod ROWS
                    const double C = __dadd_rn(c1, K);
                    const double rps = __dmul_rn(rp, ti.inv_scale);   // exact (power of two)
                    const int2 *src = a.rec + cm.rec0 + base;         // 16-byte aligned
                    const int4 *src4 = reinterpret_cast<const int4 *>(src);
                    unsigned gmin = 0xffffffffu;
                    int4 nx = make_int4(0, 0, 0, 0);
                    if (2 * lane < cnt) nx = __ldg(src4 + lane);
                    for (int g0 = 0; g0 < cnt; g0 += PK_GRAN) {
                        const int gc = min(PK_GRAN, cnt - g0);
                        __syncwarp();
                        stage4[lane] = nx;
                        __syncwarp();
                        if (g0 + PK_GRAN + 2 * lane < cnt) nx = __ldg(src4 + (g0 + PK_GRAN) / 2 + lane);
                        if (gc == PK_GRAN) {
                            // slot s takes the sample pairs s, s + SL, s + 2 SL, ...
#pragma unroll(PK_UNROLL_C)
                            for (int g = 0; g < PK_GRAN / 2; g += 2 * SL) {
                                const int4 ra = stage4[g + slot], rb = stage4[g + SL + slot];
                                pk_update<ROWLOG, IMM>((double)(unsigned)ra.x, ra.y, rps, C, p4, one, sbase, gmin);
                                pk_update<ROWLOG, IMM>((double)(unsigned)ra.z, ra.w, rps, C, p4, one, sbase, gmin);
                                pk_update<ROWLOG, IMM>((double)(unsigned)rb.x, rb.y, rps, C, p4, one, sbase, gmin);
                                pk_update<ROWLOG, IMM>((double)(unsigned)rb.z, rb.w, rps, C, p4, one, sbase, gmin);
                            }
                        } else {
                            const int2 *st2 = reinterpret_cast<const int2 *>(stage4);
#pragma unroll 1
                            for (int s = slot; s < gc; s += SL) {
                                const int2 rc = st2[s];
                                pk_update<ROWLOG, IMM>((double)(unsigned)rc.x, rc.y, rps, C, p4, one, sbase, gmin);
                            }
                        }
                    }
                    unsigned flagged = __ballot_sync(0xffffffffu, gmin < D && valid);
                    if (flagged) {
                        // rare: a row coordinate sat within the guard band of an integer.  For
                        // every flagged lane (slot, period) the WHOLE warp re-checks that lane's
                        // samples (same enumeration as above), 32 at a time, against the exact
                        // formula and moves the ones in the wrong row.
                        const double *us = a.u + cm.start + base;
                        do {
                            const int L = __ffs(flagged) - 1;
                            flagged &= flagged - 1;
                            const int pL = L & (PL - 1), slotL = L >> PLOG;
                            const double rps_l = __shfl_sync(0xffffffffu, rps, L);
                            const double C_l = __shfl_sync(0xffffffffu, C, L);
                            const double per = a.periods[p0 + pL];
                            if (a.stats && lane == 0) atomicAdd(a.stats + 1, 1ull);
                            for (int g0 = 0; g0 < cnt; g0 += PK_GRAN) {
                                const int gc = min(PK_GRAN, cnt - g0);
                                const int ns = (gc == PK_GRAN) ? PK_GRAN / SL : (gc - slotL + SL - 1) / SL;
                                for (int i = lane; i < ns; i += 32) {
                                    // i-th sample of that slot in the granule
                                    const int s = (gc == PK_GRAN) ? (((i >> 1) * SL + slotL) * 2 + (i & 1))
                                                                  : (slotL + i * SL);
                                    const int2 rc = __ldg(src + g0 + s);
                                    const double m = __fma_rd((double)(unsigned)rc.x, rps_l, C_l);
                                    if ((unsigned)__double2loint(m) < D) {
                                        const int kf = __double2hiint(m) & (ROWS - 1);
                                        const int ke = exact_bin(us[g0 + s], per, ROWS);
                                        if (ke != kf) {
                                            pk_hist_update<ROWLOG>(H, kf, pL, rc.y, -1);
                                            if (ke >= 0) pk_hist_update<ROWLOG>(H, ke, pL, rc.y, +1);
                                        }
                                    }
                                }
                            }
                        } while (flagged);
                    }
                }
            } else {
                // exact path: a period far outside the fast range or a tile spanning a huge gap
                for (;;) {
                    int t = 0;
                    if (lane == 0) t = atomicAdd(ctr, 1);
                    t = __shfl_sync(0xffffffffu, t, 0);
                    if (t >= t_n) break;
                    const int base = (t_lo + t) * GPFC_TILE;
                    const int cnt = min(GPFC_TILE, n - base);
                    const double *us = a.u + cm.start + base;
                    const int *qs = a.q + cm.start + base;
                    if (valid) {
#pragma unroll 1
                        for (int s = slot; s < cnt; s += SL) {
                            const int ke = exact_bin(us[s], per_exact, ROWS);
                            if (ke >= 0) pk_hist_update<ROWLOG>(H, ke, p, qs[s], +1);
                        }
                    }
                }
            }
            __syncthreads();   // every update of this segment is in H
            if (seg + 1 < nseg) {
                // count flush: the packed half-words go to the 32-bit side array
                for (int i = tid; i < HALF * PL; i += PK_THREADS) {
                    const unsigned w = H[PK_CNT_OFF / 4 + i];
                    const unsigned chi = w >> 16, clo = (w & 0xffffu) - chi;
                    if (seg == 0) {
                        side[i] = clo;
                        side[i + HALF * PL] = chi;
                    } else {
                        side[i] += clo;
                        side[i + HALF * PL] += chi;
                    }
                    H[PK_CNT_OFF / 4 + i] = 0u;
                }
                if (tid == 0) *ctr = 0;
                __syncthreads();
            }
        }
        // Counts that were flushed go back into the packed half-words if every row pair of
        // every period holds fewer than 65,536 points (always, unless nearly the whole curve
        // sits in one pair of rows): the epilogues then read shared memory only.
        sd = nullptr;
        if (nseg > 1) {
            int over = 0;
            for (int i = tid; i < HALF * PL; i += PK_THREADS) {
                const unsigned w = H[PK_CNT_OFF / 4 + i];
                const unsigned slo = __ldcg(side + i), shi = __ldcg(side + i + HALF * PL);
                over |= ((w & 0xffffu) + slo + shi > 0xffffu) ? 1 : 0;
            }
            over = __syncthreads_or(over);
            if (over) {
                sd = side;
            } else {
                for (int i = tid; i < HALF * PL; i += PK_THREADS) {
                    const unsigned slo = __ldcg(side + i), shi = __ldcg(side + i + HALF * PL);
                    H[PK_CNT_OFF / 4 + i] += slo + shi + (shi << 16);
                }
                __syncthreads();
            }
            break;
        }
        if (ntiles <= PK_FLUSH_TILES || !fast) break;
        {
            // optimistic attempt of a long curve: did a half-word wrap?  Thread tid only meets
            // count words of its own period p (PK_THREADS is a multiple of PL).
            unsigned *chk = reinterpret_cast<unsigned *>(smem + PK_SCR_OFF);     // [PK_WARPS][32]
            unsigned lo_sum = 0;
            for (int i = tid; i < HALF * PL; i += PK_THREADS) lo_sum += H[PK_CNT_OFF / 4 + i] & 0xffffu;
            chk[tid] = lo_sum;
            __syncthreads();
            unsigned tot = 0;
            for (int i = p; i < PK_THREADS; i += PL) tot += chk[i];
            const int wrapped = __syncthreads_or((live && valid && tot != (unsigned)n) ? 1 : 0);
            if (!wrapped) break;
            if (a.stats && tid == 0) atomicAdd(a.stats + 2, 1ull);
            for (int i = tid; i < PK_HIST_WORDS; i += PK_THREADS) H[i] = 0u;
            if (tid == 0) *ctr = 0;
            __syncthreads();
        }
        }
        const double inv_scale = cm.inv_scale, center = cm.center, pivot = cm.pivot;
        // the bins epilogues keep deviations from the curve mean in units of 2^-s (the
        // fixed-point quantum): of order 1 .. 2^31 whatever the flux scale, so they fit fp32
        const double pivot_q = __dmul_rn(pivot, __ddiv_rn(1.0, inv_scale));   // exact
        const double center_s = a.center_out ? 0.0 : center;       // FoldArgs::center_out: centred sums
        if (a.center_out && p0 == 0 && tid == 0) a.center_out[curve] = center;
        const bool ok = live && valid;

        // The epilogues are compiled twice / four times: with and without the 32-bit side
        // counts (only ever present after a count-overflow refold), and for nbins == ROWS
        // (one row per bin) separately, so that the common case carries no dead branches.
        auto bins_epilogue = [&](auto side_c, auto m1_c) {
            constexpr bool SIDE = decltype(side_c)::value;
            constexpr bool M1 = decltype(m1_c)::value;
            const int MM = M1 ? 1 : M;
            // ---- epilogue (1): bins.  Lane (slot, p) takes the bins blk * 8 SL + e * SL + slot,
            // e = 0..7, of period p: rows of different slots differ mod SL (conflict-free).
            double *ps1 = reinterpret_cast<double *>(smem + PK_PS1_OFF);
            double *ps2 = reinterpret_cast<double *>(smem + PK_PS2_OFF);
            int *pkk = reinterpret_cast<int *>(smem + PK_PKK_OFF);
            double *st_mu = reinterpret_cast<double *>(smem + PK_MU_OFF);
            double *st_isd = reinterpret_cast<double *>(smem + PK_ISD_OFF);
            int *st_kk = reinterpret_cast<int *>(smem + PK_KK_OFF);
            const bool want_norm = a.out_norm != nullptr;
            const int nblk = nb / (8 * SL);
            const long long orow = (curve * a.nperiods + j) * nb;
            double s1 = 0.0, s2 = 0.0;
            int kk = 0;
            for (int blk = warp; blk < nblk; blk += PK_WARPS) {
                float fs[8];
                unsigned fc[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int bin = blk * 8 * SL + e * SL + slot;
                    int S = 0;
                    unsigned c = 0;
                    for (int jj = 0; jj < MM; ++jj) {
                        const int row = bin * MM + jj;
                        S += (int)H[row * PL + p];
                        c += pk_count<ROWLOG>(H, SIDE ? sd : nullptr, row, p);
                        H[row * PL + p] = 0u;
                    }
                    if (e == 0 && bin == 0) {       // the samples at u == 0 (CurveMeta::n_zero)
                        S += cm.q_zero;
                        c += (unsigned)cm.n_zero;
                    }
                    if (!ok) {
                        S = 0;
                        c = 0;
                    }
                    const double Sd = (double)S;
                    fs[e] = (float)__dadd_rn(__dmul_rn(Sd, inv_scale), __dmul_rn((double)c, center_s));
                    fc[e] = c;
                    if (want_norm) {
                        // deviation of the bin mean from the curve mean, kept as fp32 in the
                        // bin's (cleared) sum word for sweep 2: NaN = empty bin
                        float df = __int_as_float(0x7fc00000);
                        if (c > 0) {
                            const double d = __dsub_rn(pk_div_by_count(Sd, c), pivot_q);
                            s1 += d;
                            s2 += __dmul_rn(d, d);
                            kk += 1;
                            df = (float)d;
                        }
                        H[bin * MM * PL + p] = __float_as_uint(df);
                    }
                }
                if (live) {
                    const long long off = orow + blk * 8 * SL + slot;
                    if (SL == 1 && a.vec_ok) {
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
#pragma unroll
                        for (int e = 0; e < 8; ++e) {
                            if (a.out_sum) a.out_sum[off + e * SL] = fs[e];
                            if (a.out_count) a.out_count[off + e * SL] = fc[e];
                        }
                    }
                }
            }
            if (want_norm) {
                ps1[warp * 32 + lane] = s1;
                ps2[warp * 32 + lane] = s2;
                pkk[warp * 32 + lane] = kk;
                __syncthreads();
                if (tid < PL) {
                    double t1 = 0.0, t2 = 0.0;
                    int tk = 0;
                    for (int w = 0; w < PK_WARPS; ++w)            // fixed order: deterministic
                        for (int s = 0; s < SL; ++s) {
                            t1 += ps1[w * 32 + s * PL + tid];
                            t2 += ps2[w * 32 + s * PL + tid];
                            tk += pkk[w * 32 + s * PL + tid];
                        }
                    // mean and population std of the deviations, in units of 2^-s
                    double dm = 0.0, isd = 0.0;
                    if (tk > 0) {
                        dm = __ddiv_rn(t1, (double)tk);
                        const double var = __dsub_rn(__ddiv_rn(t2, (double)tk), __dmul_rn(dm, dm));
                        const double sdv = (var > 0.0) ? sqrt(var) : 0.0;
                        if (tk >= 2 && sdv > 0.0) isd = __ddiv_rn(1.0, sdv);
                    }
                    st_mu[tid] = dm;
                    st_isd[tid] = isd;
                    st_kk[tid] = tk;
                }
                __syncthreads();
                // sweep 2: normalised profile from the fp32 deviations (|d| is a few profile
                // sigmas, so fp32 keeps (d - dm) / s to ~1e-6), sum words cleared
                const double dm = st_mu[p], isd = st_isd[p];
                const double mu = __dadd_rn(pivot, __dmul_rn(dm, inv_scale));    // profile mean, flux units
                const double base_o = (ok && st_kk[p] > 0) ? __dadd_rn(mu, center) : 0.0;
                for (int blk = warp; blk < nblk; blk += PK_WARPS) {
                    float fn[8];
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const int i0 = (blk * 8 * SL + e * SL + slot) * MM * PL + p;
                        const float df = __uint_as_float(H[i0]);
                        H[i0] = 0u;
                        double o = base_o;
                        if (ok && df == df && isd > 0.0)
                            o = __dadd_rn(o, __dmul_rn(__dsub_rn((double)df, dm), isd));
                        fn[e] = (float)o;
                    }
                    if (live) {
                        const long long off = orow + blk * 8 * SL + slot;
                        if (SL == 1 && a.vec_ok) {
                            float4 *o4 = reinterpret_cast<float4 *>(a.out_norm + off);
                            o4[0] = make_float4(fn[0], fn[1], fn[2], fn[3]);
                            o4[1] = make_float4(fn[4], fn[5], fn[6], fn[7]);
                        } else {
#pragma unroll
                            for (int e = 0; e < 8; ++e) a.out_norm[off + e * SL] = fn[e];
                        }
                    }
                }
            }
            // every row has been read: clear the packed counts
            __syncthreads();
            for (int i = tid; i < HALF * PL; i += PK_THREADS) H[PK_CNT_OFF / 4 + i] = 0u;
        };
        // ---- epilogue (1b): bins, ROWS = nbins = 1024 (SL = 1, no side counts): config 3's
        // case.  With lane = period every store instruction touches 32 different 128-byte
        // lines (16 bytes each), and at 384 KB of output per work item the store unit, one line
        // per cycle, was the bottleneck of the epilogue (ncu: long_sb / mio stalls, 14 % of the
        // kernel).  So the arithmetic is done with lane = bin: every row vector of 32 words
        // (sums, packed counts) is first permuted in place, column p -> p ^ (row & 31); a warp
        // that then walks the rows 32 t + l of ONE period p reads column p ^ l -- 32 different
        // banks -- and every store is one full line.  Unit of work = (period, third of its 32
        // row tiles): 96 units, 4 per warp.  Bin mean through a table of correctly rounded
        // reciprocals (q0 = sq r, one residual correction: exact whenever the quotient is
        // representable, as pk_div_by_count); sweep 2 in fp32.
        auto bins_epilogue_lanebin = [&](auto all_c) {
            constexpr bool ALL = decltype(all_c)::value;    // sums, counts and normalised profile all wanted
            double *ps1 = reinterpret_cast<double *>(smem + PK_PS1_OFF);      // [96] per unit
            double *ps2 = reinterpret_cast<double *>(smem + PK_PS2_OFF);
            int *pkk = reinterpret_cast<int *>(smem + PK_PKK_OFF);
            float *st_dm = reinterpret_cast<float *>(smem + PK_MU_OFF);       // [32] per period
            float *st_isd = st_dm + 32;
            float *st_base = st_dm + 64;
            const double2 *rt = reinterpret_cast<const double2 *>(smem + PK_RT_OFF);
            const bool want_norm = ALL || a.out_norm != nullptr;
            const bool w_sum = ALL || a.out_sum != nullptr, w_cnt = ALL || a.out_count != nullptr;
            unsigned *Hc = H + PK_CNT_OFF / 4;
            // the item's validity per period (lane = period here) for the lane = bin phases
            const unsigned livemask = __ballot_sync(0xffffffffu, live);
            const unsigned okmask = __ballot_sync(0xffffffffu, ok);
            // the samples at u == 0 (CurveMeta::n_zero) belong to row 0: warp 0 adds them to the
            // row vectors it permutes first below
            if (warp == 0 && cm.n_zero > 0) {
                H[lane] += (unsigned)cm.q_zero;
                Hc[lane] += (unsigned)cm.n_zero;
            }
            // phase A: permute the row vectors (1024 of sums, 512 of packed counts)
#pragma unroll 4
            for (int v = warp; v < ROWS + HALF; v += PK_WARPS) {
                unsigned *hv = H + v * 32;                  // the counts follow the sums
                const unsigned xw = hv[lane];
                hv[lane ^ (v & 31)] = xw;                   // the warp's loads complete before its store issues
            }
            __syncthreads();
            const long long obase = (curve * a.nperiods + p0) * ROWS;
            constexpr int UPW = 96 / PK_WARPS;                 // units per warp
            // sweep 1
#pragma unroll 1
            for (int i = 0; i < UPW; ++i) {
                const int u = warp * UPW + i;
                const int pp = u / 3, part = u - pp * 3;
                const int t_lo = part * 11, t_hi = min(32, t_lo + 11);
                const bool lv = (livemask >> pp) & 1u, okp = (okmask >> pp) & 1u;
                // running pointers (kept opaque so that they stay in registers)
                unsigned long long po = (unsigned long long)(obase + (long long)pp * ROWS + t_lo * 32 + lane) * 4ull;
                asm volatile("" : "+l"(po));
                unsigned hs = (unsigned)((t_lo * 32 + lane) * 32 + (pp ^ lane));      // word index of (row, col)
                asm volatile("" : "+r"(hs));
                double s1 = 0.0, s2 = 0.0;
                int kk = 0;
#pragma unroll 2
                for (int t = t_lo; t < t_hi; ++t) {
                    int S = (int)H[hs];
                    const unsigned w = Hc[hs & (HALF * 32 - 1)];
                    unsigned c = (t >= 16) ? (w >> 16) : ((w & 0xffffu) - (w >> 16));
                    S = okp ? S : 0;
                    c = okp ? c : 0u;
                    const double Sd = (double)S;
                    double r, cd;
                    if (c < (unsigned)PK_RT_N) {
                        const double2 tb = rt[c];          // c == 0: {inf, 0}, discarded below
                        r = tb.x;
                        cd = tb.y;
                    } else {
                        cd = (double)c;
                        r = __ddiv_rn(1.0, cd);
                    }
                    if (w_sum && lv)
                        *reinterpret_cast<float *>((char *)a.out_sum + po) =
                            (float)__dadd_rn(__dmul_rn(Sd, inv_scale), __dmul_rn(cd, center_s));
                    if (w_cnt && lv) *reinterpret_cast<uint32_t *>((char *)a.out_count + po) = c;
                    unsigned dw = 0u;
                    if (want_norm) {
                        const double q0 = __dmul_rn(Sd, r);
                        const double m = __fma_rn(__fma_rn(-q0, cd, Sd), r, q0);      // S / c, units of 2^-s
                        const bool nz = c > 0u;
                        const double d = nz ? __dsub_rn(m, pivot_q) : 0.0;
                        s1 += d;
                        s2 += __dmul_rn(d, d);
                        kk += nz ? 1 : 0;
                        dw = nz ? __float_as_uint((float)d) : 0x7fc00000u;    // NaN: empty bin
                    }
                    H[hs] = dw;
                    hs += 32 * 32;
                    po += 128;
                }
                if (want_norm) {
                    s1 = warp_sum(s1);
                    s2 = warp_sum(s2);
                    kk = warp_sum_int(kk);
                    if (lane == 0) {
                        ps1[u] = s1;
                        ps2[u] = s2;
                        pkk[u] = kk;
                    }
                }
            }
            __syncthreads();   // every packed count word has been read (twice): they can go
            if (want_norm) {
                if (tid < PL) {
                    double t1 = 0.0, t2 = 0.0;
                    int tk = 0;
                    for (int q3 = 0; q3 < 3; ++q3) {               // fixed order: deterministic
                        t1 += ps1[tid * 3 + q3];
                        t2 += ps2[tid * 3 + q3];
                        tk += pkk[tid * 3 + q3];
                    }
                    // mean and population std of the deviations, in units of 2^-s
                    double dm = 0.0, isd = 0.0;
                    if (tk > 0) {
                        dm = __ddiv_rn(t1, (double)tk);
                        const double var = __dsub_rn(__ddiv_rn(t2, (double)tk), __dmul_rn(dm, dm));
                        const double sdv = (var > 0.0) ? sqrt(var) : 0.0;
                        if (tk >= 2 && sdv > 0.0) isd = __ddiv_rn(1.0, sdv);
                    }
                    const double mu = __dadd_rn(pivot, __dmul_rn(dm, inv_scale));   // profile mean, flux units
                    // tid is the period here, as in `ok`
                    st_dm[tid] = (float)dm;
                    st_isd[tid] = ok ? (float)isd : 0.f;
                    st_base[tid] = (ok && tk > 0) ? (float)__dadd_rn(mu, center) : 0.f;
                }
                __syncthreads();
            }
            // sweep 2: out = base + (d - dm) / s from the fp32 deviations, in fp32 (a z-score of a
            // few units plus mu + center: each rounding is 6e-8 relative, the bar is 1e-4);
            // every word of the histogram cleared
#pragma unroll 1
            for (int i = 0; i < UPW; ++i) {
                const int u = warp * UPW + i;
                const int pp = u / 3, part = u - pp * 3;
                const int t_lo = part * 11, t_hi = min(32, t_lo + 11);
                const bool lv = ((livemask >> pp) & 1u) && want_norm;
                unsigned long long po = (unsigned long long)(obase + (long long)pp * ROWS + t_lo * 32 + lane) * 4ull;
                asm volatile("" : "+l"(po));
                unsigned hs = (unsigned)((t_lo * 32 + lane) * 32 + (pp ^ lane));
                asm volatile("" : "+r"(hs));
                float dmf = 0.f, isdf = 0.f, basef = 0.f;
                if (want_norm) {
                    dmf = st_dm[pp];
                    isdf = st_isd[pp];
                    basef = st_base[pp];
                }
#pragma unroll 2
                for (int t = t_lo; t < t_hi; ++t) {
                    const float df = __uint_as_float(H[hs]);
                    H[hs] = 0u;
                    if (t < 16) Hc[hs] = 0u;
                    // NaN (empty bin) or s == 0: the profile mean
                    const float z = __fmaf_rn(__fsub_rn(df, dmf), isdf, basef);
                    const float o = (df == df && isdf > 0.f) ? z : basef;
                    if (lv) *reinterpret_cast<float *>((char *)a.out_norm + po) = o;
                    hs += 32 * 32;
                    po += 128;
                }
            }
        };
        auto merge_epilogue = [&](auto side_c) {
            constexpr bool SIDE = decltype(side_c)::value;
            // ---- epilogue (2): equal-count merge of the nb = ROWS intermediary bins into nb2
            // bins ("Fourthly", reading R18), per period p:
            //   N = total count, per = N / nb2, target_b = per (b + 1) (= N for the last bin);
            //   boundary b lies in the first row k with C(k) >= target_b (C = cumulative count),
            //   Scum_b = S(k-1) + ((target_b - C(k-1)) / count_k) sum_k,
            //   mean_b = (Scum_b - Scum_{b-1}) / per.
            // Phases: every thread (chunk c, period p) adds up its 2-6 mini-chunks of MCR rows ->
            // prefix over threads: cumulative count / integer flux in front of every mini-chunk
            // (exact: |any partial sum of q| < 2^31 by the choice of the scale) -> one
            // (boundary, period) per lane: binary search of the mini-chunk, walk of at most
            // MCR rows, the fp64 part -> means, statistics, write-out.
            constexpr int MCR = (PL == 8) ? 8 : 16;        // rows per mini-chunk
            constexpr int NMC = ROWS / MCR;                // mini-chunks: 512 / 128 / 64
            constexpr int NCH = PK_THREADS / PL;           // threads per period: 96 / 48 / 24
            constexpr int MNUM = NMC / (NCH / 3);          // a thread owns MNUM / 3 mini-chunks
            constexpr int MPT = MNUM / 3 + 1;              // ... at most (6 / 3 / 3)
            static_assert(NCH % 3 == 0 && (NCH / 3) * MNUM == NMC, "mini-chunks split evenly");
            static_assert(NMC * PL * 8 + PK_WARPS * PL * 8 <= PK_SCR_BYTES, "merge-epilogue scratch");
            unsigned *ec = reinterpret_cast<unsigned *>(smem + PK_SCR_OFF);             // [NMC][PL]
            int *eq = reinterpret_cast<int *>(smem + PK_SCR_OFF) + NMC * PL;            // [NMC][PL]
            unsigned *wtc = reinterpret_cast<unsigned *>(smem + PK_SCR_OFF) + 2 * NMC * PL;   // [warp][PL]
            int *wtq = reinterpret_cast<int *>(wtc) + PK_WARPS * PL;                    // [warp][PL]
            double *part = reinterpret_cast<double *>(wtc);                             // [warp][PL], later
            double *scum = reinterpret_cast<double *>(smem);                            // [nb2 + 1][PL], over H
            const int nb2 = a.nb2;
            if (cm.n_zero > 0) {
                // the samples at u == 0 (CurveMeta::n_zero, at most 255) belong to row 0
                if (tid < PL) {
                    H[tid] += (unsigned)cm.q_zero;
                    H[PK_CNT_OFF / 4 + tid] += (unsigned)cm.n_zero;
                }
                __syncthreads();
            }
            const int ch = warp * SL + slot;
            const int m_lo = (ch * MNUM) / 3, m_hi = ((ch + 1) * MNUM) / 3;
            // phase 1: totals of this thread's mini-chunks (slot s starts s rows into each, so
            // the SL slots of a warp read rows that differ mod SL: conflict-free)
            unsigned lc[MPT];
            int lq[MPT];
            unsigned tc = 0;
            int tq = 0;
#pragma unroll
            for (int k = 0; k < MPT; ++k) {
                unsigned c1 = 0;
                int q1 = 0;
                if (m_lo + k < m_hi) {
#pragma unroll
                    for (int i = 0; i < MCR; ++i) {
                        const int row = (m_lo + k) * MCR + ((i + slot) & (MCR - 1));
                        c1 += pk_count<ROWLOG>(H, SIDE ? sd : nullptr, row, p);
                        q1 += (int)H[row * PL + p];
                    }
                }
                lc[k] = tc;            // exclusive prefix inside the thread
                lq[k] = tq;
                tc += c1;
                tq += q1;
            }
            unsigned ci = tc;
            int qi = tq;
#pragma unroll
            for (int o = 1; o < SL; o <<= 1) {
                const unsigned cu = __shfl_up_sync(0xffffffffu, ci, o * PL);
                const int qu = __shfl_up_sync(0xffffffffu, qi, o * PL);
                if (slot >= o) {
                    ci += cu;
                    qi += qu;
                }
            }
            if (slot == SL - 1) {
                wtc[warp * PL + p] = ci;
                wtq[warp * PL + p] = qi;
            }
            __syncthreads();
            // phase 2: points / integer flux in front of this thread, total of the period;
            // table of the cumulative values in front of every mini-chunk
            unsigned cb = ci - tc, ntot = 0;
            int qb = qi - tq;
            for (int w = 0; w < PK_WARPS; ++w) {
                const unsigned c = wtc[w * PL + p];
                if (w < warp) {
                    cb += c;
                    qb += wtq[w * PL + p];
                }
                ntot += c;
            }
            if (!ok) ntot = 0;
#pragma unroll
            for (int k = 0; k < MPT; ++k)
                if (m_lo + k < m_hi) {
                    ec[(m_lo + k) * PL + p] = cb + lc[k];
                    eq[(m_lo + k) * PL + p] = qb + lq[k];
                }
            __syncthreads();
            // phase 3: boundary b of period p: first row k with C(k) >= thr_b = ceil(target_b)
            // (C >= target <=> C >= thr for an integer C), then the cumulative flux there
            const double total = (double)ntot;
            const double per = __ddiv_rn(total, (double)nb2);
            double sv[3];
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                sv[k] = 0.0;
                const int b = ch + k * NCH;
                if (b < nb2 && ntot > 0u) {
                    const double target = (b == nb2 - 1) ? total : __dmul_rn(per, (double)(b + 1));
                    const unsigned thr = (unsigned)ceil(target);
                    int m = 0;                           // last mini-chunk with fewer than thr points in front
#pragma unroll
                    for (int step = NMC / 2; step >= 1; step >>= 1)
                        if (ec[(m + step) * PL + p] < thr) m += step;
                    unsigned cbef = ec[m * PL + p], cnt = 0;
                    int qbef = eq[m * PL + p], q = 0;
                    int row = m * MCR;
                    for (int i = 0; i < MCR; ++i, ++row) {
                        cnt = pk_count<ROWLOG>(H, SIDE ? sd : nullptr, row, p);
                        q = (int)H[row * PL + p];
                        if (cbef + cnt >= thr || i == MCR - 1) break;
                        cbef += cnt;
                        qbef += q;
                    }
                    const double ck = (double)cnt, cbd = (double)cbef;
                    const double sbef = __dadd_rn(__dmul_rn((double)qbef, inv_scale), __dmul_rn(cbd, center));
                    const double sk = __dadd_rn(__dmul_rn((double)q, inv_scale), __dmul_rn(ck, center));
                    double frac = (cnt > 0u) ? __ddiv_rn(__dsub_rn(target, cbd), ck) : 0.0;
                    frac = fmin(fmax(frac, 0.0), 1.0);
                    sv[k] = __dadd_rn(sbef, __dmul_rn(frac, sk));
                }
            }
            __syncthreads();   // the histogram has been read for the last time: scum goes over it
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const int b = ch + k * NCH;
                if (b < nb2) scum[(b + 1) * PL + p] = sv[k];
            }
            if (ch == 0) scum[p] = 0.0;
            __syncthreads();
            // phase 4: means; mean and population std over the nb2 bins, summed
            // in a fixed order (slots by shuffle, warps in order)
            double mv[3], s1 = 0.0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                mv[k] = 0.0;
                const int b = ch + k * NCH;
                if (b < nb2 && ntot > 0u)
                    mv[k] = __ddiv_rn(__dsub_rn(scum[(b + 1) * PL + p], scum[b * PL + p]), per);
                s1 += mv[k];
            }
#pragma unroll
            for (int o = PL; o < 32; o <<= 1) s1 += __shfl_xor_sync(0xffffffffu, s1, o);
            if (slot == 0) part[warp * PL + p] = s1;
            __syncthreads();
            double mu = 0.0;
            for (int w = 0; w < PK_WARPS; ++w) mu += part[w * PL + p];
            mu = __ddiv_rn(mu, (double)nb2);
            double s2 = 0.0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const double d = (ch + k * NCH < nb2) ? __dsub_rn(mv[k], mu) : 0.0;
                s2 += __dmul_rn(d, d);
            }
#pragma unroll
            for (int o = PL; o < 32; o <<= 1) s2 += __shfl_xor_sync(0xffffffffu, s2, o);
            __syncthreads();
            if (slot == 0) part[warp * PL + p] = s2;
            __syncthreads();
            if (live) {
                double vacc = 0.0;
                for (int w = 0; w < PK_WARPS; ++w) vacc += part[w * PL + p];
                const double sdv = sqrt(__ddiv_rn(vacc, (double)nb2));
                const bool flat = (nb2 < 2) || !(sdv > 0.0);
                const long long off = (curve * a.nperiods + j) * nb2;
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    const int b = ch + k * NCH;
                    if (b < nb2) {
                        float om = 0.f, on = 0.f;
                        if (ntot > 0u) {
                            om = (float)mv[k];
                            on = (float)(flat ? mu : __dadd_rn(mu, __ddiv_rn(__dsub_rn(mv[k], mu), sdv)));
                        }
                        if (a.out_mean2) a.out_mean2[off + b] = om;
                        if (a.out_norm2) a.out_norm2[off + b] = on;
                    }
                }
            }
            __syncthreads();
            // clear the whole histogram
            uint4 *H4 = reinterpret_cast<uint4 *>(H);
            for (int i = tid; i < PK_HIST_BYTES / 16; i += PK_THREADS) H4[i] = make_uint4(0u, 0u, 0u, 0u);
        };
        using TrueT = PkBool<true>;
        using FalseT = PkBool<false>;
        if (a.nb2 == 0) {
            if (sd)
                bins_epilogue(TrueT{}, FalseT{});
            else if (M == 1) {
                if constexpr (ROWLOG == 10) {
                    if (a.out_sum && a.out_count && a.out_norm)
                        bins_epilogue_lanebin(TrueT{});
                    else
                        bins_epilogue_lanebin(FalseT{});
                }
                else
                    bins_epilogue(FalseT{}, TrueT{});
            }
            else
                bins_epilogue(FalseT{}, FalseT{});
        } else {
            if (sd)
                merge_epilogue(TrueT{});
            else
                merge_epilogue(FalseT{});
        }
        if (tid == 0) *ctr = 0;
        __syncthreads();   // H is zero again, tile counter reset
    }
}

template <int ROWLOG>
__global__ void __launch_bounds__(PK_THREADS, 1)
fold_pk_kernel(FoldArgs a, long long ngroups, long long nitems)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    const unsigned sbase = (unsigned)__cvta_generic_to_shared(smem);
    if (sbase == PK_WINDOW_BASE)
        fold_pk_body<ROWLOG, true>(a, ngroups, nitems, smem, sbase);
    else
        fold_pk_body<ROWLOG, false>(a, ngroups, nitems, smem, sbase);
}

template <int ROWLOG>
cudaError_t pk_set_attr()
{
    return cudaFuncSetAttribute(fold_pk_kernel<ROWLOG>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                PK_SMEM_BYTES);
}

template <int ROWLOG>
cudaError_t pk_launch(const FoldArgs &a, cudaStream_t st, int sms)
{
    constexpr int PL = PkV<ROWLOG>::PL;
    const long long ngroups = (a.nperiods + PL - 1) / PL;
    const long long nitems = ngroups * a.ncurves;
    const long long grid = nitems < sms ? nitems : sms;
    fold_pk_kernel<ROWLOG><<<(unsigned)grid, PK_THREADS, PK_SMEM_BYTES, st>>>(a, ngroups, nitems);
    note_launch();
    return cudaGetLastError();
}

}  // namespace

bool fold_pk_handles(int nbins) { return nbins == 512 || nbins == 1024 || nbins == 2048 || nbins == 4096; }

int fold_pk_rows(int nbins) { return nbins <= 1024 ? 1024 : nbins; }

bool fold_pk_can_merge(int nbins, int nb2)
{
    if (!(nbins == 1024 || nbins == 2048 || nbins == 4096) || nb2 < 1) return false;
    return (32768 / nbins) * nb2 <= PK_MG_MAX;
}

size_t fold_pk_side_bytes(int sms) { return (size_t)sms * PK_CELLS * sizeof(unsigned); }

long long fold_pk_flush_samples() { return (long long)PK_FLUSH_TILES * GPFC_TILE; }

cudaError_t fold_pk_init_device()
{
    cudaError_t e = pk_set_attr<10>();
    if (e == cudaSuccess) e = pk_set_attr<11>();
    if (e == cudaSuccess) e = pk_set_attr<12>();
    return e;
}

cudaError_t launch_fold_pk(const FoldArgs &a, cudaStream_t st, int sms)
{
    if (a.nbins <= 1024) return pk_launch<10>(a, st, sms);
    if (a.nbins == 2048) return pk_launch<11>(a, st, sms);
    return pk_launch<12>(a, st, sms);
}

}  // namespace gpfc
