// Roofline calibration micro-kernels (gpfc_measure_peaks): the
// measured peak rates of the units that bound the fold on this GPU, in this run,
// at these clocks.
//   [0] conflict-free shared-memory atomic lane-updates/s: every lane owns a bank,
//       half ATOMS.ADD, half ATOMS.POPC.INC, addresses precomputed, no other work
//   [1] fp64 DMUL + DADD(round-down) pairs/s
//   [3] fp32 atomicAdd on shared memory (CAS loop), same access pattern as [0]
//   [4] plain LDS + add + STS on warp-private rows (no atomics)
//   [2] the inner loop of fold_lp_kernel<0> alone (DFMA.RM, PRMT, VIMNMX3, 2 atomics per
//       point-period, samples broadcast from shared memory): the ceiling of the fold loop
//       with no global loads, tile set-up, epilogue or barriers
#include "common.cuh"

namespace gpfc {

namespace {

extern __shared__ __align__(16) unsigned char peaks_smem[];

__global__ void __launch_bounds__(1024, 1) peak_atoms_kernel(int iters, unsigned *sink)
{
    unsigned *h = reinterpret_cast<unsigned *>(peaks_smem);   // [rows][32]
    constexpr int ROWS = 1024;
    const int lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < ROWS * 32; i += blockDim.x) h[i] = 0;
    __syncthreads();
    unsigned idx[8];
    unsigned s = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 12345u;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        s = s * 1664525u + 1013904223u;
        idx[k] = ((s >> 8) % ROWS) * 32 + lane;
    }
    const unsigned v = lane + 1;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; k += 2) {
            atomicAdd(&h[idx[k]], v);
            atomicAdd(&h[idx[k + 1]], 1u);
        }
    }
    __syncthreads();
    unsigned acc = 0;
    for (int i = threadIdx.x; i < ROWS * 32; i += blockDim.x) acc += h[i];
    if (acc == 0xdeadbeefu) sink[0] = acc;
}

// [3] the same access pattern with fp32 atomicAdd (a compare-and-swap loop on sm_100a) and
// [4] with plain LDS + IADD + STS on warp-private rows (no atomics): the two alternatives to
// native integer atomics that the design rejected.
__global__ void __launch_bounds__(1024, 1) peak_casf_kernel(int iters, float *sink)
{
    float *h = reinterpret_cast<float *>(peaks_smem);   // [rows][32]
    constexpr int ROWS = 1024;
    const int lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < ROWS * 32; i += blockDim.x) h[i] = 0.f;
    __syncthreads();
    unsigned idx[8];
    unsigned s = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 12345u;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        s = s * 1664525u + 1013904223u;
        idx[k] = ((s >> 8) % ROWS) * 32 + lane;
    }
    const float v = (float)(lane + 1);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k) atomicAdd(&h[idx[k]], v);
    }
    __syncthreads();
    float acc = 0.f;
    for (int i = threadIdx.x; i < ROWS * 32; i += blockDim.x) acc += h[i];
    if (acc == -1.f) sink[0] = acc;
}

__global__ void __launch_bounds__(1024, 1) peak_ldsts_kernel(int iters, unsigned *sink)
{
    unsigned *h = reinterpret_cast<unsigned *>(peaks_smem);   // [warp][rows][32]: private per warp
    constexpr int ROWS = 32;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < 32 * ROWS * 32; i += blockDim.x) h[i] = 0;
    __syncthreads();
    unsigned idx[8];
    unsigned s = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 12345u;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        s = s * 1664525u + 1013904223u;
        idx[k] = (warp * ROWS + ((s >> 8) % ROWS)) * 32 + lane;
    }
    const unsigned v = lane + 1;
    volatile unsigned *hv = h;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k) hv[idx[k]] = hv[idx[k]] + v;
    }
    __syncthreads();
    unsigned acc = 0;
    for (int i = threadIdx.x; i < 32 * ROWS * 32; i += blockDim.x) acc += h[i];
    if (acc == 0xdeadbeefu) sink[0] = acc;
}

__global__ void __launch_bounds__(1024, 1) peak_fp64_kernel(int iters, double seed, double *sink)
{
    double u[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) u[k] = seed * (double)(threadIdx.x + 32 * k + 1);
    double r = 1.0 + seed;
    const double M = 6755399441055744.0 / 16777216.0;
    unsigned acc = 0;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            double y = __dmul_rn(u[k], r);
            double m = __dadd_rd(y, M);
            acc ^= (unsigned)__double2loint(m);
        }
        r = __longlong_as_double(__double_as_longlong(r) + 1);
    }
    if (acc == 0xdeadbeefu) sink[0] = (double)acc;
}

// [2] the inner loop of fold_lp_kernel<false> alone (lane = period, 3 periods per lane, 8-byte
// sample records broadcast from shared memory, DFMA.RM + PRMT + VIMNMX3 + ATOMS.ADD +
// ATOMS.POPC.INC per point-period, 32 samples per iteration): no global loads, tile set-up,
// epilogue or barriers.
template <int IMM>
__device__ __forceinline__ void pk_red_add(unsigned addr, int v)
{
    asm volatile("red.shared.add.u32 [%0+%2], %1;" ::"r"(addr), "r"(v), "n"(IMM) : "memory");
}
template <int IMM>
__device__ __forceinline__ void pk_red_inc(unsigned addr)
{
    asm volatile("red.shared.add.u32 [%0+%1], 1;" ::"r"(addr), "n"(IMM) : "memory");
}

__global__ void __launch_bounds__(768, 1) peak_loop_kernel(int nsamples, double seed, unsigned *sink)
{
    unsigned *H = reinterpret_cast<unsigned *>(peaks_smem);          // [3][256][2][32]
    int4 *rec = reinterpret_cast<int4 *>(peaks_smem + 196608);        // 64 records of 8 bytes x 2
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < 49152; i += blockDim.x) H[i] = 0;
    if (threadIdx.x < 64)
        rec[threadIdx.x] = make_int4(threadIdx.x * 40503 + 17, (int)threadIdx.x - 30,
                                     threadIdx.x * 65599 + 3, 31 - (int)threadIdx.x);
    __syncthreads();
    const unsigned sbase = (unsigned)__cvta_generic_to_shared(peaks_smem);   // kept in a uniform register
    const unsigned lane4 = (unsigned)lane << 2;
    double rp[3], C[3];
#pragma unroll
    for (int r = 0; r < 3; ++r) {
        rp[r] = (256.0 + 8.0 * (r * 32 + lane)) * 0.020433 * (1.0 / 33554432.0) * (1.0 + seed);
        C[r] = 1048576.0 + (double)((r * 97 + lane * 13) & 255) + 0.375;
    }
    unsigned gmin = 0xffffffffu;
    // as fold_lp.cu's fold_granule: 32 samples per iteration, per sample the three sums before
    // the three counts
    for (int s0 = warp * 32; s0 < nsamples; s0 += 32 * (blockDim.x >> 5)) {
#pragma unroll
        for (int g = 0; g < 8; ++g) {
            const int4 ra = rec[((s0 >> 1) + 2 * g) & 31], rb = rec[((s0 >> 1) + 2 * g + 1) & 31];
            const unsigned iv[4] = {(unsigned)ra.x + s0, (unsigned)ra.z + s0, (unsigned)rb.x + s0,
                                    (unsigned)rb.z + s0};
            const int q[4] = {ra.y, ra.w, rb.y, rb.w};
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const double v = (double)iv[k];
                unsigned addr[3];
#pragma unroll
                for (int r = 0; r < 3; ++r) {
                    double m = __fma_rd(v, rp[r], C[r]);
                    unsigned lo = (unsigned)__double2loint(m), hi = (unsigned)__double2hiint(m);
                    addr[r] = __byte_perm(lane4, hi, 0x3240) + sbase;
                    gmin = min(gmin, lo);
                }
                pk_red_add<0>(addr[0], q[k]);
                pk_red_add<65536>(addr[1], q[k]);
                pk_red_add<131072>(addr[2], q[k]);
                pk_red_inc<128>(addr[0]);
                pk_red_inc<65536 + 128>(addr[1]);
                pk_red_inc<131072 + 128>(addr[2]);
            }
        }
    }
    __syncthreads();
    unsigned acc = gmin;
    for (int i = threadIdx.x; i < 49152; i += blockDim.x) acc += H[i];
    if (acc == 0xdeadbeefu) sink[0] = acc;
}

}  // namespace

cudaError_t measure_peaks(double *out, cudaStream_t st)
{
    for (int i = 0; i < 8; ++i) out[i] = 0.0;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    void *sink = nullptr;
    cudaError_t e = cudaMalloc(&sink, 256);
    if (e != cudaSuccess) return e;
    cudaEvent_t a, b;
    cudaEventCreate(&a);
    cudaEventCreate(&b);
    const size_t smem_atoms = 1024 * 32 * 4, smem_loop = 196608 + 1024;
    cudaFuncSetAttribute(peak_atoms_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         (int)smem_atoms);
    cudaFuncSetAttribute(peak_loop_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         (int)smem_loop);
    cudaFuncSetAttribute(peak_casf_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         (int)smem_atoms);
    cudaFuncSetAttribute(peak_ldsts_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         (int)smem_atoms);
    const int iters = 4000, nper = 400000;   // nper: samples per CTA of the loop kernel
    for (int which = 0; which < 5; ++which) {
        float best = 1e30f;
        for (int rep = 0; rep < 4; ++rep) {
            cudaEventRecord(a, st);
            if (which == 0)
                peak_atoms_kernel<<<sms, 1024, smem_atoms, st>>>(iters, (unsigned *)sink);
            else if (which == 1)
                peak_fp64_kernel<<<sms * 2, 1024, 0, st>>>(iters, 1e-3, (double *)sink);
            else if (which == 2)
                peak_loop_kernel<<<sms, 768, smem_loop, st>>>(nper, 0.25, (unsigned *)sink);
            else if (which == 3)
                peak_casf_kernel<<<sms, 1024, smem_atoms, st>>>(iters / 4, (float *)sink);
            else
                peak_ldsts_kernel<<<sms, 1024, smem_atoms, st>>>(iters, (unsigned *)sink);
            cudaEventRecord(b, st);
            e = cudaEventSynchronize(b);
            if (e != cudaSuccess) break;
            float ms = 0;
            cudaEventElapsedTime(&ms, a, b);
            if (rep > 0 && ms < best) best = ms;
        }
        if (e != cudaSuccess) break;
        double units = 0;
        if (which == 0) units = (double)sms * 1024 * iters * 8.0;
        if (which == 1) units = (double)sms * 2 * 1024 * iters * 8.0;
        if (which == 2) units = (double)sms * (double)nper * 96.0;
        if (which == 3) units = (double)sms * 1024 * (iters / 4) * 8.0;
        if (which == 4) units = (double)sms * 1024 * iters * 8.0;
        out[which] = units / (best * 1e-3);
    }
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    cudaFree(sink);
    if (e == cudaSuccess) e = cudaGetLastError();
    return e;
}

}  // namespace gpfc
