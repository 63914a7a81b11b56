// Trial-period grid: every operation individually rounded
// (intrinsics), so the device grid is bit-identical to the formula in gpfc.h.
#include "common.cuh"

namespace gpfc {

namespace {

__global__ void grid_kernel(double pmin, double pmax, long long nperiods, int mode_flags,
                            double *__restrict__ out)
{
    long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= nperiods) return;
    long long d = (mode_flags & GPFC_GRID_ENDPOINT_EXCLUSIVE) ? nperiods : nperiods - 1;
    if (d < 1) d = 1;
    const double dd = (double)d;
    double v;
    if (mode_flags & GPFC_GRID_UNIFORM_PERIOD) {
        double span = __dsub_rn(pmax, pmin);
        double step = __ddiv_rn(__dmul_rn(span, (double)j), dd);
        v = __dadd_rn(pmin, step);
    } else {
        double fmin = __ddiv_rn(1.0, pmax);
        double fmax = __ddiv_rn(1.0, pmin);
        double span = __dsub_rn(fmax, fmin);
        double step = __ddiv_rn(__dmul_rn(span, (double)j), dd);
        double f = __dadd_rn(fmin, step);
        v = __ddiv_rn(1.0, f);
    }
    out[j] = v;
}

}  // namespace

cudaError_t launch_grid(double pmin, double pmax, long long nperiods, int mode_flags,
                        double *out, cudaStream_t st)
{
    if (nperiods <= 0) return cudaSuccess;
    unsigned blocks = (unsigned)((nperiods + 255) / 256);
    grid_kernel<<<blocks, 256, 0, st>>>(pmin, pmax, nperiods, mode_flags, out);
    note_launch();
    return cudaGetLastError();
}

}  // namespace gpfc
