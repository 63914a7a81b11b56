// C ABI of libgpfc.so (include/gpfc.h): argument validation, scratch carving,
// launches.  No compute happens on the host and there is no CPU fallback.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <vector>

#include "common.cuh"

namespace {

struct ThreadState {
    cudaStream_t stream = nullptr;
    void *ws = nullptr;
    size_t ws_bytes = 0;
    char err[512] = "";
    // gpfc_profile: CUDA-event pairs around every fold-kernel launch + launch counter
    bool profiling = false;
    long long launches = 0;
    std::vector<cudaEvent_t> ev;      // start, stop, start, stop, ...
};

thread_local ThreadState g_ts;

int fail(int code, const char *fmt, const char *detail = "")
{
    snprintf(g_ts.err, sizeof(g_ts.err), fmt, detail);
    return code;
}

int cuda_fail(cudaError_t e, const char *where)
{
    snprintf(g_ts.err, sizeof(g_ts.err), "%s: %s", where, cudaGetErrorString(e));
    return GPFC_ERR_CUDA;
}

size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

size_t scratch_bytes(int64_t ncurves, int64_t n_total, int64_t nperiods)
{
    size_t b = 0;
    b += align_up((size_t)n_total * sizeof(double));
    b += align_up((size_t)n_total * sizeof(int));
    b += align_up(((size_t)n_total + (size_t)ncurves + 2) * sizeof(int2));
    b += align_up(((size_t)n_total / gpfc::GPFC_TILE + (size_t)ncurves + 1) * sizeof(gpfc::TileInfo));
    b += align_up((size_t)ncurves * sizeof(gpfc::CurveMeta));
    b += align_up((size_t)nperiods * sizeof(double));
    b += align_up(2 * sizeof(int64_t));   // offsets of the single-curve call
    return b + 256;
}

__global__ void set_offsets_kernel(int64_t *o, int64_t n)
{
    o[0] = 0;
    o[1] = n;
}

// The device path shared by every fold entry point.
int fold_device(const double *times, const float *flux, const int64_t *offsets, int64_t ncurves,
                int64_t n_total, const double *periods, int64_t nperiods, int nbins,
                const double *t0v, double t0_scalar, float *out_sum, uint32_t *out_count,
                float *out_norm)
{
    if (ncurves < 0 || nperiods < 0 || n_total < 0)
        return fail(GPFC_ERR_INVALID_ARG, "negative size%s");
    if (nbins < 1 || nbins > GPFC_MAX_NBINS)
        return fail(GPFC_ERR_UNSUPPORTED, "nbins must be in [1, 4096]%s");
    if (ncurves == 0 || nperiods == 0) return GPFC_OK;
    if (!periods) return fail(GPFC_ERR_INVALID_ARG, "periods is NULL%s");
    if (n_total > 0 && (!times || !flux)) return fail(GPFC_ERR_INVALID_ARG, "times/flux is NULL%s");
    if (!out_sum && !out_count && !out_norm) return GPFC_OK;

    cudaStream_t st = g_ts.stream;
    size_t need = scratch_bytes(ncurves, n_total, nperiods);
    char *base = nullptr;
    bool own = false;
    if (g_ts.ws && g_ts.ws_bytes >= need) {
        base = static_cast<char *>(g_ts.ws);
    } else {
        void *p = nullptr;
        cudaError_t e = cudaMallocAsync(&p, need, st);
        if (e != cudaSuccess) {
            cuda_fail(e, "scratch allocation");
            return GPFC_ERR_WORKSPACE;
        }
        base = static_cast<char *>(p);
        own = true;
    }
    char *cur = reinterpret_cast<char *>(align_up(reinterpret_cast<size_t>(base)));
    gpfc::Scratch s;
    s.u = reinterpret_cast<double *>(cur);
    cur += align_up((size_t)n_total * sizeof(double));
    s.q = reinterpret_cast<int *>(cur);
    cur += align_up((size_t)n_total * sizeof(int));
    s.rec = reinterpret_cast<int2 *>(cur);
    cur += align_up(((size_t)n_total + (size_t)ncurves + 2) * sizeof(int2));
    s.tiles = reinterpret_cast<gpfc::TileInfo *>(cur);
    cur += align_up(((size_t)n_total / gpfc::GPFC_TILE + (size_t)ncurves + 1) * sizeof(gpfc::TileInfo));
    s.meta = reinterpret_cast<gpfc::CurveMeta *>(cur);
    cur += align_up((size_t)ncurves * sizeof(gpfc::CurveMeta));
    s.rp = reinterpret_cast<double *>(cur);
    cur += align_up((size_t)nperiods * sizeof(double));
    int64_t *own_off = reinterpret_cast<int64_t *>(cur);

    cudaError_t e = cudaSuccess;
    if (!offsets) {   // single-curve entry point
        set_offsets_kernel<<<1, 1, 0, st>>>(own_off, n_total);
        offsets = own_off;
        g_ts.launches += 1;
    }
    g_ts.launches += 3;   // prep_curves, prep_periods, fold
    e = gpfc::launch_prep(times, flux, offsets, ncurves, t0v, t0_scalar, periods, nperiods, nbins,
                          s, st);
    if (e == cudaSuccess) {
        gpfc::FoldArgs a;
        a.u = s.u;
        a.q = s.q;
        a.rec = s.rec;
        a.tiles = s.tiles;
        a.meta = s.meta;
        a.rp = s.rp;
        a.periods = periods;
        a.ncurves = ncurves;
        a.nperiods = nperiods;
        a.nbins = nbins;
        a.out_sum = out_sum;
        a.out_count = out_count;
        a.out_norm = out_norm;
        a.n_min = 0;
        a.n_max = 0x7fffffff;
        cudaEvent_t e0 = nullptr, e1 = nullptr;
        if (g_ts.profiling && cudaEventCreate(&e0) == cudaSuccess &&
            cudaEventCreate(&e1) == cudaSuccess)
            cudaEventRecord(e0, st);
        e = gpfc::launch_fold(a, st);
        if (e0 && e1) {
            cudaEventRecord(e1, st);
            g_ts.ev.push_back(e0);
            g_ts.ev.push_back(e1);
        }
    }
    if (own) {
        cudaError_t e2 = cudaFreeAsync(base, st);
        if (e == cudaSuccess) e = e2;
    }
    if (e != cudaSuccess) return cuda_fail(e, "fold launch");
    return GPFC_OK;
}

}  // namespace

extern "C" {

const char *gpfc_version(void) { return "gpfc-b200 0.1 (sm_100a)"; }

const char *gpfc_last_error(void) { return g_ts.err; }

int gpfc_set_stream(void *cuda_stream)
{
    g_ts.stream = static_cast<cudaStream_t>(cuda_stream);
    return GPFC_OK;
}

size_t gpfc_workspace_bytes(int64_t ncurves, int64_t n_total, int64_t nperiods, int nbins)
{
    (void)nbins;
    if (ncurves < 0 || n_total < 0 || nperiods < 0) return 0;
    return scratch_bytes(ncurves, n_total, nperiods);
}

int gpfc_set_workspace(void *dev_ptr, size_t bytes)
{
    if (!dev_ptr && bytes) return fail(GPFC_ERR_INVALID_ARG, "workspace NULL with non-zero size%s");
    g_ts.ws = dev_ptr;
    g_ts.ws_bytes = dev_ptr ? bytes : 0;
    return GPFC_OK;
}

double gpfc_n_sample(double n_o, double t_window, double l_width)
{
    return n_o * t_window / l_width;
}

static int grid_args_ok(double pmin, double pmax, int64_t nperiods)
{
    return nperiods >= 0 && pmin > 0.0 && pmax >= pmin && std::isfinite(pmax) &&
           std::isfinite(pmin);
}

int gpfc_make_period_grid(double pmin, double pmax, int64_t nperiods, int mode_flags,
                          double *periods_out)
{
    if (!grid_args_ok(pmin, pmax, nperiods))
        return fail(GPFC_ERR_INVALID_ARG, "period grid: need 0 < pmin <= pmax, nperiods >= 0%s");
    if (nperiods == 0) return GPFC_OK;
    if (!periods_out) return fail(GPFC_ERR_INVALID_ARG, "periods_out is NULL%s");
    cudaError_t e = gpfc::launch_grid(pmin, pmax, nperiods, mode_flags, periods_out, g_ts.stream);
    if (e != cudaSuccess) return cuda_fail(e, "grid launch");
    g_ts.launches += 1;
    return GPFC_OK;
}

int gpfc_fold(const double *times, const float *flux, int64_t n, const double *periods,
              int64_t nperiods, int nbins, double t0, float *out_sum, uint32_t *out_count)
{
    if (n < 0) return fail(GPFC_ERR_INVALID_ARG, "negative size%s");
    return fold_device(times, flux, nullptr, 1, n, periods, nperiods, nbins, nullptr, t0, out_sum,
                       out_count, nullptr);
}

int gpfc_normalize(const float *sum, const uint32_t *count, int64_t nprofiles, int nbins,
                   float *out_norm)
{
    if (nprofiles < 0) return fail(GPFC_ERR_INVALID_ARG, "negative size%s");
    if (nbins < 1 || nbins > GPFC_MAX_NBINS)
        return fail(GPFC_ERR_UNSUPPORTED, "nbins must be in [1, 4096]%s");
    if (nprofiles == 0) return GPFC_OK;
    if (!sum || !count || !out_norm) return fail(GPFC_ERR_INVALID_ARG, "NULL pointer%s");
    cudaError_t e = gpfc::launch_normalize(sum, count, nprofiles, nbins, out_norm, g_ts.stream);
    if (e != cudaSuccess) return cuda_fail(e, "normalize launch");
    g_ts.launches += 1;
    return GPFC_OK;
}

int gpfc_merge_equal_count(const float *sum, const uint32_t *count, int64_t nprofiles, int nb1,
                           int nb2, float *out_mean, float *out_norm)
{
    if (nprofiles < 0) return fail(GPFC_ERR_INVALID_ARG, "negative size%s");
    if (nb1 < 1 || nb1 > GPFC_MAX_NBINS || nb2 < 1 || nb2 > GPFC_MAX_NBINS)
        return fail(GPFC_ERR_UNSUPPORTED, "nb1 and nb2 must be in [1, 4096]%s");
    if (nprofiles == 0) return GPFC_OK;
    if (!sum || !count || (!out_mean && !out_norm)) return fail(GPFC_ERR_INVALID_ARG, "NULL pointer%s");
    cudaError_t e = gpfc::launch_merge(sum, count, nprofiles, nb1, nb2, out_mean, out_norm,
                                       g_ts.stream);
    if (e != cudaSuccess) return cuda_fail(e, "merge launch");
    g_ts.launches += 1;
    return GPFC_OK;
}

int gpfc_fold_batch(const double *times, const float *flux, const int64_t *offsets,
                    int64_t ncurves, int64_t n_total, const double *periods, int64_t nperiods,
                    int nbins, const double *t0, float *out_sum, uint32_t *out_count,
                    float *out_norm)
{
    if (ncurves > 0 && !offsets) return fail(GPFC_ERR_INVALID_ARG, "offsets is NULL%s");
    return fold_device(times, flux, offsets, ncurves, n_total, periods, nperiods, nbins, t0, 0.0,
                       out_sum, out_count, out_norm);
}

int gpfc_make_period_grid_host(double pmin, double pmax, int64_t nperiods, int mode_flags,
                               double *periods_out)
{
    if (!grid_args_ok(pmin, pmax, nperiods))
        return fail(GPFC_ERR_INVALID_ARG, "period grid: need 0 < pmin <= pmax, nperiods >= 0%s");
    if (nperiods == 0) return GPFC_OK;
    if (!periods_out) return fail(GPFC_ERR_INVALID_ARG, "periods_out is NULL%s");
    cudaStream_t st = g_ts.stream;
    double *d = nullptr;
    cudaError_t e = cudaMallocAsync(reinterpret_cast<void **>(&d), (size_t)nperiods * 8, st);
    if (e != cudaSuccess) return cuda_fail(e, "grid alloc");
    e = gpfc::launch_grid(pmin, pmax, nperiods, mode_flags, d, st);
    g_ts.launches += 1;
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(periods_out, d, (size_t)nperiods * 8, cudaMemcpyDeviceToHost, st);
    cudaFreeAsync(d, st);
    cudaError_t e2 = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = e2;
    if (e != cudaSuccess) return cuda_fail(e, "grid host path");
    return GPFC_OK;
}

int gpfc_fold_batch_host(const double *times, const float *flux, const int64_t *offsets,
                         int64_t ncurves, int64_t n_total, const double *periods,
                         int64_t nperiods, int nbins, const double *t0, float *out_sum,
                         uint32_t *out_count, float *out_norm)
{
    // Streaming host path: inputs go up once; the curves are folded in chunks whose outputs
    // land in one of two device slabs, and the device->host copy of chunk k (copy stream)
    // overlaps the fold of chunk k+1 (the caller's stream).
    if (ncurves < 0 || nperiods < 0 || n_total < 0)
        return fail(GPFC_ERR_INVALID_ARG, "negative size%s");
    if (nbins < 1 || nbins > GPFC_MAX_NBINS)
        return fail(GPFC_ERR_UNSUPPORTED, "nbins must be in [1, 4096]%s");
    if (ncurves == 0 || nperiods == 0) return GPFC_OK;
    if (!offsets || !periods || (n_total > 0 && (!times || !flux)))
        return fail(GPFC_ERR_INVALID_ARG, "NULL pointer%s");
    for (int64_t c = 0; c < ncurves; ++c)
        if (offsets[c + 1] < offsets[c] || offsets[c] < 0 || offsets[c + 1] > n_total)
            return fail(GPFC_ERR_INVALID_ARG, "offsets must be non-decreasing within [0, n_total]%s");
    cudaStream_t st = g_ts.stream;
    const int nout = (out_sum ? 1 : 0) + (out_count ? 1 : 0) + (out_norm ? 1 : 0);
    const size_t row = (size_t)nperiods * (size_t)nbins;      // elements per curve and array
    // chunk: about 512 MB of output per slab, at least one curve
    int64_t chunk = nout ? (int64_t)((size_t)(512u << 20) / (row * 4 * (size_t)nout)) : ncurves;
    if (chunk < 1) chunk = 1;
    if (chunk > ncurves) chunk = ncurves;
    const size_t b_t = align_up((size_t)n_total * 8), b_f = align_up((size_t)n_total * 4);
    const size_t b_o = align_up((size_t)(ncurves + 1) * 8), b_p = align_up((size_t)nperiods * 8);
    const size_t b_t0 = t0 ? align_up((size_t)ncurves * 8) : 0;
    const size_t b_arr = align_up((size_t)chunk * row * 4);
    const size_t total = b_t + b_f + b_o + b_p + b_t0 + 2 * (size_t)nout * b_arr + 256;
    char *base = nullptr;
    cudaError_t e = cudaMallocAsync(reinterpret_cast<void **>(&base), total, st);
    if (e != cudaSuccess) {
        cuda_fail(e, "device buffer allocation");
        return GPFC_ERR_WORKSPACE;
    }
    char *cur = base;
    double *d_t = reinterpret_cast<double *>(cur); cur += b_t;
    float *d_f = reinterpret_cast<float *>(cur); cur += b_f;
    int64_t *d_o = reinterpret_cast<int64_t *>(cur); cur += b_o;
    double *d_p = reinterpret_cast<double *>(cur); cur += b_p;
    double *d_t0 = nullptr;
    if (t0) { d_t0 = reinterpret_cast<double *>(cur); cur += b_t0; }
    char *slab[2][3] = {{nullptr, nullptr, nullptr}, {nullptr, nullptr, nullptr}};
    for (int s = 0; s < 2; ++s)
        for (int k = 0; k < 3; ++k) {
            const bool want = (k == 0 && out_sum) || (k == 1 && out_count) || (k == 2 && out_norm);
            if (want) { slab[s][k] = cur; cur += b_arr; }
        }

    cudaStream_t cs = nullptr;
    cudaEvent_t done[2] = {nullptr, nullptr}, freed[2] = {nullptr, nullptr};
    e = cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking);
    for (int s = 0; s < 2 && e == cudaSuccess; ++s) {
        e = cudaEventCreateWithFlags(&done[s], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&freed[s], cudaEventDisableTiming);
    }
    int rc = GPFC_OK;
    if (e == cudaSuccess && n_total > 0) {
        e = cudaMemcpyAsync(d_t, times, (size_t)n_total * 8, cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(d_f, flux, (size_t)n_total * 4, cudaMemcpyHostToDevice, st);
    }
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(d_o, offsets, (size_t)(ncurves + 1) * 8, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(d_p, periods, (size_t)nperiods * 8, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess && t0)
        e = cudaMemcpyAsync(d_t0, t0, (size_t)ncurves * 8, cudaMemcpyHostToDevice, st);
    int64_t k = 0;
    for (int64_t c0 = 0; c0 < ncurves && e == cudaSuccess && rc == GPFC_OK; c0 += chunk, ++k) {
        const int s = (int)(k & 1);
        const int64_t nc = (ncurves - c0 < chunk) ? ncurves - c0 : chunk;
        if (k >= 2) e = cudaStreamWaitEvent(st, freed[s], 0);     // slab s copied out
        if (e != cudaSuccess) break;
        // the prepass scratch covers the samples offsets[c0] .. offsets[c0 + nc]: pass the
        // whole arrays (offsets are absolute) and size the scratch by n_total
        rc = fold_device(d_t, d_f, d_o + c0, nc, n_total, d_p, nperiods, nbins,
                         d_t0 ? d_t0 + c0 : nullptr, 0.0,
                         reinterpret_cast<float *>(slab[s][0]),
                         reinterpret_cast<uint32_t *>(slab[s][1]),
                         reinterpret_cast<float *>(slab[s][2]));
        if (rc != GPFC_OK) break;
        e = cudaEventRecord(done[s], st);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(cs, done[s], 0);
        const size_t bytes = (size_t)nc * row * 4, off = (size_t)c0 * row;
        if (e == cudaSuccess && out_sum)
            e = cudaMemcpyAsync(out_sum + off, slab[s][0], bytes, cudaMemcpyDeviceToHost, cs);
        if (e == cudaSuccess && out_count)
            e = cudaMemcpyAsync(out_count + off, slab[s][1], bytes, cudaMemcpyDeviceToHost, cs);
        if (e == cudaSuccess && out_norm)
            e = cudaMemcpyAsync(out_norm + off, slab[s][2], bytes, cudaMemcpyDeviceToHost, cs);
        if (e == cudaSuccess) e = cudaEventRecord(freed[s], cs);
    }
    cudaError_t e2 = cs ? cudaStreamSynchronize(cs) : cudaSuccess;
    cudaError_t e3 = cudaStreamSynchronize(st);
    cudaFreeAsync(base, st);
    for (int s = 0; s < 2; ++s) {
        if (done[s]) cudaEventDestroy(done[s]);
        if (freed[s]) cudaEventDestroy(freed[s]);
    }
    if (cs) cudaStreamDestroy(cs);
    if (rc != GPFC_OK) return rc;
    if (e == cudaSuccess) e = e2;
    if (e == cudaSuccess) e = e3;
    if (e != cudaSuccess) return cuda_fail(e, "host-buffer fold");
    return GPFC_OK;
}

int gpfc_profile(int enable)
{
    for (cudaEvent_t ev : g_ts.ev) cudaEventDestroy(ev);
    g_ts.ev.clear();
    g_ts.launches = 0;
    g_ts.profiling = enable != 0;
    return GPFC_OK;
}

int gpfc_profile_read(double *fold_kernel_ms, int64_t *fold_launches, int64_t *kernel_launches)
{
    double total = 0.0;
    for (size_t i = 0; i + 1 < g_ts.ev.size(); i += 2) {
        cudaError_t e = cudaEventSynchronize(g_ts.ev[i + 1]);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, g_ts.ev[i], g_ts.ev[i + 1]);
        if (e != cudaSuccess) return cuda_fail(e, "gpfc_profile_read");
        total += ms;
    }
    if (fold_kernel_ms) *fold_kernel_ms = total;
    if (fold_launches) *fold_launches = (int64_t)(g_ts.ev.size() / 2);
    if (kernel_launches) *kernel_launches = g_ts.launches;
    return GPFC_OK;
}

int gpfc_measure_peaks(double *out)
{
    if (!out) return fail(GPFC_ERR_INVALID_ARG, "out is NULL%s");
    cudaError_t e = gpfc::measure_peaks(out, g_ts.stream);
    if (e != cudaSuccess) return cuda_fail(e, "measure_peaks");
    return GPFC_OK;
}

}  // extern "C"
