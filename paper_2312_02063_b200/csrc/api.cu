// C ABI of libgpfc.so (include/gpfc.h): argument validation, scratch carving,
// launches.  No compute happens on the host and there is no CPU fallback.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "common.cuh"

// ---- gpfc_fold_noalloc: the scratch of one single-curve fold, held by the library itself.
// Every GPU that loads the library holds these GPFC_NOALLOC_BYTES (4.8 MB) until exit.  In host
// code the array's name is only a stand-in for the symbol: the device address comes from
// cudaGetSymbolAddress (noalloc_scratch_ptr below), once per device with that device current.
constexpr int64_t GPFC_NOALLOC_SAMPLES = GPFC_NOALLOC_MAX_SAMPLES;
constexpr int64_t GPFC_NOALLOC_PERIODS = GPFC_NOALLOC_MAX_PERIODS;
constexpr size_t noalloc_up(size_t x) { return (x + 255) & ~(size_t)255; }
constexpr size_t GPFC_NOALLOC_BYTES =          // the terms of scratch_bytes(1, n, np, 0) below
    noalloc_up((size_t)GPFC_NOALLOC_SAMPLES * sizeof(double)) +
    noalloc_up((size_t)GPFC_NOALLOC_SAMPLES * sizeof(int)) +
    noalloc_up(((size_t)GPFC_NOALLOC_SAMPLES + 3) * sizeof(int2)) +
    noalloc_up(((size_t)GPFC_NOALLOC_SAMPLES / gpfc::GPFC_TILE + 2) * sizeof(gpfc::TileInfo)) +
    noalloc_up(sizeof(gpfc::CurveMeta)) +
    noalloc_up((size_t)GPFC_NOALLOC_PERIODS * sizeof(double)) +
    noalloc_up(2 * sizeof(int64_t)) + noalloc_up(gpfc::PREP_PART_BYTES) + 256;
static __device__ __align__(256) unsigned char gpfc_noalloc_scratch[GPFC_NOALLOC_BYTES];

namespace {

struct ThreadState {
    cudaStream_t stream = nullptr;
    void *ws = nullptr;
    size_t ws_bytes = 0;
    char err[512] = "";
    // gpfc_profile: CUDA-event pairs around every fold-kernel launch + launch counters
    bool profiling = false;
    long long launches = 0;           // kernels of this library launched by this thread
    long long generic_launches = 0;   // ... of which fold_generic_kernel (nbins > 256, not a power of two)
    long long unfused_two_tier = 0;   // gpfc_fold_two_tier calls that took fold + merge kernels
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

// ---- per-device state (kernel attributes are per device; so is the SM count)
constexpr int MAX_DEVICES = 64;
__device__ unsigned long long g_dev_stats[4];

struct DeviceSlot {
    bool ready = false;
    gpfc::DeviceInfo info{};
};
DeviceSlot g_dev[MAX_DEVICES];
std::mutex g_dev_mutex;

}  // namespace

namespace gpfc {

cudaError_t device_info(const DeviceInfo **out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    DeviceSlot &s = g_dev[dev];
    if (!s.ready) {
        int n = 0;
        e = cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        if (n <= 0) return cudaErrorInvalidDevice;
        // opt-in dynamic shared memory of every kernel that needs more than 48 KB; none of
        // these calls touches a stream
        e = fold_lp_init_device();
        if (e == cudaSuccess) e = fold_pk_init_device();
        if (e == cudaSuccess) e = merge_init_device();
        void *p = nullptr;
        if (e == cudaSuccess) e = cudaGetSymbolAddress(&p, g_dev_stats);
        if (e != cudaSuccess) return e;
        s.info.num_sms = n;
        s.info.stats = static_cast<unsigned long long *>(p);
        s.ready = true;
    }
    *out = &s.info;
    return cudaSuccess;
}

void note_launch(int n) { g_ts.launches += n; }

}  // namespace gpfc

namespace {

size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

// scratch of one fold call; `side` > 0 adds the count overflow area of fold_pk.cu
size_t scratch_bytes(int64_t ncurves, int64_t n_total, int64_t nperiods, size_t side)
{
    size_t b = 0;
    b += align_up((size_t)n_total * sizeof(double));
    b += align_up((size_t)n_total * sizeof(int));
    b += align_up(((size_t)n_total + (size_t)ncurves + 2) * sizeof(int2));
    b += align_up(((size_t)n_total / gpfc::GPFC_TILE + (size_t)ncurves + 1) * sizeof(gpfc::TileInfo));
    b += align_up((size_t)ncurves * sizeof(gpfc::CurveMeta));
    b += align_up((size_t)nperiods * sizeof(double));
    b += align_up(2 * sizeof(int64_t));   // offsets of the single-curve call
    b += align_up(gpfc::PREP_PART_BYTES);
    b += align_up(side);
    return b + 256;
}

// curves longer than the flush interval of fold_pk.cu need its 32-bit count overflow area;
// the curve lengths live on the device, so n_total is the bound the host can test
size_t side_bytes_for(int64_t n_total, int nbins, int sms)
{
    if (!gpfc::fold_pk_handles(nbins) || n_total <= gpfc::fold_pk_flush_samples()) return 0;
    return gpfc::fold_pk_side_bytes(sms);
}

__global__ void set_offsets_kernel(int64_t *o, int64_t n)
{
    o[0] = 0;
    o[1] = n;
}

struct FoldOut {
    float *sum = nullptr;
    uint32_t *count = nullptr;
    float *norm = nullptr;
    int nb2 = 0;                 // > 0: fused equal-count merge
    float *mean2 = nullptr;
    float *norm2 = nullptr;
    double *center_out = nullptr;   // FoldArgs::center_out: centred sums, the center per curve
};

// The device path shared by every fold entry point.
int fold_device(const double *times, const float *flux, const int64_t *offsets, int64_t ncurves,
                int64_t n_total, const double *periods, int64_t nperiods, int nbins,
                const double *t0v, double t0_scalar, const FoldOut &o)
{
    if (ncurves < 0 || nperiods < 0 || n_total < 0)
        return fail(GPFC_ERR_INVALID_ARG, "negative size%s");
    if (nbins < 1 || nbins > GPFC_MAX_NBINS)
        return fail(GPFC_ERR_UNSUPPORTED, "nbins must be in [1, 4096]%s");
    if (ncurves == 0 || nperiods == 0) return GPFC_OK;
    if (!periods) return fail(GPFC_ERR_INVALID_ARG, "periods is NULL%s");
    if (n_total > 0 && (!times || !flux)) return fail(GPFC_ERR_INVALID_ARG, "times/flux is NULL%s");
    if (o.nb2 == 0 && !o.sum && !o.count && !o.norm) return GPFC_OK;
    if (o.nb2 > 0 && !o.mean2 && !o.norm2) return GPFC_OK;

    const gpfc::DeviceInfo *di = nullptr;
    cudaError_t e = gpfc::device_info(&di);
    if (e != cudaSuccess) return cuda_fail(e, "device initialisation");
    cudaStream_t st = g_ts.stream;
    const size_t side = side_bytes_for(n_total, nbins, di->num_sms);
    size_t need = scratch_bytes(ncurves, n_total, nperiods, side);
    char *base = nullptr;
    bool own = false;
    if (g_ts.ws && g_ts.ws_bytes >= need) {
        base = static_cast<char *>(g_ts.ws);
    } else {
        void *p = nullptr;
        e = cudaMallocAsync(&p, need, st);
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
    cur += align_up(2 * sizeof(int64_t));
    s.part = reinterpret_cast<double *>(cur);
    cur += align_up(gpfc::PREP_PART_BYTES);
    unsigned *side_p = side ? reinterpret_cast<unsigned *>(cur) : nullptr;

    if (!offsets) {   // single-curve entry point
        set_offsets_kernel<<<1, 1, 0, st>>>(own_off, n_total);
        gpfc::note_launch();
        offsets = own_off;
    }
    e = gpfc::launch_prep(times, flux, offsets, ncurves, t0v, t0_scalar, periods, nperiods,
                          gpfc::fold_rows(nbins), s, n_total, di->num_sms, st);
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
        a.out_sum = o.sum;
        a.out_count = o.count;
        a.out_norm = o.norm;
        a.vec_ok = ((reinterpret_cast<uintptr_t>(o.sum) | reinterpret_cast<uintptr_t>(o.count) |
                     reinterpret_cast<uintptr_t>(o.norm)) & 15) == 0;
        a.nb2 = o.nb2;
        a.out_mean2 = o.mean2;
        a.out_norm2 = o.norm2;
        a.side = side_p;
        a.center_out = o.center_out;
        a.stats = di->stats;
        if (!gpfc::fold_lp_handles(nbins) && !gpfc::fold_pk_handles(nbins)) g_ts.generic_launches += 1;
        cudaEvent_t e0 = nullptr, e1 = nullptr;
        if (g_ts.profiling) {
            if (cudaEventCreate(&e0) == cudaSuccess && cudaEventCreate(&e1) != cudaSuccess) {
                cudaEventDestroy(e0);
                e0 = nullptr;
            }
            if (e0 && e1) cudaEventRecord(e0, st);
        }
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

int check_bins(int nb)
{
    if (nb < 1 || nb > GPFC_MAX_NBINS) return fail(GPFC_ERR_UNSUPPORTED, "bin counts must be in [1, 4096]%s");
    return GPFC_OK;
}

// Device address of gpfc_noalloc_scratch on the current device: asked for once per device, with
// that device current (a symbol has one address per device); no allocation.
void *g_noalloc_ptr[MAX_DEVICES];
std::mutex g_noalloc_mutex;

cudaError_t noalloc_scratch_ptr(void **out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, gpfc_noalloc_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_noalloc_ptr[dev] = p;
    }
    *out = g_noalloc_ptr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" {

const char *gpfc_version(void) { return "gpfc-b200 0.2 (sm_100a)"; }

const char *gpfc_last_error(void) { return g_ts.err; }

int gpfc_init(void)
{
    const gpfc::DeviceInfo *di = nullptr;
    cudaError_t e = gpfc::device_info(&di);
    if (e != cudaSuccess) return cuda_fail(e, "gpfc_init");
    return GPFC_OK;
}

int gpfc_set_stream(void *cuda_stream)
{
    g_ts.stream = static_cast<cudaStream_t>(cuda_stream);
    return GPFC_OK;
}

size_t gpfc_workspace_bytes(int64_t ncurves, int64_t n_total, int64_t nperiods, int nbins)
{
    if (ncurves < 0 || n_total < 0 || nperiods < 0) return 0;
    // the count overflow area is sized for the largest SM count of the family (no device query:
    // this call works without a GPU)
    return scratch_bytes(ncurves, n_total, nperiods, side_bytes_for(n_total, nbins, 160));
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
    return GPFC_OK;
}

int gpfc_lc_params_default(gpfc_lc_params *prm)
{
    if (!prm) return fail(GPFC_ERR_INVALID_ARG, "prm is NULL%s");
    std::memset(prm, 0, sizeof(*prm));
    prm->period_lo = 0.3;          // Table 2
    prm->period_hi = 1.0;
    prm->duration_lo = 0.03;
    prm->duration_hi = 0.09;
    prm->ratio_lo = 0.04;
    prm->ratio_hi = 0.12;
    prm->sigma_lo = 0.0001;
    prm->sigma_hi = 0.0005;
    prm->snr_lo = 6.0;
    prm->snr_hi = 10.0;
    prm->transit_fraction = 0.5;   // as many transit as non-transit samples
    prm->cadence = 0.020433;       // Kepler long cadence (R16)
    prm->t_start = 0.0;
    return GPFC_OK;
}

int gpfc_make_light_curves(uint64_t seed, int64_t ncurves, int64_t n, const gpfc_lc_params *prm,
                           double *times, float *flux, int64_t *offsets, double *params_out)
{
    if (ncurves < 0 || n < 0) return fail(GPFC_ERR_INVALID_ARG, "negative size%s");
    if (ncurves > 4294967295ll || n > 4294967295ll)
        return fail(GPFC_ERR_INVALID_ARG, "ncurves and n must be below 2^32%s");
    if (!prm) return fail(GPFC_ERR_INVALID_ARG, "prm is NULL%s");
    if (!(prm->period_lo > 0.0) || !(prm->period_hi >= prm->period_lo) || !(prm->duration_lo > 0.0) ||
        !(prm->duration_hi >= prm->duration_lo) || !(prm->ratio_lo > 0.0) ||
        !(prm->ratio_hi >= prm->ratio_lo) || !(prm->sigma_lo >= 0.0) ||
        !(prm->sigma_hi >= prm->sigma_lo) || !(prm->snr_hi >= prm->snr_lo) || !(prm->cadence > 0.0) ||
        !std::isfinite(prm->period_hi) || !std::isfinite(prm->duration_hi) ||
        !std::isfinite(prm->ratio_hi) || !std::isfinite(prm->sigma_hi) || !std::isfinite(prm->snr_lo) ||
        !std::isfinite(prm->snr_hi) || !std::isfinite(prm->cadence) || !std::isfinite(prm->t_start) ||
        !std::isfinite(prm->transit_fraction))
        return fail(GPFC_ERR_INVALID_ARG, "light-curve parameters: empty, reversed or non-finite range%s");
    if (ncurves == 0) return GPFC_OK;
    if (n > 0 && !flux) return fail(GPFC_ERR_INVALID_ARG, "flux is NULL%s");
    const gpfc::DeviceInfo *di = nullptr;
    cudaError_t e = gpfc::device_info(&di);
    if (e != cudaSuccess) return cuda_fail(e, "device initialisation");
    cudaStream_t st = g_ts.stream;
    const size_t need = gpfc::simulate_scratch_bytes(ncurves) + 256;
    void *scratch = nullptr;
    bool own = false;
    if (g_ts.ws && g_ts.ws_bytes >= need) {
        scratch = reinterpret_cast<void *>(align_up(reinterpret_cast<size_t>(g_ts.ws)));
    } else {
        e = cudaMallocAsync(&scratch, need, st);
        if (e != cudaSuccess) {
            cuda_fail(e, "scratch allocation");
            return GPFC_ERR_WORKSPACE;
        }
        own = true;
    }
    e = gpfc::launch_simulate(seed, ncurves, n, *prm, times, flux, reinterpret_cast<long long *>(offsets),
                              params_out, scratch, di->num_sms, st);
    if (own) cudaFreeAsync(scratch, st);
    if (e != cudaSuccess) return cuda_fail(e, "light-curve generator launch");
    return GPFC_OK;
}

int gpfc_fold(const double *times, const float *flux, int64_t n, const double *periods,
              int64_t nperiods, int nbins, double t0, float *out_sum, uint32_t *out_count)
{
    if (n < 0) return fail(GPFC_ERR_INVALID_ARG, "negative size%s");
    FoldOut o;
    o.sum = out_sum;
    o.count = out_count;
    return fold_device(times, flux, nullptr, 1, n, periods, nperiods, nbins, nullptr, t0, o);
}

int gpfc_fold_noalloc(const double *times, const float *flux, int64_t n, const double *periods,
                      int64_t nperiods, int nbins, double t0, float *out_sum,
                      uint32_t *out_count, float *out_norm)
{
    if (n < 0 || nperiods < 0) return fail(GPFC_ERR_INVALID_ARG, "negative size%s");
    if (n > GPFC_NOALLOC_SAMPLES)
        return fail(GPFC_ERR_UNSUPPORTED, "gpfc_fold_noalloc: more than GPFC_NOALLOC_MAX_SAMPLES "
                                          "(131072) samples%s");
    if (nperiods > GPFC_NOALLOC_PERIODS)
        return fail(GPFC_ERR_UNSUPPORTED, "gpfc_fold_noalloc: more than GPFC_NOALLOC_MAX_PERIODS "
                                          "(262144) periods%s");
    if (check_bins(nbins) != GPFC_OK) return GPFC_ERR_UNSUPPORTED;
    const gpfc::DeviceInfo *di = nullptr;
    cudaError_t e = gpfc::device_info(&di);          // kernel attributes, SM count: no allocation
    if (e != cudaSuccess) return cuda_fail(e, "device initialisation");
    if (side_bytes_for(n, nbins, di->num_sms) != 0)
        return fail(GPFC_ERR_UNSUPPORTED, "gpfc_fold_noalloc: nbins >= 512 takes at most 65408 samples "
                                          "(the count overflow area is not part of the static scratch)%s");
    if (scratch_bytes(1, n, nperiods, 0) > GPFC_NOALLOC_BYTES)
        return fail(GPFC_ERR_WORKSPACE, "gpfc_fold_noalloc: static scratch too small%s");
    void *scratch = nullptr;
    e = noalloc_scratch_ptr(&scratch);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(gpfc_noalloc_scratch)");
    // The fold itself is the library's one device path, run on the static scratch as its
    // workspace for this call (it allocates only when the workspace is too small, which was
    // ruled out above) and without the profiling events (cudaEventCreate) of gpfc_profile.
    void *const ws0 = g_ts.ws;
    const size_t wsb0 = g_ts.ws_bytes;
    const bool prof0 = g_ts.profiling;
    g_ts.ws = scratch;
    g_ts.ws_bytes = GPFC_NOALLOC_BYTES;
    g_ts.profiling = false;
    FoldOut o;
    o.sum = out_sum;
    o.count = out_count;
    o.norm = out_norm;
    const int rc = fold_device(times, flux, nullptr, 1, n, periods, nperiods, nbins, nullptr, t0, o);
    g_ts.ws = ws0;
    g_ts.ws_bytes = wsb0;
    g_ts.profiling = prof0;
    return rc;
}

int gpfc_normalize(const float *sum, const uint32_t *count, int64_t nprofiles, int nbins,
                   float *out_norm)
{
    if (nprofiles < 0) return fail(GPFC_ERR_INVALID_ARG, "negative size%s");
    if (check_bins(nbins) != GPFC_OK) return GPFC_ERR_UNSUPPORTED;
    if (nprofiles == 0) return GPFC_OK;
    if (!sum || !count || !out_norm) return fail(GPFC_ERR_INVALID_ARG, "NULL pointer%s");
    cudaError_t e = gpfc::launch_normalize(sum, count, nprofiles, nbins, out_norm, g_ts.stream);
    if (e != cudaSuccess) return cuda_fail(e, "normalize launch");
    return GPFC_OK;
}

int gpfc_merge_equal_count(const float *sum, const uint32_t *count, int64_t nprofiles, int nb1,
                           int nb2, float *out_mean, float *out_norm)
{
    if (nprofiles < 0) return fail(GPFC_ERR_INVALID_ARG, "negative size%s");
    if (check_bins(nb1) != GPFC_OK || check_bins(nb2) != GPFC_OK) return GPFC_ERR_UNSUPPORTED;
    if (nprofiles == 0) return GPFC_OK;
    if (!sum || !count || (!out_mean && !out_norm)) return fail(GPFC_ERR_INVALID_ARG, "NULL pointer%s");
    const gpfc::DeviceInfo *di = nullptr;
    cudaError_t e = gpfc::device_info(&di);
    if (e == cudaSuccess)
        e = gpfc::launch_merge(sum, count, nprofiles, nb1, nb2, out_mean, out_norm, nullptr, g_ts.stream);
    if (e != cudaSuccess) return cuda_fail(e, "merge launch");
    return GPFC_OK;
}

int gpfc_fold_batch(const double *times, const float *flux, const int64_t *offsets,
                    int64_t ncurves, int64_t n_total, const double *periods, int64_t nperiods,
                    int nbins, const double *t0, float *out_sum, uint32_t *out_count,
                    float *out_norm)
{
    if (ncurves > 0 && !offsets) return fail(GPFC_ERR_INVALID_ARG, "offsets is NULL%s");
    FoldOut o;
    o.sum = out_sum;
    o.count = out_count;
    o.norm = out_norm;
    return fold_device(times, flux, offsets, ncurves, n_total, periods, nperiods, nbins, t0, 0.0, o);
}

int gpfc_fold_two_tier(const double *times, const float *flux, const int64_t *offsets,
                       int64_t ncurves, int64_t n_total, const double *periods,
                       int64_t nperiods, int nb1, int nb2, const double *t0, float *out_mean,
                       float *out_norm)
{
    if (ncurves < 0 || nperiods < 0 || n_total < 0)
        return fail(GPFC_ERR_INVALID_ARG, "negative size%s");
    if (check_bins(nb1) != GPFC_OK || check_bins(nb2) != GPFC_OK) return GPFC_ERR_UNSUPPORTED;
    if (ncurves > 1 && !offsets) return fail(GPFC_ERR_INVALID_ARG, "offsets is NULL%s");
    if (ncurves == 0 || nperiods == 0 || (!out_mean && !out_norm)) return GPFC_OK;
    if (gpfc::fold_pk_can_merge(nb1, nb2)) {
        // fused: the nb1 intermediary bins never leave shared memory
        FoldOut o;
        o.nb2 = nb2;
        o.mean2 = out_mean;
        o.norm2 = out_norm;
        return fold_device(times, flux, offsets, ncurves, n_total, periods, nperiods, nb1, t0, 0.0, o);
    }
    // any other (nb1, nb2): fold into a temporary intermediary profile, chunk by chunk over the
    // period axis (<= 256 MB of sums + counts at a time), then the stand-alone merge kernel
    if (!periods) return fail(GPFC_ERR_INVALID_ARG, "periods is NULL%s");
    g_ts.unfused_two_tier += 1;
    cudaStream_t st = g_ts.stream;
    int64_t chunk = (int64_t)((size_t)(128u << 20) / ((size_t)nb1 * 4));
    if (chunk < 1) chunk = 1;
    if (chunk > nperiods) chunk = nperiods;
    char *tmp = nullptr;
    const size_t arr = align_up((size_t)chunk * (size_t)nb1 * 4);
    cudaError_t e = cudaMallocAsync(reinterpret_cast<void **>(&tmp), 2 * arr + 16 * (size_t)(ncurves + 1), st);
    if (e != cudaSuccess) {
        cuda_fail(e, "intermediary profile allocation");
        return GPFC_ERR_WORKSPACE;
    }
    float *t_sum = reinterpret_cast<float *>(tmp);
    uint32_t *t_cnt = reinterpret_cast<uint32_t *>(tmp + arr);
    // The intermediary sums are fp32: taken relative to the curve's center (written here by the
    // fold kernel, added back to the merged means by the merge kernel), so that an uncentred
    // relative flux near 1 does not cost 6e-8 per sum -- 1e-4 of a normalised profile's unit.
    double *t_center = reinterpret_cast<double *>(tmp + 2 * arr);
    int rc = GPFC_OK;
    for (int64_t c = 0; c < ncurves && rc == GPFC_OK; ++c) {
        for (int64_t j0 = 0; j0 < nperiods && rc == GPFC_OK; j0 += chunk) {
            const int64_t nj = (nperiods - j0 < chunk) ? nperiods - j0 : chunk;
            FoldOut o;
            o.sum = t_sum;
            o.count = t_cnt;
            o.center_out = t_center;
            rc = fold_device(times, flux, offsets ? offsets + c : nullptr, 1, n_total, periods + j0, nj,
                             nb1, t0 ? t0 + c : nullptr, 0.0, o);
            if (rc != GPFC_OK) break;
            e = gpfc::launch_merge(t_sum, t_cnt, nj, nb1, nb2,
                                   out_mean ? out_mean + ((size_t)c * nperiods + j0) * nb2 : nullptr,
                                   out_norm ? out_norm + ((size_t)c * nperiods + j0) * nb2 : nullptr,
                                   t_center, st);
            if (e != cudaSuccess) rc = cuda_fail(e, "merge launch");
        }
    }
    cudaFreeAsync(tmp, st);
    return rc;
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
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(periods_out, d, (size_t)nperiods * 8, cudaMemcpyDeviceToHost, st);
    cudaFreeAsync(d, st);
    cudaError_t e2 = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = e2;
    if (e != cudaSuccess) return cuda_fail(e, "grid host path");
    return GPFC_OK;
}

int gpfc_fold_stream(const double *times, const float *flux, const int64_t *offsets,
                     int64_t ncurves, int64_t n_total, const double *periods, int64_t nperiods,
                     int nbins, const double *t0, int outputs, size_t slab_bytes,
                     void *consumer_stream, gpfc_chunk_fn on_chunk, void *user)
{
    if (ncurves < 0 || nperiods < 0 || n_total < 0)
        return fail(GPFC_ERR_INVALID_ARG, "negative size%s");
    if (nbins < 1 || nbins > GPFC_MAX_NBINS)
        return fail(GPFC_ERR_UNSUPPORTED, "nbins must be in [1, 4096]%s");
    if (!on_chunk) return fail(GPFC_ERR_INVALID_ARG, "on_chunk is NULL%s");
    outputs &= GPFC_OUT_SUM | GPFC_OUT_COUNT | GPFC_OUT_NORM;
    if (!outputs) return fail(GPFC_ERR_INVALID_ARG, "outputs selects no array%s");
    if (ncurves == 0 || nperiods == 0) return GPFC_OK;
    if (!periods || (n_total > 0 && (!times || !flux)))
        return fail(GPFC_ERR_INVALID_ARG, "NULL pointer%s");
    if (!offsets && ncurves != 1)
        return fail(GPFC_ERR_INVALID_ARG, "offsets may be NULL only for a single curve%s");
    cudaStream_t st = g_ts.stream;
    cudaStream_t cs = consumer_stream ? static_cast<cudaStream_t>(consumer_stream) : st;
    const int nout = ((outputs & GPFC_OUT_SUM) ? 1 : 0) + ((outputs & GPFC_OUT_COUNT) ? 1 : 0) +
                     ((outputs & GPFC_OUT_NORM) ? 1 : 0);
    const size_t slab = slab_bytes ? slab_bytes : ((size_t)512 << 20) * (size_t)nout;
    const size_t prof = (size_t)nbins * 4 * (size_t)nout;     // bytes of one profile, all arrays
    const size_t row = prof * (size_t)nperiods;               // ... of one curve
    // a chunk is a run of whole curves, or (when one curve's profiles exceed the slab) a run of
    // periods of one curve; either way its profiles are contiguous in [curve][period][bin]
    int64_t cchunk = 1, pchunk = nperiods;
    if (row <= slab) {
        cchunk = (int64_t)(slab / row);
        if (cchunk > ncurves) cchunk = ncurves;
    } else {
        pchunk = (int64_t)(slab / prof);
        if (pchunk < 1) pchunk = 1;
    }
    const size_t b_arr = align_up((size_t)cchunk * (size_t)pchunk * (size_t)nbins * 4);
    char *base = nullptr;
    cudaError_t e = cudaMallocAsync(reinterpret_cast<void **>(&base), 2 * (size_t)nout * b_arr + 256, st);
    if (e != cudaSuccess) {
        cuda_fail(e, "output slab allocation");
        return GPFC_ERR_WORKSPACE;
    }
    char *cur = reinterpret_cast<char *>(align_up(reinterpret_cast<size_t>(base)));
    char *arr[2][3] = {{nullptr, nullptr, nullptr}, {nullptr, nullptr, nullptr}};
    for (int sl = 0; sl < 2; ++sl)
        for (int k = 0; k < 3; ++k)
            if (outputs & (1 << k)) {
                arr[sl][k] = cur;
                cur += b_arr;
            }
    // one scratch for all chunks (unless the caller registered a workspace that is large
    // enough): a stream-ordered allocation per chunk costs more than the prepass it serves
    const gpfc::DeviceInfo *di = nullptr;
    e = gpfc::device_info(&di);
    void *saved_ws = g_ts.ws, *own_ws = nullptr;
    const size_t saved_ws_bytes = g_ts.ws_bytes;
    if (e == cudaSuccess) {
        const size_t need = scratch_bytes(cchunk, n_total, pchunk, side_bytes_for(n_total, nbins, di->num_sms));
        if (!(g_ts.ws && g_ts.ws_bytes >= need) && cudaMallocAsync(&own_ws, need, st) == cudaSuccess) {
            g_ts.ws = own_ws;
            g_ts.ws_bytes = need;
        }
    }
    cudaEvent_t ready[2] = {nullptr, nullptr}, consumed[2] = {nullptr, nullptr};
    for (int sl = 0; sl < 2 && e == cudaSuccess; ++sl) {
        e = cudaEventCreateWithFlags(&ready[sl], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&consumed[sl], cudaEventDisableTiming);
    }
    int rc = GPFC_OK;
    int64_t k = 0;
    for (int64_t c0 = 0; c0 < ncurves && e == cudaSuccess && rc == GPFC_OK; c0 += cchunk) {
        const int64_t nc = (ncurves - c0 < cchunk) ? ncurves - c0 : cchunk;
        for (int64_t p0 = 0; p0 < nperiods && e == cudaSuccess && rc == GPFC_OK; p0 += pchunk, ++k) {
            const int64_t np = (nperiods - p0 < pchunk) ? nperiods - p0 : pchunk;
            const int sl = (int)(k & 1);
            if (k >= 2) e = cudaStreamWaitEvent(st, consumed[sl], 0);   // the consumer is done with it
            if (e != cudaSuccess) break;
            FoldOut o;
            o.sum = reinterpret_cast<float *>(arr[sl][0]);
            o.count = reinterpret_cast<uint32_t *>(arr[sl][1]);
            o.norm = reinterpret_cast<float *>(arr[sl][2]);
            // offsets are absolute: pass the whole sample arrays, the curves' slice of offsets
            rc = fold_device(times, flux, offsets ? offsets + c0 : nullptr, nc, n_total, periods + p0, np,
                             nbins, t0 ? t0 + c0 : nullptr, 0.0, o);
            if (rc != GPFC_OK) break;
            e = cudaEventRecord(ready[sl], st);
            if (e == cudaSuccess && cs != st) e = cudaStreamWaitEvent(cs, ready[sl], 0);
            if (e != cudaSuccess) break;
            gpfc_chunk ch;
            ch.curve0 = c0;
            ch.ncurves = nc;
            ch.period0 = p0;
            ch.nperiods = np;
            ch.nbins = nbins;
            ch.slot = sl;
            ch.sum = o.sum;
            ch.count = o.count;
            ch.norm = o.norm;
            ch.ready = ready[sl];
            if (on_chunk(&ch, cs, user) != 0) {
                rc = fail(GPFC_ERR_ABORTED, "the chunk consumer returned non-zero%s");
                break;
            }
            e = cudaEventRecord(consumed[sl], cs);
        }
    }
    // the slabs are released once the consumer stream is past its last chunk (stream-ordered,
    // the host does not wait)
    if (cs != st) {
        cudaEvent_t tail = nullptr;
        if (cudaEventCreateWithFlags(&tail, cudaEventDisableTiming) == cudaSuccess) {
            cudaEventRecord(tail, cs);
            cudaStreamWaitEvent(st, tail, 0);
            cudaEventDestroy(tail);
        }
    }
    cudaFreeAsync(base, st);
    if (own_ws) {
        cudaFreeAsync(own_ws, st);
        g_ts.ws = saved_ws;
        g_ts.ws_bytes = saved_ws_bytes;
    }
    for (int sl = 0; sl < 2; ++sl) {
        if (ready[sl]) cudaEventDestroy(ready[sl]);
        if (consumed[sl]) cudaEventDestroy(consumed[sl]);
    }
    if (rc != GPFC_OK) return rc;
    if (e != cudaSuccess) return cuda_fail(e, "gpfc_fold_stream");
    return GPFC_OK;
}

namespace {

// consumer of gpfc_fold_batch_host: device -> host copies of the chunk on the copy stream
struct HostSink {
    float *sum;
    uint32_t *count;
    float *norm;
    int64_t nperiods;
    cudaError_t err;
};

int host_sink_chunk(const gpfc_chunk *ch, void *stream, void *user)
{
    HostSink *hs = static_cast<HostSink *>(user);
    cudaStream_t cs = static_cast<cudaStream_t>(stream);
    const size_t off = ((size_t)ch->curve0 * (size_t)hs->nperiods + (size_t)ch->period0) * (size_t)ch->nbins;
    const size_t bytes = (size_t)ch->ncurves * (size_t)ch->nperiods * (size_t)ch->nbins * 4;
    cudaError_t e = cudaSuccess;
    if (hs->sum) e = cudaMemcpyAsync(hs->sum + off, ch->sum, bytes, cudaMemcpyDeviceToHost, cs);
    if (e == cudaSuccess && hs->count)
        e = cudaMemcpyAsync(hs->count + off, ch->count, bytes, cudaMemcpyDeviceToHost, cs);
    if (e == cudaSuccess && hs->norm)
        e = cudaMemcpyAsync(hs->norm + off, ch->norm, bytes, cudaMemcpyDeviceToHost, cs);
    hs->err = e;
    return e == cudaSuccess ? 0 : 1;
}

}  // namespace

int gpfc_fold_batch_host(const double *times, const float *flux, const int64_t *offsets,
                         int64_t ncurves, int64_t n_total, const double *periods,
                         int64_t nperiods, int nbins, const double *t0, float *out_sum,
                         uint32_t *out_count, float *out_norm)
{
    // Streaming host path: inputs go up once; gpfc_fold_stream folds the batch in chunks whose
    // outputs land in one of two device slabs, and the device->host copy of chunk k (copy
    // stream) overlaps the fold of chunk k+1 (the caller's stream).
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
    const int outputs = (out_sum ? GPFC_OUT_SUM : 0) | (out_count ? GPFC_OUT_COUNT : 0) |
                        (out_norm ? GPFC_OUT_NORM : 0);
    if (!outputs) return GPFC_OK;
    cudaStream_t st = g_ts.stream;
    const size_t b_t = align_up((size_t)n_total * 8), b_f = align_up((size_t)n_total * 4);
    const size_t b_o = align_up((size_t)(ncurves + 1) * 8), b_p = align_up((size_t)nperiods * 8);
    const size_t b_t0 = t0 ? align_up((size_t)ncurves * 8) : 0;
    char *base = nullptr;
    cudaError_t e = cudaMallocAsync(reinterpret_cast<void **>(&base), b_t + b_f + b_o + b_p + b_t0 + 256, st);
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
    cudaStream_t cs = nullptr;
    e = cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking);
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
    int rc = GPFC_OK;
    HostSink hs{out_sum, out_count, out_norm, nperiods, cudaSuccess};
    if (e == cudaSuccess)
        rc = gpfc_fold_stream(d_t, d_f, d_o, ncurves, n_total, d_p, nperiods, nbins, d_t0, outputs, 0, cs,
                              host_sink_chunk, &hs);
    cudaError_t e2 = cs ? cudaStreamSynchronize(cs) : cudaSuccess;
    cudaError_t e3 = cudaStreamSynchronize(st);
    cudaFreeAsync(base, st);
    if (cs) cudaStreamDestroy(cs);
    if (e == cudaSuccess && hs.err != cudaSuccess) e = hs.err;
    if (e == cudaSuccess && rc != GPFC_OK) return rc;
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
    g_ts.generic_launches = 0;
    g_ts.unfused_two_tier = 0;
    g_ts.profiling = enable != 0;
    const gpfc::DeviceInfo *di = nullptr;
    if (gpfc::device_info(&di) == cudaSuccess)
        cudaMemsetAsync(di->stats, 0, 4 * sizeof(unsigned long long), g_ts.stream);
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

int gpfc_path_counters(int64_t *out)
{
    if (!out) return fail(GPFC_ERR_INVALID_ARG, "out is NULL%s");
    out[0] = g_ts.generic_launches;
    out[1] = out[2] = out[4] = out[5] = out[6] = out[7] = 0;
    out[3] = g_ts.unfused_two_tier;
    const gpfc::DeviceInfo *di = nullptr;
    cudaError_t e = gpfc::device_info(&di);
    unsigned long long h[4] = {0, 0, 0, 0};
    if (e == cudaSuccess) e = cudaStreamSynchronize(g_ts.stream);
    if (e == cudaSuccess) e = cudaMemcpy(h, di->stats, sizeof(h), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(e, "gpfc_path_counters");
    out[1] = (int64_t)h[0];
    out[2] = (int64_t)h[1];
    out[4] = (int64_t)h[2];
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
