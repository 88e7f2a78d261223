// api.cu — host-side plumbing of libgbfg: status strings, device check, grid, launch counter.
#include <stdio.h>
#include <string.h>

#include <vector>

#include "gbfg_common.cuh"

namespace gbfg {

static thread_local char g_cuda_error[512] = "";
static thread_local int64_t g_launches = 0;

int set_cuda_error(cudaError_t e, const char *where)
{
    snprintf(g_cuda_error, sizeof(g_cuda_error), "%s: %s (%s)", where, cudaGetErrorString(e), cudaGetErrorName(e));
    (void)cudaGetLastError();   // clear the sticky-less error state
    return GBFG_ERR_CUDA;
}

void count_launch(int n) { g_launches += n; }

// ---- per-kernel timing helper (measurement only; off by default)
struct TimedLaunch { cudaEvent_t a, b; int kid; };
static thread_local bool g_prof_on = false;
static thread_local std::vector<TimedLaunch> *g_prof = nullptr;   // event pairs, reused across reads
static thread_local size_t g_prof_used = 0;

LaunchTimer::LaunchTimer(int kernel_id, cudaStream_t stream) : slot(-1), st(stream)
{
    if (!g_prof_on) return;
    if (!g_prof) g_prof = new std::vector<TimedLaunch>();
    if (g_prof_used == g_prof->size()) {
        TimedLaunch t;
        if (cudaEventCreate(&t.a) != cudaSuccess || cudaEventCreate(&t.b) != cudaSuccess) { (void)cudaGetLastError(); return; }
        g_prof->push_back(t);
    }
    slot = (int)g_prof_used++;
    (*g_prof)[slot].kid = kernel_id;
    cudaEventRecord((*g_prof)[slot].a, st);
}

LaunchTimer::~LaunchTimer()
{
    if (slot >= 0) cudaEventRecord((*g_prof)[slot].b, st);
}

struct DevInfo { int ok; int status; int sms; };
static DevInfo g_dev[64];

static int probe_device(int *sms)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return set_cuda_error(e, "cudaGetDevice");
    if (dev < 0 || dev >= 64) return GBFG_ERR_ARCH;
    if (!g_dev[dev].ok) {
        int major = 0, n = 0;
        e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        if (e != cudaSuccess) return set_cuda_error(e, "cudaDeviceGetAttribute");
        e = cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return set_cuda_error(e, "cudaDeviceGetAttribute");
        g_dev[dev].status = (major == 10) ? GBFG_OK : GBFG_ERR_ARCH;
        g_dev[dev].sms = n;
        g_dev[dev].ok = 1;
    }
    if (sms) *sms = g_dev[dev].sms;
    return g_dev[dev].status;
}

int check_device() { return probe_device(nullptr); }

int sm_count()
{
    int n = 148;
    probe_device(&n);
    return n > 0 ? n : 148;
}

}  // namespace gbfg

using namespace gbfg;

extern "C" int gbfg_version(void) { return 100; /* 0.1.0 */ }

extern "C" const char *gbfg_strerror(int status)
{
    switch (status) {
    case GBFG_OK: return "ok";
    case GBFG_ERR_INVALID_ARG: return "invalid argument";
    case GBFG_ERR_WORKSPACE: return "workspace missing or too small";
    case GBFG_ERR_CUDA: return "CUDA runtime error (see gbfg_last_cuda_error)";
    case GBFG_ERR_ARCH: return "device is not compute capability 10.x (sm_100)";
    case GBFG_ERR_UNSUPPORTED: return "unsupported size or parameter (window > GBFG_MAX_WINDOW, n_cat > GBFG_MAX_CAT, alpha_gamma outside its stated range)";
    case GBFG_ERR_STATIC_LIMIT: return "the call needs more scratch than the library's static array holds (GBFG_STATIC_SCRATCH_BYTES): use the variant that takes a workspace";
    default: return "unknown status";
    }
}

extern "C" const char *gbfg_last_cuda_error(void) { return g_cuda_error; }

extern "C" int64_t gbfg_kernel_launch_count(void) { return g_launches; }

extern "C" int gbfg_profile_enable(int on)
{
    g_prof_on = on != 0;
    g_prof_used = 0;
    return GBFG_OK;
}

extern "C" int gbfg_profile_read(gbfg_kernel_time *out, int32_t n_out)
{
    if (!out || n_out < GBFG_K_COUNT) return GBFG_ERR_INVALID_ARG;
    for (int k = 0; k < GBFG_K_COUNT; ++k) { out[k].launches = 0; out[k].total_ms = 0.0; out[k].max_ms = 0.0; }
    for (size_t i = 0; i < g_prof_used; ++i) {
        TimedLaunch &t = (*g_prof)[i];
        GBFG_CUDA(cudaEventSynchronize(t.b));
        float ms = 0.f;
        GBFG_CUDA(cudaEventElapsedTime(&ms, t.a, t.b));
        out[t.kid].launches += 1;
        out[t.kid].total_ms += (double)ms;
        if ((double)ms > out[t.kid].max_ms) out[t.kid].max_ms = (double)ms;
    }
    g_prof_used = 0;
    return GBFG_OK;
}

extern "C" int gbfg_profile_timeline(gbfg_launch_time *out, int32_t cap, int32_t *n_written, int32_t *n_total)
{
    if (!out || cap < 0 || !n_written || !n_total) return GBFG_ERR_INVALID_ARG;
    *n_total = (int32_t)g_prof_used;
    *n_written = 0;
    for (size_t i = 0; i < g_prof_used && (int32_t)i < cap; ++i) {
        TimedLaunch &t = (*g_prof)[i];
        GBFG_CUDA(cudaEventSynchronize(t.b));
        float a_ms = 0.f, b_ms = 0.f;
        if (i) GBFG_CUDA(cudaEventElapsedTime(&a_ms, (*g_prof)[0].a, t.a));
        GBFG_CUDA(cudaEventElapsedTime(&b_ms, (*g_prof)[0].a, t.b));
        out[i].kernel = t.kid;
        out[i].start_ms = a_ms;
        out[i].end_ms = b_ms;
        *n_written = (int32_t)i + 1;
    }
    return GBFG_OK;
}

extern "C" int gbfg_grid_init(double f_min, double f_max, double t_obs, int32_t scale_log2, gbfg_grid *out)
{
    if (!out) return GBFG_ERR_INVALID_ARG;
    if (!(f_min > 0.0) || !(f_max > f_min) || !(t_obs > 0.0)) return GBFG_ERR_INVALID_ARG;
    if (!(f_max < 1e300) || !(t_obs < 1e300)) return GBFG_ERR_INVALID_ARG;
    if (scale_log2 < -1000 || scale_log2 > 0) return GBFG_ERR_INVALID_ARG;
    double nb = ceil((f_max - f_min) * t_obs);          // DESIGN.md R2
    if (!(nb >= 1.0) || !(nb < 2147483648.0)) return GBFG_ERR_INVALID_ARG;
    memset(out, 0, sizeof(*out));
    out->struct_size = (uint32_t)sizeof(gbfg_grid);
    out->scale_log2 = scale_log2;
    out->f_min = f_min; out->f_max = f_max; out->t_obs = t_obs;
    out->n_bins = (int64_t)nb;
    return GBFG_OK;
}
