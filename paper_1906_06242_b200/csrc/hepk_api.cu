// hepk_api.cu — error reporting, device queries, version.
#include <stdarg.h>

#include <atomic>
#include <mutex>

#include "hepk_common.cuh"

namespace hepk {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

int32_t cuda_fail(cudaError_t e, const char* what)
{
    set_error("CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
    return HEPK_ERR_CUDA;
}

struct DevInfo { int sms = 0; int smem_optin = 0; };
static DevInfo g_dev[64];

static DevInfo& devinfo()
{
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64) dev = 0;
    DevInfo& d = g_dev[dev];
    if (d.sms == 0) {
        cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev);
        cudaDeviceGetAttribute(&d.smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        if (d.sms <= 0) d.sms = 148;
        if (d.smem_optin <= 0) d.smem_optin = 227 * 1024;
    }
    return d;
}

// ---- optional device-side timing of the dominant kernel (hepk_profile_begin / hepk_profile_end) -------------
static std::atomic<long long> g_launches{0};
void count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }

static std::mutex g_prof_mutex;      // the event table is shared by every thread that launches the chain
static const int PROF_MAX = 4096;
static bool g_prof_on = false;
static int g_prof_n = 0;
static cudaEvent_t g_prof_ev[PROF_MAX][2];
static bool g_prof_created = false;

void profile_mark(cudaStream_t st, int which)
{
    std::lock_guard<std::mutex> lock(g_prof_mutex);
    if (!g_prof_on || g_prof_n >= PROF_MAX) return;
    cudaEventRecord(g_prof_ev[g_prof_n][which], st);
    if (which == 1) g_prof_n++;
}

int sm_count() { return devinfo().sms; }
int max_smem_optin() { return devinfo().smem_optin; }

}  // namespace hepk

extern "C" int64_t hepk_kernel_launches(void) { return hepk::g_launches.load(std::memory_order_relaxed); }

extern "C" int32_t hepk_profile_begin(void)
{
    using namespace hepk;
    std::lock_guard<std::mutex> lock(g_prof_mutex);
    if (!g_prof_created) {
        for (int i = 0; i < PROF_MAX; ++i)
            for (int k = 0; k < 2; ++k) HEPK_CUDA_TRY(cudaEventCreate(&g_prof_ev[i][k]));
        g_prof_created = true;
    }
    g_prof_n = 0;
    g_prof_on = true;
    return HEPK_OK;
}

extern "C" int32_t hepk_profile_end(double* total_ms, int32_t* n_launches)
{
    using namespace hepk;
    std::lock_guard<std::mutex> lock(g_prof_mutex);
    g_prof_on = false;
    double tot = 0.0;
    for (int i = 0; i < g_prof_n; ++i) {
        float ms = 0.f;
        HEPK_CUDA_TRY(cudaEventSynchronize(g_prof_ev[i][1]));
        HEPK_CUDA_TRY(cudaEventElapsedTime(&ms, g_prof_ev[i][0], g_prof_ev[i][1]));
        tot += ms;
    }
    if (total_ms) *total_ms = tot;
    if (n_launches) *n_launches = g_prof_n;
    return HEPK_OK;
}

extern "C" int32_t hepk_version(void) { return 100; }
extern "C" const char* hepk_last_error(void) { return hepk::g_err; }
