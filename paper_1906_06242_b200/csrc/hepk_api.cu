// hepk_api.cu — error reporting, device queries, version.
#include <stdarg.h>

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

int sm_count() { return devinfo().sms; }
int max_smem_optin() { return devinfo().smem_optin; }

}  // namespace hepk

extern "C" int32_t hepk_version(void) { return 100; }
extern "C" const char* hepk_last_error(void) { return hepk::g_err; }
