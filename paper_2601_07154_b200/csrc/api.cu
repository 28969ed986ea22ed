// Status strings, error buffer, device check and window arithmetic of the mf C ABI (include/mf.h).
#include "common.h"

#include <atomic>
#include <cstring>

namespace mf {

char* error_buffer() {
    static thread_local char buf[512] = "";
    return buf;
}

mf_status fail(mf_status s, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(error_buffer(), 512, fmt, ap);
    va_end(ap);
    return s;
}

bool& validate_only() {
    static thread_local bool flag = false;
    return flag;
}

// SM count of every device that passed the check (0 = not checked yet).  The library is called from several host
// threads at once (bench.py's end-to-end path), so the cache is one atomic per device, written after the check.
constexpr int kMaxDevices = 64;
static std::atomic<int> g_sm_count[kMaxDevices];

mf_status require_sm100() {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(MF_ERR_CUDA, "cudaGetDevice failed: %s", cudaGetErrorString(e));
    if (dev >= 0 && dev < kMaxDevices && g_sm_count[dev].load(std::memory_order_acquire) > 0) return MF_OK;
    int major = 0, minor = 0, sms = 0;
    if ((e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev)) != cudaSuccess ||
        (e = cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev)) != cudaSuccess ||
        (e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess)
        return fail(MF_ERR_CUDA, "cudaDeviceGetAttribute failed: %s", cudaGetErrorString(e));
    if (major != 10)
        return fail(MF_ERR_CUDA, "device %d is sm_%d%d; this library is built for sm_100a only (no fallback)", dev, major, minor);
    if (dev >= 0 && dev < kMaxDevices) g_sm_count[dev].store(sms > 0 ? sms : 148, std::memory_order_release);
    return MF_OK;
}

int sm_count() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return 148;
    const int n = g_sm_count[dev].load(std::memory_order_acquire);
    return n > 0 ? n : 148;
}

}  // namespace mf

extern "C" {

const char* mf_status_string(mf_status s) {
    switch (s) {
        case MF_OK: return "MF_OK";
        case MF_ERR_INVALID_ARG: return "MF_ERR_INVALID_ARG";
        case MF_ERR_UNSUPPORTED: return "MF_ERR_UNSUPPORTED";
        case MF_ERR_ALIGNMENT: return "MF_ERR_ALIGNMENT";
        case MF_ERR_WORKSPACE: return "MF_ERR_WORKSPACE";
        case MF_ERR_CUDA: return "MF_ERR_CUDA";
    }
    return "MF_ERR_UNKNOWN";
}

const char* mf_last_error(void) { return mf::error_buffer(); }

int mf_version(void) { return 200; }     // 0.2.0: round 2 (mf_window_attention_noalloc, score-bound path)

// P:70; tail window starts at num_frames - W (reading B6 in DESIGN.md).
int mf_num_windows(int num_frames, int W, int stride) {
    if (W < 1 || num_frames < W || stride < 1 || stride >= W) return -1;
    return (num_frames - W + stride - 1) / stride + 1;
}

int mf_window_start(int num_frames, int W, int stride, int n) {
    int nw = mf_num_windows(num_frames, W, stride);
    if (nw < 0 || n < 0 || n >= nw) return -1;
    long long s = static_cast<long long>(n) * stride;
    return s < num_frames - W ? static_cast<int>(s) : num_frames - W;
}

}  // extern "C"
