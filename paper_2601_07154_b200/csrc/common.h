// Shared host-side plumbing for the mf C-ABI library (error reporting, argument checks).
#pragma once
#include <cuda_runtime.h>
#include <cstdarg>
#include <cstdint>
#include <cstdio>

#include "../../include/mf.h"

namespace mf {

// Thread-local message returned by mf_last_error().
char* error_buffer();
mf_status fail(mf_status s, const char* fmt, ...);

// Checks that the current device is an sm_100 part; caches the answer per device (thread-safe).
mf_status require_sm100();
int sm_count();

// Thread-local "validate only" switch.  While it is set, every device entry point runs its complete argument / shape /
// device validation and returns MF_OK just before its first enqueue.  The *_host entry points use it to validate the
// whole chain of calls they are about to make BEFORE they allocate or copy anything ("on any error nothing has been
// enqueued", include/mf.h).
bool& validate_only();
struct ValidateOnlyScope {
    ValidateOnlyScope() { validate_only() = true; }
    ~ValidateOnlyScope() { validate_only() = false; }
};

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

#define MF_CUDA_OK(expr)                                                                   \
    do {                                                                                   \
        cudaError_t e__ = (expr);                                                          \
        if (e__ != cudaSuccess)                                                            \
            return mf::fail(MF_ERR_CUDA, "%s failed: %s", #expr, cudaGetErrorString(e__)); \
    } while (0)

// fp64 arithmetic that can never be contracted into FMA (bit-exact vs an IEEE-754 CPU).
__device__ __forceinline__ double dmul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double dadd(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double dsub(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ double ddiv(double a, double b) { return __ddiv_rn(a, b); }
__device__ __forceinline__ double dot3(double a0, double a1, double a2, double b0, double b1, double b2) {
    return dadd(dadd(dmul(a0, b0), dmul(a1, b1)), dmul(a2, b2));
}

// Rigid transform: rotation rows r[9] (row-major) and translation t[3].
struct Rigid {
    double r[9];
    double t[3];
};

__device__ __forceinline__ Rigid rigid_identity() {
    Rigid x;
#pragma unroll
    for (int i = 0; i < 9; ++i) x.r[i] = (i % 4 == 0) ? 1.0 : 0.0;
    x.t[0] = x.t[1] = x.t[2] = 0.0;
    return x;
}

// (Ra,ta).(Rb,tb) = (Ra Rb, Ra tb + ta)
__device__ __forceinline__ Rigid rigid_compose(const Rigid& a, const Rigid& b) {
    Rigid c;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
#pragma unroll
        for (int j = 0; j < 3; ++j)
            c.r[3 * i + j] = dot3(a.r[3 * i], a.r[3 * i + 1], a.r[3 * i + 2], b.r[j], b.r[3 + j], b.r[6 + j]);
        c.t[i] = dadd(dot3(a.r[3 * i], a.r[3 * i + 1], a.r[3 * i + 2], b.t[0], b.t[1], b.t[2]), a.t[i]);
    }
    return c;
}

// [R^T | -R^T t]
__device__ __forceinline__ Rigid rigid_inverse(const Rigid& a) {
    Rigid c;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
#pragma unroll
        for (int j = 0; j < 3; ++j) c.r[3 * i + j] = a.r[3 * j + i];
        c.t[i] = -dot3(a.r[i], a.r[3 + i], a.r[6 + i], a.t[0], a.t[1], a.t[2]);
    }
    return c;
}

}  // namespace mf
