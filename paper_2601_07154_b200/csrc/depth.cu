// mf_align_depth: per-window depth scale on the window overlap and stitching of the emitted frames into one stream
// (Fig. 3 "Depth alignment"; emitted frames P:76; reading F2 in DESIGN.md).
//
//   r_n = sum D_{n-1} D_n / sum D_n^2  over the frames windows n-1 and n share (pixels where both are finite and > 0),
//   c_0 = 1, c_n = c_{n-1} r_n,  D_out[t] = c_n D_n[t - start_n]  for the frames window n emits.
//
// Three launches, all HBM-bound streams:
//   overlap_sums_kernel  grid (Nw-1, kSumBlocks): the shared frames of a window pair are two contiguous runs of floats;
//                        every CTA sums its slice in fp64 (products of two fp32 are exact in fp64) in a fixed order and
//                        writes one partial pair, so the result does not depend on scheduling.   8 B per shared pixel.
//   scale_chain_kernel   one CTA: folds the partials of each window in index order, then the running product c_n.
//   stitch_kernel        grid (N, chunks): out[t] = fp32(c_n * D_n[k]) for the (n, k) that emits frame t.   8 B per pixel.
#include "common.h"

#include <algorithm>

namespace mf {

constexpr int kSumBlocks = 128;     // partial sums per window pair
constexpr int kSumThreads = 256;
constexpr int kStitchThreads = 256;

__device__ __forceinline__ int depth_win_start(int n, int stride, int num_frames, int W) {
    const int s = n * stride;
    return s < num_frames - W ? s : num_frames - W;
}

__device__ __forceinline__ float4 ld_nc4(const float4* p) {
    float4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_cs4(float4* p, float4 v) {
    asm volatile("st.global.cs.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

__device__ __forceinline__ void accumulate(float a, float b, double& sab, double& sbb) {
    if (a > 0.f && a < INFINITY && b > 0.f && b < INFINITY) {       // both finite and positive (NaN fails every test)
        const double bd = static_cast<double>(b);
        sab = fma(static_cast<double>(a), bd, sab);
        sbb = fma(bd, bd, sbb);
    }
}

// sum a b and sum b b over `count` floats (a: previous window, b: current), CTA blockIdx.y of kSumBlocks; out[2*blockIdx.y..]
template <bool VEC>
__device__ __forceinline__ void overlap_sums(const float* __restrict__ a, const float* __restrict__ b, size_t count,
                                             double* __restrict__ out) {
    double sab = 0.0, sbb = 0.0;
    const size_t tid = static_cast<size_t>(blockIdx.y) * kSumThreads + threadIdx.x;
    const size_t nthreads = static_cast<size_t>(kSumBlocks) * kSumThreads;
    if (VEC) {
        const size_t n4 = count >> 2;
        const float4* a4 = reinterpret_cast<const float4*>(a);
        const float4* b4 = reinterpret_cast<const float4*>(b);
        size_t i = tid;
        for (; i + 3 * nthreads < n4; i += 4 * nthreads) {       // four independent 16-byte loads per array in flight
            float4 av[4], bv[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                av[u] = ld_nc4(a4 + i + u * nthreads);
                bv[u] = ld_nc4(b4 + i + u * nthreads);
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                accumulate(av[u].x, bv[u].x, sab, sbb);
                accumulate(av[u].y, bv[u].y, sab, sbb);
                accumulate(av[u].z, bv[u].z, sab, sbb);
                accumulate(av[u].w, bv[u].w, sab, sbb);
            }
        }
        for (; i < n4; i += nthreads) {
            const float4 av = ld_nc4(a4 + i), bv = ld_nc4(b4 + i);
            accumulate(av.x, bv.x, sab, sbb);
            accumulate(av.y, bv.y, sab, sbb);
            accumulate(av.z, bv.z, sab, sbb);
            accumulate(av.w, bv.w, sab, sbb);
        }
    } else {
        for (size_t i = tid; i < count; i += nthreads) accumulate(__ldg(a + i), __ldg(b + i), sab, sbb);
    }
    // fixed-shape tree: lanes, then warps
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        sab += __shfl_down_sync(0xffffffffu, sab, o);
        sbb += __shfl_down_sync(0xffffffffu, sbb, o);
    }
    __shared__ double s_ab[kSumThreads / 32], s_bb[kSumThreads / 32];
    if ((threadIdx.x & 31) == 0) {
        s_ab[threadIdx.x >> 5] = sab;
        s_bb[threadIdx.x >> 5] = sbb;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double tab = 0.0, tbb = 0.0;
        for (int w = 0; w < kSumThreads / 32; ++w) {
            tab += s_ab[w];
            tbb += s_bb[w];
        }
        out[blockIdx.y * 2] = tab;
        out[blockIdx.y * 2 + 1] = tbb;
    }
}

template <bool VEC>
__global__ void __launch_bounds__(kSumThreads)
overlap_sums_kernel(const float* __restrict__ depth_local, int W, int stride, int num_frames, size_t px,
                    double* __restrict__ partials) {
    const int n = blockIdx.x + 1;
    const int s_prev = depth_win_start(n - 1, stride, num_frames, W), s_cur = depth_win_start(n, stride, num_frames, W);
    const size_t count = static_cast<size_t>(s_prev + W - s_cur) * px;                 // shared frames x pixels
    overlap_sums<VEC>(depth_local + (static_cast<size_t>(n - 1) * W + (s_cur - s_prev)) * px,
                      depth_local + static_cast<size_t>(n) * W * px, count, partials + static_cast<size_t>(n) * kSumBlocks * 2);
}

// Streaming form: one window pair per call, partials and the running scale in a small device-resident state.
struct DepthState {
    double c;                               // c_{n-1} before the call, c_n after it
    double partials[kSumBlocks * 2];
};

template <bool VEC>
__global__ void __launch_bounds__(kSumThreads)
overlap_sums_step_kernel(const float* __restrict__ prev_shared, const float* __restrict__ cur, size_t count, DepthState* st) {
    overlap_sums<VEC>(prev_shared, cur, count, st->partials);
}

__global__ void scale_step_kernel(DepthState* st, int first_window) {
    if (first_window) {
        st->c = 1.0;
        return;
    }
    double sab = 0.0, sbb = 0.0;
    for (int b = 0; b < kSumBlocks; ++b) {  // same fold order as scale_chain_kernel
        sab += st->partials[b * 2];
        sbb += st->partials[b * 2 + 1];
    }
    st->c *= sbb > 0.0 ? sab / sbb : 1.0;
}

template <bool VEC>
__global__ void __launch_bounds__(kStitchThreads)
stitch_step_kernel(const float* __restrict__ src_frames, const DepthState* __restrict__ st, size_t px, float* __restrict__ out) {
    const double c = st->c;
    const float* src = src_frames + static_cast<size_t>(blockIdx.x) * px;
    float* dst = out + static_cast<size_t>(blockIdx.x) * px;
    const size_t tid = static_cast<size_t>(blockIdx.y) * kStitchThreads + threadIdx.x;
    const size_t nthreads = static_cast<size_t>(gridDim.y) * kStitchThreads;
    auto scale1 = [c](float d) { return static_cast<float>(c * static_cast<double>(d)); };
    if (VEC) {
        for (size_t i = tid; i < (px >> 2); i += nthreads) {
            const float4 d = ld_nc4(reinterpret_cast<const float4*>(src) + i);
            st_cs4(reinterpret_cast<float4*>(dst) + i, make_float4(scale1(d.x), scale1(d.y), scale1(d.z), scale1(d.w)));
        }
    } else {
        for (size_t i = tid; i < px; i += nthreads) dst[i] = scale1(__ldg(src + i));
    }
}

__global__ void __launch_bounds__(256)
scale_chain_kernel(const double* __restrict__ partials, int num_windows, double* __restrict__ scales,
                   double* __restrict__ scales_out) {
    for (int n = 1 + threadIdx.x; n < num_windows; n += blockDim.x) {
        double sab = 0.0, sbb = 0.0;
        for (int b = 0; b < kSumBlocks; ++b) {
            sab += partials[(static_cast<size_t>(n) * kSumBlocks + b) * 2];
            sbb += partials[(static_cast<size_t>(n) * kSumBlocks + b) * 2 + 1];
        }
        scales[n] = sbb > 0.0 ? sab / sbb : 1.0;        // r_n
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double c = 1.0;
        scales[0] = 1.0;
        for (int n = 1; n < num_windows; ++n) {          // the "incremental" product, inherently ordered
            c *= scales[n];
            scales[n] = c;
        }
    }
    __syncthreads();
    if (scales_out)
        for (int n = threadIdx.x; n < num_windows; n += blockDim.x) scales_out[n] = scales[n];
}

template <bool VEC>
__global__ void __launch_bounds__(kStitchThreads)
stitch_kernel(const float* __restrict__ depth_local, const double* __restrict__ scales, int num_windows, int W,
              int stride, int num_frames, size_t px, float* __restrict__ depth_out) {
    const int t = blockIdx.x;
    // window that emits frame t: window 0 emits [0, W), window n >= 1 emits [start_{n-1} + W, start_n + W)
    int n = t < W ? 0 : (t - W) / stride + 1;
    n = n < num_windows - 1 ? n : num_windows - 1;
    const int k = t - depth_win_start(n, stride, num_frames, W);
    const double c = scales[n];
    const float* src = depth_local + (static_cast<size_t>(n) * W + k) * px;
    float* dst = depth_out + static_cast<size_t>(t) * px;
    const size_t tid = static_cast<size_t>(blockIdx.y) * kStitchThreads + threadIdx.x;
    const size_t nthreads = static_cast<size_t>(gridDim.y) * kStitchThreads;
    auto scale1 = [c](float d) { return static_cast<float>(c * static_cast<double>(d)); };   // one rounding
    if (VEC) {
        const size_t n4 = px >> 2;
        for (size_t i = tid; i < n4; i += nthreads) {
            const float4 d = ld_nc4(reinterpret_cast<const float4*>(src) + i);
            st_cs4(reinterpret_cast<float4*>(dst) + i, make_float4(scale1(d.x), scale1(d.y), scale1(d.z), scale1(d.w)));
        }
    } else {
        for (size_t i = tid; i < px; i += nthreads) dst[i] = scale1(__ldg(src + i));
    }
}

}  // namespace mf

extern "C" size_t mf_align_depth_workspace_size(int num_windows) {
    if (num_windows < 1) return 0;
    return sizeof(double) * (static_cast<size_t>(num_windows) * mf::kSumBlocks * 2 + num_windows);
}

extern "C" mf_status mf_align_depth(const float* depth_local, int num_windows, int W, int stride, int num_frames,
                                    int height, int width, float* depth_out, double* window_scale, void* workspace,
                                    size_t workspace_bytes, void* stream) {
    using namespace mf;
    if (!depth_local || !depth_out) return fail(MF_ERR_INVALID_ARG, "mf_align_depth: NULL depth pointer");
    if (W < 2 || stride < 1 || stride >= W || num_frames < W)
        return fail(MF_ERR_INVALID_ARG, "mf_align_depth: need 1 <= stride < W <= num_frames (W=%d stride=%d N=%d)", W, stride,
                    num_frames);
    if (num_windows != mf_num_windows(num_frames, W, stride))
        return fail(MF_ERR_INVALID_ARG, "mf_align_depth: num_windows=%d, expected %d", num_windows,
                    mf_num_windows(num_frames, W, stride));
    if (width < 1 || height < 1) return fail(MF_ERR_INVALID_ARG, "mf_align_depth: bad image size %dx%d", width, height);
    if (!workspace || workspace_bytes < mf_align_depth_workspace_size(num_windows) ||
        (reinterpret_cast<uintptr_t>(workspace) & 7u))
        return fail(MF_ERR_INVALID_ARG, "mf_align_depth: workspace too small or not 8-byte aligned");
    if (mf_status s = require_sm100()) return s;
    cudaStream_t q = static_cast<cudaStream_t>(stream);
    const size_t px = static_cast<size_t>(height) * width;
    double* partials = static_cast<double*>(workspace);
    double* scales = partials + static_cast<size_t>(num_windows) * kSumBlocks * 2;
    const bool vec = (px % 4 == 0) && aligned16(depth_local) && aligned16(depth_out);
    if (num_windows > 1) {
        const dim3 grid(num_windows - 1, kSumBlocks);
        if (vec)
            overlap_sums_kernel<true><<<grid, kSumThreads, 0, q>>>(depth_local, W, stride, num_frames, px, partials);
        else
            overlap_sums_kernel<false><<<grid, kSumThreads, 0, q>>>(depth_local, W, stride, num_frames, px, partials);
    }
    scale_chain_kernel<<<1, 256, 0, q>>>(partials, num_windows, scales, window_scale);
    const size_t units = vec ? px / 4 : px;
    const unsigned chunks = static_cast<unsigned>(std::min<size_t>((units + kStitchThreads * 4 - 1) / (kStitchThreads * 4), 1024));
    const dim3 sgrid(num_frames, chunks < 1 ? 1 : chunks);
    if (vec)
        stitch_kernel<true><<<sgrid, kStitchThreads, 0, q>>>(depth_local, scales, num_windows, W, stride, num_frames, px, depth_out);
    else
        stitch_kernel<false><<<sgrid, kStitchThreads, 0, q>>>(depth_local, scales, num_windows, W, stride, num_frames, px, depth_out);
    MF_CUDA_OK(cudaGetLastError());
    return MF_OK;
}

extern "C" size_t mf_align_depth_state_size(void) { return sizeof(mf::DepthState); }

extern "C" mf_status mf_align_depth_step(const float* prev_window, const float* cur_window, void* state, int W, int new_frames,
                                         int first_window, int height, int width, float* depth_out, void* stream) {
    using namespace mf;
    if (!cur_window || !state || !depth_out) return fail(MF_ERR_INVALID_ARG, "mf_align_depth_step: NULL pointer");
    if (reinterpret_cast<uintptr_t>(state) & 7u) return fail(MF_ERR_ALIGNMENT, "mf_align_depth_step: state must be 8-byte aligned");
    if (W < 2 || width < 1 || height < 1) return fail(MF_ERR_INVALID_ARG, "mf_align_depth_step: bad sizes");
    if (!first_window && (!prev_window || new_frames < 1 || new_frames >= W))
        return fail(MF_ERR_INVALID_ARG, "mf_align_depth_step: need the previous window and 1 <= new_frames < W (got %d, W=%d)",
                    new_frames, W);
    if (mf_status s = require_sm100()) return s;
    cudaStream_t q = static_cast<cudaStream_t>(stream);
    DepthState* st = static_cast<DepthState*>(state);
    const size_t px = static_cast<size_t>(height) * width;
    const int emit = first_window ? W : new_frames;
    const bool vec = (px % 4 == 0) && aligned16(cur_window) && aligned16(depth_out) && (first_window || aligned16(prev_window));
    if (!first_window) {
        const size_t count = static_cast<size_t>(W - new_frames) * px;
        const float* a = prev_window + static_cast<size_t>(new_frames) * px;      // the frames both windows hold
        if (vec)
            overlap_sums_step_kernel<true><<<dim3(1, kSumBlocks), kSumThreads, 0, q>>>(a, cur_window, count, st);
        else
            overlap_sums_step_kernel<false><<<dim3(1, kSumBlocks), kSumThreads, 0, q>>>(a, cur_window, count, st);
    }
    scale_step_kernel<<<1, 1, 0, q>>>(st, first_window);
    const size_t units = vec ? px / 4 : px;
    const unsigned chunks = static_cast<unsigned>(std::min<size_t>((units + kStitchThreads * 4 - 1) / (kStitchThreads * 4), 1024));
    const float* src = cur_window + static_cast<size_t>(W - emit) * px;
    if (vec)
        stitch_step_kernel<true><<<dim3(emit, chunks < 1 ? 1 : chunks), kStitchThreads, 0, q>>>(src, st, px, depth_out);
    else
        stitch_step_kernel<false><<<dim3(emit, chunks < 1 ? 1 : chunks), kStitchThreads, 0, q>>>(src, st, px, depth_out);
    MF_CUDA_OK(cudaGetLastError());
    return MF_OK;
}
