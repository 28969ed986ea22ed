// Host-buffer entry points (end-to-end path): validate the whole chain of device calls first (mf::validate_only), then
// allocate device buffers from the stream-ordered pool, copy in, run the device entry points, copy out, synchronise.
// See include/mf.h.
#include "common.h"

namespace {

// Fake, distinct, 16-byte aligned device addresses for the validation pass (never dereferenced).
inline void* fake(int i) { return reinterpret_cast<void*>(static_cast<uintptr_t>(0x1000) * (i + 1)); }

struct DeviceBuf {
    void* p = nullptr;
    cudaStream_t s;
    explicit DeviceBuf(cudaStream_t st) : s(st) {}
    cudaError_t alloc(size_t bytes) { return cudaMallocAsync(&p, bytes ? bytes : 16, s); }
    ~DeviceBuf() {
        if (p) cudaFreeAsync(p, s);
    }
};

}  // namespace

extern "C" mf_status mf_window_attention_host(const void* q, const void* k, const void* v, void* out, int windows,
                                              int frames_per_window, int tokens_per_frame, int heads, int head_dim,
                                              int num_layers, mf_attn_mode first_mode, float softmax_scale,
                                              void* stream) {
    if (!q || !k || !v || !out) return mf::fail(MF_ERR_INVALID_ARG, "mf_window_attention_host: NULL tensor");
    if (windows < 1 || frames_per_window < 1 || tokens_per_frame < 1 || heads < 1 || head_dim < 1 || num_layers < 1)
        return mf::fail(MF_ERR_INVALID_ARG, "mf_window_attention_host: non-positive dimension");
    if (first_mode != MF_ATTN_GLOBAL && first_mode != MF_ATTN_FRAME)
        return mf::fail(MF_ERR_INVALID_ARG, "mf_window_attention_host: bad mode");
    {   // everything the per-layer calls below would reject, before anything is allocated or copied
        mf::ValidateOnlyScope dry;
        for (int l = 0; l < (num_layers > 1 ? 2 : 1); ++l) {
            const mf_attn_mode m = (l % 2 == 0) ? first_mode : (first_mode == MF_ATTN_GLOBAL ? MF_ATTN_FRAME : MF_ATTN_GLOBAL);
            mf_status st = mf_window_attention(fake(0), fake(1), fake(2), fake(3), nullptr, windows, frames_per_window,
                                               tokens_per_frame, heads, head_dim, m, softmax_scale, stream);
            if (st != MF_OK) return st;
        }
    }
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const size_t bytes = static_cast<size_t>(windows) * frames_per_window * tokens_per_frame * heads * head_dim * 2;
    DeviceBuf dq(s), dk(s), dv(s), dout(s), dout2(s);
    MF_CUDA_OK(dq.alloc(bytes));
    MF_CUDA_OK(dk.alloc(bytes));
    MF_CUDA_OK(dv.alloc(bytes));
    MF_CUDA_OK(dout.alloc(bytes));
    if (num_layers > 1) MF_CUDA_OK(dout2.alloc(bytes));
    MF_CUDA_OK(cudaMemcpyAsync(dq.p, q, bytes, cudaMemcpyHostToDevice, s));
    MF_CUDA_OK(cudaMemcpyAsync(dk.p, k, bytes, cudaMemcpyHostToDevice, s));
    MF_CUDA_OK(cudaMemcpyAsync(dv.p, v, bytes, cudaMemcpyHostToDevice, s));
    void* last = dout.p;
    for (int l = 0; l < num_layers; ++l) {
        const mf_attn_mode m = (l % 2 == 0) ? first_mode : (first_mode == MF_ATTN_GLOBAL ? MF_ATTN_FRAME : MF_ATTN_GLOBAL);
        last = (l % 2 == 0) ? dout.p : dout2.p;
        mf_status st = mf_window_attention(dq.p, dk.p, dv.p, last, nullptr, windows, frames_per_window,
                                           tokens_per_frame, heads, head_dim, m, softmax_scale, stream);
        if (st != MF_OK) return st;
    }
    MF_CUDA_OK(cudaMemcpyAsync(out, last, bytes, cudaMemcpyDeviceToHost, s));
    MF_CUDA_OK(cudaStreamSynchronize(s));
    return MF_OK;
}

extern "C" mf_status mf_chain_and_focus_host(const float* local_w2c, int num_windows, int W, int stride, int num_frames,
                                             mf_align_mode align, mf_intrinsics K, int render_begin, int render_end,
                                             int width, int height, const float* depth, const mf_focus_params* params,
                                             double* global_w2c, float* focus_map, float* guided_depth, float* focus_uv,
                                             int32_t* focus_index, void* stream) {
    if (!local_w2c || !params) return mf::fail(MF_ERR_INVALID_ARG, "mf_chain_and_focus_host: NULL pointer");
    if (num_windows < 1 || W < 1 || num_frames < 1 || render_end <= render_begin || width < 1 || height < 1)
        return mf::fail(MF_ERR_INVALID_ARG, "mf_chain_and_focus_host: bad dimensions");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int count = render_end - render_begin;
    const size_t loc_bytes = static_cast<size_t>(num_windows) * W * 16 * sizeof(float);
    const size_t pose_bytes = static_cast<size_t>(num_frames) * 16 * sizeof(double);
    const size_t img_bytes = static_cast<size_t>(count) * width * height * sizeof(float);
    const size_t ws_bytes = mf_motion_focus_workspace_size(count, width, height, params->n_points);
    if (ws_bytes == 0) return mf::fail(MF_ERR_INVALID_ARG, "mf_chain_and_focus_host: bad n_points or image size");
    {   // everything mf_chain_poses / mf_motion_focus below would reject, before anything is allocated or copied
        mf::ValidateOnlyScope dry;
        mf_status st = mf_chain_poses(static_cast<const float*>(fake(0)), 1, num_windows, W, stride, num_frames, align,
                                      static_cast<double*>(fake(1)), stream);
        if (st != MF_OK) return st;
        st = mf_motion_focus(static_cast<const double*>(fake(1)), K, num_frames, render_begin, render_end, width, height,
                             depth ? static_cast<const float*>(fake(2)) : nullptr, params,
                             focus_map ? static_cast<float*>(fake(3)) : nullptr, guided_depth ? static_cast<float*>(fake(4)) : nullptr,
                             static_cast<float*>(fake(5)), static_cast<int32_t*>(fake(6)), fake(7), ws_bytes, stream);
        if (st != MF_OK) return st;
    }
    DeviceBuf dloc(s), dpose(s), ddepth(s), dmap(s), dg(s), duv(s), didx(s), dws(s);
    MF_CUDA_OK(dloc.alloc(loc_bytes));
    MF_CUDA_OK(dpose.alloc(pose_bytes));
    MF_CUDA_OK(dws.alloc(ws_bytes));
    MF_CUDA_OK(duv.alloc(static_cast<size_t>(count) * 2 * sizeof(float)));
    MF_CUDA_OK(didx.alloc(static_cast<size_t>(count) * sizeof(int32_t)));
    if (depth) MF_CUDA_OK(ddepth.alloc(img_bytes));
    if (focus_map) MF_CUDA_OK(dmap.alloc(img_bytes));
    if (guided_depth) MF_CUDA_OK(dg.alloc(img_bytes));
    MF_CUDA_OK(cudaMemcpyAsync(dloc.p, local_w2c, loc_bytes, cudaMemcpyHostToDevice, s));
    if (depth) MF_CUDA_OK(cudaMemcpyAsync(ddepth.p, depth, img_bytes, cudaMemcpyHostToDevice, s));
    mf_status st = mf_chain_poses(static_cast<const float*>(dloc.p), 1, num_windows, W, stride, num_frames, align,
                                  static_cast<double*>(dpose.p), stream);
    if (st != MF_OK) return st;
    st = mf_motion_focus(static_cast<const double*>(dpose.p), K, num_frames, render_begin, render_end, width, height,
                         static_cast<const float*>(ddepth.p), params, static_cast<float*>(dmap.p),
                         static_cast<float*>(dg.p), static_cast<float*>(duv.p), static_cast<int32_t*>(didx.p), dws.p,
                         ws_bytes, stream);
    if (st != MF_OK) return st;
    if (global_w2c) MF_CUDA_OK(cudaMemcpyAsync(global_w2c, dpose.p, pose_bytes, cudaMemcpyDeviceToHost, s));
    if (focus_map) MF_CUDA_OK(cudaMemcpyAsync(focus_map, dmap.p, img_bytes, cudaMemcpyDeviceToHost, s));
    if (guided_depth) MF_CUDA_OK(cudaMemcpyAsync(guided_depth, dg.p, img_bytes, cudaMemcpyDeviceToHost, s));
    if (focus_uv) MF_CUDA_OK(cudaMemcpyAsync(focus_uv, duv.p, static_cast<size_t>(count) * 2 * sizeof(float), cudaMemcpyDeviceToHost, s));
    if (focus_index) MF_CUDA_OK(cudaMemcpyAsync(focus_index, didx.p, static_cast<size_t>(count) * sizeof(int32_t), cudaMemcpyDeviceToHost, s));
    MF_CUDA_OK(cudaStreamSynchronize(s));
    return MF_OK;
}
