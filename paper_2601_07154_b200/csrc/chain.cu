// mf_chain_poses: incremental anchoring of window-local poses.
//
// One CTA per sequence.  Phase 1: every boundary transform B_n in parallel.  Phase 2: one thread
// left-folds A_n = A_{n-1}.B_n (the paper's "incremental" step, inherently ordered) and stores
// inv(A_n).  Phase 3: every emitted frame T^G_t = T^L_k . inv(A_n) in parallel.
// All arithmetic is fp64 through the non-contractible helpers of common.h so that the result is
// bit-identical to the same operation sequence on a CPU (needed for the bit-exact focus pixel).
#include "common.h"

namespace mf {

__device__ __forceinline__ Rigid load_local(const float* __restrict__ m) {
    Rigid x;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
#pragma unroll
        for (int j = 0; j < 3; ++j) x.r[3 * i + j] = static_cast<double>(m[4 * i + j]);
        x.t[i] = static_cast<double>(m[4 * i + 3]);
    }
    return x;
}

__device__ __forceinline__ int win_start(int n, int stride, int num_frames, int W) {
    int s = n * stride;
    return s < num_frames - W ? s : num_frames - W;
}

// Boundary transform B_n (RIGID: Cp.Tc; YAW: [Y | p(Cp) - Y p(Cc)]).
__device__ Rigid boundary(const Rigid& prev_last, const Rigid& cur_anchor, int mode) {
    Rigid cp = rigid_inverse(prev_last);
    if (mode == MF_ALIGN_RIGID) return rigid_compose(cp, cur_anchor);
    Rigid cc = rigid_inverse(cur_anchor);
    // R_rel = R(Cp) . R(Cc)^T ; only entries [2][2] and [0][2] are needed
    double a = dot3(cp.r[6], cp.r[7], cp.r[8], cc.r[6], cc.r[7], cc.r[8]);
    double b = dot3(cp.r[0], cp.r[1], cp.r[2], cc.r[6], cc.r[7], cc.r[8]);
    double r = __dsqrt_rn(dadd(dmul(a, a), dmul(b, b)));
    double c = 1.0, s = 0.0;
    if (!(r < 1e-12)) {
        c = ddiv(a, r);
        s = ddiv(b, r);
    }
    Rigid y;
    y.r[0] = c;   y.r[1] = 0.0; y.r[2] = s;
    y.r[3] = 0.0; y.r[4] = 1.0; y.r[5] = 0.0;
    y.r[6] = -s;  y.r[7] = 0.0; y.r[8] = c;
#pragma unroll
    for (int i = 0; i < 3; ++i)
        y.t[i] = dsub(cp.t[i], dot3(y.r[3 * i], y.r[3 * i + 1], y.r[3 * i + 2], cc.t[0], cc.t[1], cc.t[2]));
    return y;
}

__global__ void __launch_bounds__(256)
chain_poses_kernel(const float* __restrict__ local_w2c, int num_windows, int W, int stride, int num_frames,
                   int mode, double* __restrict__ global_w2c) {
    extern __shared__ double sm_a[];                 // [num_windows][12]: B_n, then inv(A_n)
    const int seq = blockIdx.x;
    const float* loc = local_w2c + static_cast<size_t>(seq) * num_windows * W * 16;
    double* out = global_w2c + static_cast<size_t>(seq) * num_frames * 16;

    for (int n = threadIdx.x; n < num_windows; n += blockDim.x) {
        Rigid b = rigid_identity();
        if (n > 0) {
            int k_a = (win_start(n - 1, stride, num_frames, W) + W - 1) - win_start(n, stride, num_frames, W);
            b = boundary(load_local(loc + (static_cast<size_t>(n - 1) * W + (W - 1)) * 16),
                         load_local(loc + (static_cast<size_t>(n) * W + k_a) * 16), mode);
        }
#pragma unroll
        for (int i = 0; i < 9; ++i) sm_a[12 * n + i] = b.r[i];
#pragma unroll
        for (int i = 0; i < 3; ++i) sm_a[12 * n + 9 + i] = b.t[i];
    }
    __syncthreads();

    if (threadIdx.x == 0) {
        Rigid a = rigid_identity();
        for (int n = 0; n < num_windows; ++n) {
            if (n > 0) {
                Rigid b;
#pragma unroll
                for (int i = 0; i < 9; ++i) b.r[i] = sm_a[12 * n + i];
#pragma unroll
                for (int i = 0; i < 3; ++i) b.t[i] = sm_a[12 * n + 9 + i];
                a = rigid_compose(a, b);
            }
            Rigid ai = rigid_inverse(a);
#pragma unroll
            for (int i = 0; i < 9; ++i) sm_a[12 * n + i] = ai.r[i];
#pragma unroll
            for (int i = 0; i < 3; ++i) sm_a[12 * n + 9 + i] = ai.t[i];
        }
    }
    __syncthreads();

    for (int t = threadIdx.x; t < num_frames; t += blockDim.x) {
        int n = t < W ? 0 : (t - W) / stride + 1;
        if (n > num_windows - 1) n = num_windows - 1;
        int k = t - win_start(n, stride, num_frames, W);
        Rigid ai;
#pragma unroll
        for (int i = 0; i < 9; ++i) ai.r[i] = sm_a[12 * n + i];
#pragma unroll
        for (int i = 0; i < 3; ++i) ai.t[i] = sm_a[12 * n + 9 + i];
        Rigid g = rigid_compose(load_local(loc + (static_cast<size_t>(n) * W + k) * 16), ai);
        double* o = out + static_cast<size_t>(t) * 16;
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            o[4 * i + 0] = g.r[3 * i + 0];
            o[4 * i + 1] = g.r[3 * i + 1];
            o[4 * i + 2] = g.r[3 * i + 2];
            o[4 * i + 3] = g.t[i];
        }
        o[12] = 0.0; o[13] = 0.0; o[14] = 0.0; o[15] = 1.0;
    }
}

// Streaming form ("incremental"): one window per call, A_{n-1} and the previous window's terminal local pose
// carried in a small device-resident state.  Same operations in the same order as chain_poses_kernel: bit-identical.
struct ChainState {
    double a[12];           // A_{n-1}: rotation rows then translation
    float prev_last[16];    // T^{L_{n-1} -> c}_{W-1}
    int windows_seen;
    int pad[3];
};

__global__ void __launch_bounds__(128)
chain_step_kernel(const float* __restrict__ win, ChainState* __restrict__ state, int W, int new_frames, int first, int mode,
                  double* __restrict__ out) {
    __shared__ double s_ai[12];
    const int emit_from = first ? 0 : W - new_frames;
    if (threadIdx.x == 0) {
        Rigid a = rigid_identity();
        if (!first) {
#pragma unroll
            for (int i = 0; i < 9; ++i) a.r[i] = state->a[i];
#pragma unroll
            for (int i = 0; i < 3; ++i) a.t[i] = state->a[9 + i];
            const Rigid b = boundary(load_local(state->prev_last), load_local(win + static_cast<size_t>(emit_from - 1) * 16), mode);
            a = rigid_compose(a, b);
        }
        const Rigid ai = rigid_inverse(a);
#pragma unroll
        for (int i = 0; i < 9; ++i) {
            s_ai[i] = ai.r[i];
            state->a[i] = a.r[i];
        }
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            s_ai[9 + i] = ai.t[i];
            state->a[9 + i] = a.t[i];
        }
        state->windows_seen = first ? 1 : state->windows_seen + 1;
    }
    __syncthreads();
    if (threadIdx.x < 16) state->prev_last[threadIdx.x] = win[static_cast<size_t>(W - 1) * 16 + threadIdx.x];
    Rigid ai;
#pragma unroll
    for (int i = 0; i < 9; ++i) ai.r[i] = s_ai[i];
#pragma unroll
    for (int i = 0; i < 3; ++i) ai.t[i] = s_ai[9 + i];
    for (int k = emit_from + threadIdx.x; k < W; k += blockDim.x) {
        const Rigid g = rigid_compose(load_local(win + static_cast<size_t>(k) * 16), ai);
        double* o = out + static_cast<size_t>(k - emit_from) * 16;
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            o[4 * i + 0] = g.r[3 * i + 0];
            o[4 * i + 1] = g.r[3 * i + 1];
            o[4 * i + 2] = g.r[3 * i + 2];
            o[4 * i + 3] = g.t[i];
        }
        o[12] = 0.0; o[13] = 0.0; o[14] = 0.0; o[15] = 1.0;
    }
}

}  // namespace mf

extern "C" mf_status mf_chain_poses(const float* local_w2c, int sequences, int num_windows, int W, int stride,
                                    int num_frames, mf_align_mode mode, double* global_w2c, void* stream) {
    if (!local_w2c || !global_w2c) return mf::fail(MF_ERR_INVALID_ARG, "mf_chain_poses: NULL pointer");
    if (sequences < 1) return mf::fail(MF_ERR_INVALID_ARG, "mf_chain_poses: sequences=%d", sequences);
    int expect = mf_num_windows(num_frames, W, stride);
    if (expect < 0)
        return mf::fail(MF_ERR_INVALID_ARG, "mf_chain_poses: need num_frames>=W and 1<=stride<W (N=%d W=%d stride=%d)",
                        num_frames, W, stride);
    if (num_windows != expect)
        return mf::fail(MF_ERR_INVALID_ARG, "mf_chain_poses: num_windows=%d but partition has %d", num_windows, expect);
    if (mode != MF_ALIGN_YAW_TRANSLATION && mode != MF_ALIGN_RIGID)
        return mf::fail(MF_ERR_INVALID_ARG, "mf_chain_poses: bad mode %d", static_cast<int>(mode));
    mf_status st = mf::require_sm100();
    if (st != MF_OK) return st;
    size_t smem = static_cast<size_t>(num_windows) * 12 * sizeof(double);
    if (smem > 200 * 1024)
        return mf::fail(MF_ERR_UNSUPPORTED, "mf_chain_poses: num_windows=%d exceeds the on-chip fold buffer (max 2133)",
                        num_windows);
    if (mf::validate_only()) return MF_OK;
    if (smem > 48 * 1024)
        MF_CUDA_OK(cudaFuncSetAttribute(mf::chain_poses_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        static_cast<int>(smem)));
    mf::chain_poses_kernel<<<sequences, 256, smem, static_cast<cudaStream_t>(stream)>>>(
        local_w2c, num_windows, W, stride, num_frames, static_cast<int>(mode), global_w2c);
    MF_CUDA_OK(cudaGetLastError());
    return MF_OK;
}

extern "C" size_t mf_chain_state_size(void) { return sizeof(mf::ChainState); }

extern "C" mf_status mf_chain_poses_step(const float* window_local_w2c, void* state, int W, int new_frames, int first_window,
                                         mf_align_mode mode, double* out_w2c, void* stream) {
    if (!window_local_w2c || !state || !out_w2c) return mf::fail(MF_ERR_INVALID_ARG, "mf_chain_poses_step: NULL pointer");
    if (W < 1) return mf::fail(MF_ERR_INVALID_ARG, "mf_chain_poses_step: W=%d", W);
    if (!first_window && (new_frames < 1 || new_frames >= W))
        return mf::fail(MF_ERR_INVALID_ARG, "mf_chain_poses_step: need 1 <= new_frames < W (overlap >= 1), got %d", new_frames);
    if (mode != MF_ALIGN_YAW_TRANSLATION && mode != MF_ALIGN_RIGID)
        return mf::fail(MF_ERR_INVALID_ARG, "mf_chain_poses_step: bad mode %d", static_cast<int>(mode));
    if ((reinterpret_cast<uintptr_t>(state) & 7u) != 0) return mf::fail(MF_ERR_ALIGNMENT, "mf_chain_poses_step: state must be 8-byte aligned");
    mf_status st = mf::require_sm100();
    if (st != MF_OK) return st;
    mf::chain_step_kernel<<<1, 128, 0, static_cast<cudaStream_t>(stream)>>>(window_local_w2c, static_cast<mf::ChainState*>(state), W,
                                                                           new_frames, first_window ? 1 : 0, static_cast<int>(mode),
                                                                           out_w2c);
    MF_CUDA_OK(cudaGetLastError());
    return MF_OK;
}
