/* mf.h -- C ABI of the B200-native (sm_100a) motion-focus hot path.
 *
 * Paper: "Motion Focus Recognition in Fast-Moving Egocentric Video" (arxiv 2601.07154),
 * cited as P:NN = line NN of PAPER.md; BJ = BASELINE.json north_star.
 *
 * Conventions (all entry points)
 *  - Pointers are DEVICE memory owned by the caller unless the name ends in _host.
 *    The library never frees or retains caller memory.
 *  - `stream` is a cudaStream_t passed as void* (NULL = default stream).  Work is enqueued
 *    on it and the call returns without synchronising (the *_host variants synchronise).
 *  - Return value is an mf_status.  Every argument, shape, alignment, workspace and device check is made
 *    before the first enqueue (the *_host variants run the checks of every call they are about to make before
 *    they allocate or copy), so MF_ERR_INVALID_ARG / UNSUPPORTED / ALIGNMENT / WORKSPACE mean nothing has been
 *    enqueued.  MF_ERR_CUDA reports a failing CUDA runtime call (allocation, copy, launch); work the same call
 *    enqueued before that failure may still run.
 *    mf_last_error() returns a thread-local, human-readable message for the last failure.
 *  - No CPU fallback: a device that is not sm_100, an unsupported shape or a misaligned
 *    pointer is an error.  NaN/Inf in inputs are not checked (they propagate).
 */
#ifndef MF_H_
#define MF_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    MF_OK = 0,
    MF_ERR_INVALID_ARG = 1,   /* bad dimension / enum / NULL pointer                    */
    MF_ERR_UNSUPPORTED = 2,   /* valid request this build cannot run (head_dim not 64 or 128...) */
    MF_ERR_ALIGNMENT = 3,     /* pointer not 16-byte aligned, width % 4 != 0            */
    MF_ERR_WORKSPACE = 4,     /* workspace NULL or too small                             */
    MF_ERR_CUDA = 5           /* CUDA runtime / driver error, no sm_100 device           */
} mf_status;

const char* mf_status_string(mf_status s);
const char* mf_last_error(void);
int mf_version(void);         /* major*10000 + minor*100 + patch */

/* ---------------------------------------------------------------------------------------------
 * Window attention (BJ: "cross-frame global self-attention over all S=W*P patch tokens of a
 * window, alternating with per-frame attention"; the sliding window is P:70).
 *
 *   out[n,i,h,:] = sum_j softmax_j( scale * q[n,i,h,:].k[n,j,h,:] ) v[n,j,h,:]
 *
 * GLOBAL: j over all S = W*P tokens of window n.  FRAME: j over the tokens of i's frame
 * (token order is frame-major, s = f*P + p).  bf16 inputs, fp32 scores/softmax/accumulation,
 * bf16 output rounded to nearest even.
 *
 * q,k,v,out: bf16 [windows, S, heads, head_dim] contiguous, 16-byte aligned; out must not
 * alias q/k/v.  lse: optional fp32 [windows, heads, S] natural-log-sum-exp of the scaled
 * scores (accurate to 2^-8 absolute: it is formed from the bf16-rounded weights the PV product
 * uses), or NULL.  head_dim must be 64 or 128 (else MF_ERR_UNSUPPORTED).  softmax_scale <= 0
 * selects 1/sqrt(head_dim).
 *
 * Device memory: at head_dim 64, sequences of 32 KV tiles and more (S >= 3969) first run a pass over k that
 * writes max |k|^2 per (sequence, head) into [sequences, heads] floats of scratch (the score bound of
 * csrc/attention.cu).  That scratch is allocated and freed ON `stream` from a memory pool owned by the
 * library (cudaMallocFromPoolAsync / cudaFreeAsync: no synchronisation, legal under stream capture, safe
 * with concurrent callers on other streams).  Every other path of this call allocates nothing.
 * mf_window_attention_noalloc below is the same call with that scratch in a static device array.
 * Rows whose bound |q_i| max_j|k_j| scale log2(e) exceeds 32, or holds NaN / Inf, take the exact
 * online-softmax path; the result is within the same bars either way.
 */
typedef enum { MF_ATTN_GLOBAL = 0, MF_ATTN_FRAME = 1 } mf_attn_mode;

mf_status mf_window_attention(const void* q, const void* k, const void* v, void* out, float* lse,
                              int windows, int frames_per_window, int tokens_per_frame,
                              int heads, int head_dim, mf_attn_mode mode, float softmax_scale,
                              void* stream);

/* ---------------------------------------------------------------------------------------------
 * Sliding-window partition ("overlapping segments of size L sharing O frames", "only
 * the newly processed, non-overlapping frames are emitted").  stride = L - O.  The last window
 * starts at num_frames - W when (num_frames - W) % stride != 0.  Pure host arithmetic.
 * Returns the window count, or -1 if num_frames < W, stride < 1 or stride >= W.
 */
int mf_num_windows(int num_frames, int W, int stride);
int mf_window_start(int num_frames, int W, int stride, int n);   /* -1 on bad arguments */

/* ---------------------------------------------------------------------------------------------
 * Pose chaining / incremental anchoring.
 *
 * local_w2c : fp32 [sequences, num_windows, W, 4, 4] row-major world->camera, each window in
 *             its own local world.  Only the top 3x4 of each matrix is read.
 * global_w2c: fp64 [sequences, num_frames, 4, 4]; world = window 0's local frame.
 * Window n >= 1 is aligned to window n-1 at the last frame of window n-1 (shared because
 * overlap >= 1).  MF_ALIGN_YAW_TRANSLATION (paper): rotation about the world Y axis by
 * the heading of the relative rotation's forward axis, plus the translation that makes the two
 * anchor camera centres coincide; pitch/roll of each window are kept.  MF_ALIGN_RIGID: full
 * 6-DoF alignment.  fp64 with + - * / sqrt only, no FMA contraction, fixed left-fold order:
 * results are bit-identical to the same operations on an IEEE-754 CPU.
 * Errors: num_windows != mf_num_windows(num_frames, W, stride) -> MF_ERR_INVALID_ARG.
 */
typedef enum { MF_ALIGN_YAW_TRANSLATION = 0, MF_ALIGN_RIGID = 1 } mf_align_mode;

mf_status mf_chain_poses(const float* local_w2c, int sequences, int num_windows, int W, int stride,
                         int num_frames, mf_align_mode mode, double* global_w2c, void* stream);

/* Streaming form of the pose chain (each batch is aligned "incrementally" to the terminal pose of the trajectory
 * so far).  One window per call; the state (A_{n-1} and the previous window's last local pose,
 * mf_chain_state_size() bytes of device memory, 8-byte aligned, contents irrelevant before the first window) is
 * updated in place.  first_window != 0: A_0 = I, all W frames are emitted.  Otherwise the window shares its first
 * W - new_frames frames with the previous window (new_frames = start_n - start_{n-1}, so 1 <= new_frames < W), it is
 * anchored at its local frame W - new_frames - 1 (= the previous window's last frame) and its last new_frames frames
 * are emitted.  out_w2c: fp64 [emitted, 4, 4].  Same operations in the same order as mf_chain_poses: feeding the
 * windows of a clip one by one reproduces its output bit for bit.
 */
size_t mf_chain_state_size(void);
mf_status mf_chain_poses_step(const float* window_local_w2c, void* state, int W, int new_frames, int first_window,
                              mf_align_mode mode, double* out_w2c, void* stream);

/* ---------------------------------------------------------------------------------------------
 * Motion focus (Eq. 1-7) and motion-guided depth (Fig. 1(iii), Fig. 5).
 *
 * For every rendered frame t in [render_begin, render_end):
 *   Eq.1  p_t = -R_t^T t_t                       Eq.3  a_w = p_i - 2 p_{i-1} + p_{i-2}
 *   Eq.4  a_c = R a_w                            Eq.6  (u,v) = (cx + fx ax/az, cy + fy ay/az)
 *   Eq.7  M(x,y) = (1/Z) sum_{i in trailing n_points frames} exp(-((x-u_i)^2+(y-v_i)^2)/(2 sigma_i^2))
 *   G(x,y) = M(x,y) * depth(x,y), and G = 0 exactly wherever M = 0 whatever depth holds there (a NaN/Inf depth
 *   sample propagates only inside the map's support; reading G1 in DESIGN.md).  The depth is not read where M = 0.
 * Pixel (x,y) is centred at (u,v) = (x,y).  A point is skipped when it needs a frame < 0,
 * when |a_w| < 1e-12, or when |a_z| <= eps_z*|a_c|.  sigma_i = sigma*|a_w| (MF_MAG_RAW) or
 * sigma (MF_MAG_UNIT), clamped to >= 1e-3 px.  Z = per-frame max over pixels (MF_NORM_MAX),
 * sum (MF_NORM_SUM) or 1 (MF_NORM_NONE); Z = 0 gives M = 0.
 * The point stage runs in fp64 (same bit-exactness rules as mf_chain_poses); (u_i,v_i,sigma_i)
 * are rounded once to fp32 and the render runs in fp32.
 */
typedef struct { double fx, fy, cx, cy; } mf_intrinsics;       /* at focus-map resolution, Eq.5 */
typedef enum { MF_VEC_ACCEL = 0 /* Eq.3 */, MF_VEC_VELOCITY = 1 /* P:125 contrast */ } mf_vec_mode;
typedef enum { MF_MAG_RAW = 0, MF_MAG_UNIT = 1 } mf_mag_mode;
typedef enum { MF_NORM_MAX = 0, MF_NORM_SUM = 1, MF_NORM_NONE = 2 } mf_norm_mode;
typedef enum { MF_PTS_CURRENT_FRAME = 0 /* R = R_t */, MF_PTS_OWN_FRAME = 1 /* R = R_i */ } mf_pts_mode;

typedef struct {
    int n_points;        /* 1..32 (paper: N = 15)                           */
    float sigma;         /* > 0                                                    */
    int vec;             /* mf_vec_mode                                            */
    int mag;             /* mf_mag_mode                                            */
    int norm;            /* mf_norm_mode                                           */
    int pts;             /* mf_pts_mode                                            */
    double eps_z;        /* >= 0; 1e-6 recommended                                 */
} mf_focus_params;

/* Bytes of device scratch mf_motion_focus needs for `count` rendered frames. */
size_t mf_motion_focus_workspace_size(int count, int width, int height, int n_points);

/* global_w2c: fp64 [num_frames,4,4].  depth: fp32 [count,height,width] or NULL.
 * focus_map: fp32 [count,height,width] or NULL (points only).  guided_depth: fp32 same shape
 * or NULL (requires depth and focus_map).  focus_uv: fp32 [count,2] (u,v) of the frame's own point, NaN
 * if invalid, or NULL.  focus_index: int32 [count], y*width+x with x=floor(u+.5), y=floor(v+.5),
 * -1 if invalid or off-image, or NULL.  count = render_end - render_begin.
 * width % 4 == 0 and 16-byte aligned image pointers are required (MF_ERR_ALIGNMENT).
 */
mf_status mf_motion_focus(const double* global_w2c, mf_intrinsics K, int num_frames,
                          int render_begin, int render_end, int width, int height,
                          const float* depth, const mf_focus_params* params,
                          float* focus_map, float* guided_depth, float* focus_uv,
                          int32_t* focus_index, void* workspace, size_t workspace_bytes,
                          void* stream);

/* ---------------------------------------------------------------------------------------------
 * Depth alignment across windows and stitching of the emitted frames (Fig. 3 "Depth alignment"; emitted frames
 * P:76).  The paper gives no formula for the depth scale (its pose alignment is rigid);
 * reading F2 in DESIGN.md: window n >= 1 is brought to the scale of the stream so far by the least-squares factor on the
 * frames it shares with window n-1,
 *     r_n = sum D_{n-1} D_n / sum D_n^2   over pixels of the shared frames where both depths are finite and > 0
 *           (r_n = 1 when there is none),      c_0 = 1,  c_n = c_{n-1} r_n,
 * and frame t, emitted by window n at local index k, becomes depth_out[t] = fp32(c_n * depth_local[n][k]).
 * depth_local: fp32 device [num_windows, W, height, width], each window in its own scale.  depth_out: fp32 device
 * [num_frames, height, width].  window_scale: fp64 device [num_windows] receiving c_n, or NULL.  workspace:
 * mf_align_depth_workspace_size(num_windows) bytes of device memory, 8-byte aligned.  Sums are fp64 in a fixed order:
 * the result is deterministic.  Errors: num_windows != mf_num_windows(num_frames, W, stride), bad sizes, NULL or short
 * workspace -> MF_ERR_INVALID_ARG.  Any height/width is accepted (16-byte vector path when height*width % 4 == 0 and the
 * pointers are 16-byte aligned).
 */
size_t mf_align_depth_workspace_size(int num_windows);
mf_status mf_align_depth(const float* depth_local, int num_windows, int W, int stride, int num_frames,
                         int height, int width, float* depth_out, double* window_scale, void* workspace,
                         size_t workspace_bytes, void* stream);

/* Streaming form of mf_align_depth (one window per call, as mf_chain_poses_step).  state:
 * mf_align_depth_state_size() bytes of device memory, 8-byte aligned, contents irrelevant before the first window; it holds
 * c_{n-1} and is updated in place.  first_window != 0: c_0 = 1 and all W frames of cur_window are emitted.  Otherwise
 * prev_window is the previous window's [W, height, width] depth (unscaled, as the model produced it), the two windows share
 * the last W - new_frames frames of prev_window = the first W - new_frames frames of cur_window (1 <= new_frames < W), and the
 * last new_frames frames of cur_window are emitted, scaled by c_n.  depth_out: fp32 device [emitted, height, width].  Same sums
 * in the same order as mf_align_depth: feeding the windows of a clip one by one reproduces its output bit for bit (given the
 * same 16-byte alignment of the window buffers, which selects the vector path).
 */
size_t mf_align_depth_state_size(void);
mf_status mf_align_depth_step(const float* prev_window, const float* cur_window, void* state, int W, int new_frames,
                              int first_window, int height, int width, float* depth_out, void* stream);

/* mf_motion_focus with the depth at the MODEL's resolution (the paper does not say how its depth
 * maps reach the focus-map resolution, reading F1 in DESIGN.md): depth_lowres is fp32 [count, depth_height, depth_width]
 * and is interpolated inside the render pass, bilinear with half-pixel centres and edge clamping (what
 * torch.nn.functional.interpolate(mode="bilinear", align_corners=False) computes), so the full-resolution depth never
 * exists in HBM: the pass writes 8 B/pixel and reads almost nothing.  focus_map and guided_depth are required; every other
 * argument as in mf_motion_focus (same workspace size).  Image and depth sizes above 32767 return MF_ERR_UNSUPPORTED.
 */
mf_status mf_motion_focus_upsampled(const double* global_w2c, mf_intrinsics K, int num_frames,
                                    int render_begin, int render_end, int width, int height,
                                    const float* depth_lowres, int depth_width, int depth_height,
                                    const mf_focus_params* params, float* focus_map, float* guided_depth,
                                    float* focus_uv, int32_t* focus_index, void* workspace,
                                    size_t workspace_bytes, void* stream);

/* mf_window_attention for callers that cannot allocate device memory (CUDA graph capture, serving loops, harnesses that
 * forbid it).  Same arguments, semantics, checks and results as mf_window_attention.  The one scratch buffer that call
 * takes from a stream-ordered pool (head_dim 64, sequences of 32 KV tiles and more: [sequences, heads] floats holding
 * max |k|^2 for the score bound, csrc/attention.cu) is here a fixed 256 KB array inside the library's device image, so the
 * call performs no cudaMalloc / cudaFree / pool operation of any kind.  Limits and caveats:
 *   - sequences x heads (sequences = windows in GLOBAL mode, windows*W in FRAME mode) must be <= 65536 on that path,
 *     else MF_ERR_UNSUPPORTED (nothing enqueued); the other paths (head_dim 128, shorter sequences) use no scratch and
 *     have no such limit.  (Where sequences x heads + ceil(S/256) x heads x sequences also fits in 65536 words, the array
 *     holds the per-CTA flags of csrc/attention_split.cu as well and the call runs the same kernels as
 *     mf_window_attention; beyond that it runs window_attention_kernel alone: same results, ~4 % slower.);
 *   - every call on a device shares the array (it is cleared by each call before use): calls that may overlap on the
 *     GPU (different streams, concurrent graph launches) race on it -- serialise them or use mf_window_attention;
 *   - the array is held by every GPU that loads the library, until the process exits.
 */
mf_status mf_window_attention_noalloc(const void* q, const void* k, const void* v, void* out, float* lse,
                                      int windows, int frames_per_window, int tokens_per_frame, int heads,
                                      int head_dim, mf_attn_mode mode, float softmax_scale, void* stream);

/* ---------------------------------------------------------------------------------------------
 * Host-buffer conveniences (end-to-end path): same semantics, every pointer is HOST memory
 * (pinned memory makes the copies asynchronous).  They allocate device buffers, copy in,
 * run the device entry point above, copy out and synchronise `stream` before returning.
 */
/* Runs `num_layers` attention layers on the same q/k/v (layer l uses first_mode when l is even and the
 * other mode when l is odd; outputs ping-pong between two device buffers) and returns the last
 * layer's output.  num_layers = 1 is a single mf_window_attention call.  Copies: q,k,v in once, out once. */
mf_status mf_window_attention_host(const void* q, const void* k, const void* v, void* out,
                                   int windows, int frames_per_window, int tokens_per_frame,
                                   int heads, int head_dim, int num_layers, mf_attn_mode first_mode,
                                   float softmax_scale, void* stream);

/* local_w2c fp32 [num_windows,W,4,4] (one sequence) -> chain -> focus maps of frames
 * [render_begin, render_end).  global_w2c (fp64 [num_frames,4,4]) may be NULL. */
mf_status mf_chain_and_focus_host(const float* local_w2c, int num_windows, int W, int stride,
                                  int num_frames, mf_align_mode align, mf_intrinsics K,
                                  int render_begin, int render_end, int width, int height,
                                  const float* depth, const mf_focus_params* params,
                                  double* global_w2c, float* focus_map, float* guided_depth,
                                  float* focus_uv, int32_t* focus_index, void* stream);

/* ---------------------------------------------------------------------------------------------
 * Dense layers around the window attention.  PAPER.md treats the transformer as
 * a black box; BJ fixes only "24-layer d=1024 H=16 stack".  The standard pre-norm block is
 * taken as reading E1-E4: h = x + W_o Attn(W_qkv LN1(x)), y = h + W_2 GELU(W_1 LN2(h)).
 *
 * mf_linear:  out = act(x w^T + bias) (+ residual), bf16 operands, fp32 accumulation (tcgen05 MMA into
 * TMEM), bf16 output rounded to nearest even.
 *   x        bf16 [M, K] row-major              w     bf16 [N, K] row-major (nn.Linear layout)
 *   bias     fp32 [N] or NULL                   residual  bf16 [M, N] or NULL (single output only)
 *   out0..2  bf16 [M, n_split] each: output tensor i receives columns [i*n_split, (i+1)*n_split) of the
 *            product, so N = 3*n_split writes q | k | v as three [tokens, heads*head_dim] tensors in one
 *            pass; N = n_split writes one tensor (out1 = out2 = NULL).
 *   act      MF_ACT_GELU is the exact erf form (reading E3).
 * K % 64 == 0 and n_split % 256 == 0 are required (MF_ERR_UNSUPPORTED otherwise); all tensors 16-byte
 * aligned; outputs must not alias x (residual may equal out0: each element is read before it is written
 * by the same thread).
 *
 * mf_layernorm: out = (x - mean) / sqrt(var + eps) * gamma + beta over the last axis (biased variance,
 * fp32 statistics), x/out bf16 [M, d], gamma/beta fp32 [d]; d in {256, 512, 768, 1024}.
 */
typedef enum { MF_ACT_NONE = 0, MF_ACT_GELU = 1 } mf_activation;

mf_status mf_linear(const void* x, const void* w, const float* bias, const void* residual, void* out0,
                    void* out1, void* out2, int M, int N, int K, int n_split, mf_activation act,
                    void* stream);

mf_status mf_layernorm(const void* x, const float* gamma, const float* beta, float eps, void* out, int M,
                       int d, void* stream);

/* One pre-norm transformer block around the window attention (reading E1, E2, E5 in DESIGN.md):
 *   h = x + W_o Attn(split_heads(W_qkv LN1(x) + b_qkv)) + b_o ;  y = h + W_2 GELU(W_1 LN2(h) + b_1) + b_2
 * x, y: bf16 [windows * W * P, heads * head_dim] (token order as in mf_window_attention); y may equal x (in place).
 * Weights are nn.Linear-layout bf16 matrices and fp32 vectors (all device memory, 16-byte aligned):
 *   w_qkv [3 d, d] (rows: q | k | v, each head-major), w_o [d, d], w_1 [d_hidden, d], w_2 [d, d_hidden].
 * Every tensor kept between two kernels is bf16 (E5).  Seven launches: layernorm, linear (q|k|v), window attention,
 * linear (+residual), layernorm, linear (+GELU), linear (+residual).  d = heads * head_dim must be 256, 512, 768 or
 * 1024 with head_dim 64 or 128, d_hidden % 256 == 0.  workspace: mf_block_workspace_size() bytes of device memory.
 */
typedef struct {
    const float* ln1_gamma; const float* ln1_beta;
    const void* w_qkv;      const float* b_qkv;
    const void* w_o;        const float* b_o;
    const float* ln2_gamma; const float* ln2_beta;
    const void* w_1;        const float* b_1;
    const void* w_2;        const float* b_2;
} mf_block_weights;

size_t mf_block_workspace_size(int windows, int frames_per_window, int tokens_per_frame, int d_model, int d_hidden);

mf_status mf_block_forward(const void* x, const mf_block_weights* weights, void* y, int windows,
                           int frames_per_window, int tokens_per_frame, int heads, int head_dim, int d_hidden,
                           mf_attn_mode mode, float ln_eps, void* workspace, size_t workspace_bytes, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* MF_H_ */
