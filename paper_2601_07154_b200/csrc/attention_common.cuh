// Pieces shared by the head_dim 64 and head_dim 128 attention kernels (attention.cu, attention_d128.cu).
#pragma once
#include "common.h"
#include "sm100_ptx.cuh"

#include <cuda_bf16.h>

// Of every 16 score pairs, this many are exponentiated on the FMA pipe instead of the MUFU (the two head_dim 64 kernels share
// the value: their exact paths are compared bit for bit, tests/test_gpu_attention_differential.py).
#ifndef MF_POLY_PAIRS
#define MF_POLY_PAIRS 5
#endif

namespace mf {

struct AttnParams {
    int seq_len;        // tokens per attention sequence (S, or P in frame mode)
    int heads;
    int q_blocks;       // ceil(seq_len / 256)
    float scale_log2;   // softmax_scale * log2(e)
    __nv_bfloat16* out;
    float* lse;         // [windows, heads, S] or nullptr
    int lse_frames;     // sequences per window (W in frame mode, 1 in global mode)
    const float* key_norm2_max;   // [sequences, heads] max over the keys of |k|^2 (attention.cu: the score bound), or nullptr
    const uint32_t* only_flagged; // window_attention_kernel: if not nullptr, CTAs whose word is 0 return at once (attention_split.cu did them)
};

// (2^x0, 2^x1) on the FMA pipe.  x = n + f with n = round(x), f in [-0.5, 0.5]; 2^f by a cubic (minimax in
// relative error, 7.5e-5); n is added into the exponent field.  x is clamped to >= -125 so the result stays normal.
__device__ __forceinline__ void exp2_poly2(uint32_t& a0, uint32_t& a1) {
    const float x0 = fmaxf(__uint_as_float(a0), -125.0f), x1 = fmaxf(__uint_as_float(a1), -125.0f);
    const uint64_t magic = ptx::pack2(12582912.0f, 12582912.0f);          // 1.5 * 2^23: x + magic holds round(x) in its low bits
    const uint64_t c3 = ptx::pack2(0.055171407759189606f, 0.055171407759189606f);
    const uint64_t c2 = ptx::pack2(0.24261075258255005f, 0.24261075258255005f);
    const uint64_t c1 = ptx::pack2(0.6932609677314758f, 0.6932609677314758f);
    const uint64_t c0 = ptx::pack2(0.9999281167984009f, 0.9999281167984009f);
    const uint64_t x = ptx::pack2(x0, x1);
    uint64_t t, n, f, p;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(t) : "l"(x), "l"(magic));
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(n) : "l"(t), "l"(magic));
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(f) : "l"(x), "l"(n));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(p) : "l"(c3), "l"(f), "l"(c2));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(p) : "l"(p), "l"(f), "l"(c1));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(p) : "l"(p), "l"(f), "l"(c0));
    uint32_t p0, p1, t0, t1;
    asm("mov.b64 {%0, %1}, %2;" : "=r"(p0), "=r"(p1) : "l"(p));
    asm("mov.b64 {%0, %1}, %2;" : "=r"(t0), "=r"(t1) : "l"(t));
    a0 = p0 + (t0 << 23);
    a1 = p1 + (t1 << 23);
}

// The same from the RAW scores on the score-bound path (attention.cu), where the subtracted constant m is an INTEGER and
// x = s * scale - m lies in [-64, 0]:  t = s * scale + (magic - m) holds n = round(x) in its low bits after one FFMA (magic - m
// is exact),  q = (magic - m) - t = -(n + m) exactly,  f = s * scale + q in [-0.5, 0.5] by a second FFMA.  No clamp (x >= -64
// keeps 2^n p normal) and no separate scaling: 6 packed instructions + 2 integer per pair instead of 9 + 2.
__device__ __forceinline__ void exp2_poly2_bounded(uint32_t& a0, uint32_t& a1, uint64_t scale2, uint64_t magic_minus_m2) {
    const uint64_t c3 = ptx::pack2(0.055171407759189606f, 0.055171407759189606f);
    const uint64_t c2 = ptx::pack2(0.24261075258255005f, 0.24261075258255005f);
    const uint64_t c1 = ptx::pack2(0.6932609677314758f, 0.6932609677314758f);
    const uint64_t c0 = ptx::pack2(0.9999281167984009f, 0.9999281167984009f);
    uint64_t s, t, q, f, p;
    asm("mov.b64 %0, {%1, %2};" : "=l"(s) : "r"(a0), "r"(a1));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(t) : "l"(s), "l"(scale2), "l"(magic_minus_m2));
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(q) : "l"(magic_minus_m2), "l"(t));             // -(n + m)
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(f) : "l"(s), "l"(scale2), "l"(q));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(p) : "l"(c3), "l"(f), "l"(c2));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(p) : "l"(p), "l"(f), "l"(c1));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(p) : "l"(p), "l"(f), "l"(c0));
    uint32_t p0, p1, t0, t1;
    asm("mov.b64 {%0, %1}, %2;" : "=r"(p0), "=r"(p1) : "l"(p));
    asm("mov.b64 {%0, %1}, %2;" : "=r"(t0), "=r"(t1) : "l"(t));
    a0 = p0 + (t0 << 23);
    a1 = p1 + (t1 << 23);
}

// head_dim 64, short sequences: persistent kernel driven by cluster launch control (attention_clc.cu); the caller supplies the
// tensor maps of q, k, v and out (box 64 x 1 x 128 x 1, SWIZZLE_128B)
mf_status launch_attention_clc(const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv, const CUtensorMap& mo,
                               int sequences, int seq_len, int heads, const AttnParams& prm, cudaStream_t stream);

// head_dim 64, long sequences, CTAs whose rows are all within the score bound (attention_split.cu); the others set their word
// of exact_flags (zeroed by the caller) and are left to window_attention_kernel
mf_status launch_attention_split(const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv, long long grid,
                                 const AttnParams& prm, uint32_t* exact_flags, cudaStream_t stream);

// head_dim 128 variant (attention_d128.cu); same contract as the head_dim 64 launch inside mf_window_attention
mf_status launch_attention_d128(const void* q, const void* k, const void* v, int sequences, int seq_len, int heads,
                                const AttnParams& prm, cudaStream_t stream);

}  // namespace mf
