// mf_window_attention, head_dim 64, long sequences, rows on the SCORE-BOUND path only (attention.cu explains the bound): the tile
// pipeline of window_attention_kernel with FOUR softmax warps per scheduler instead of two.
//
// On the score-bound path a row's exponentials depend on nothing but its scores (the subtracted constant is known before the
// first tile, the row sum accumulates on the tensor core through the ones column), so the 128 scores of a row and KV tile can be
// split between two threads without any exchange: warpgroup "half 0" of a Q tile takes keys 0-63 of every KV tile, warpgroup
// "half 1" keys 64-127.  Each thread holds 64 scores instead of 128, and a scheduler has four independent softmax warps to
// cover each other's tcgen05.ld / barrier / MUFU latencies (window_attention_kernel: two warps, 51 % of the issue slots used, MUFU
// 69 % busy; profiles/r2_ncu_attn.md).  Everything else is window_attention_kernel's: TMA producer, one MMA issuer per Q tile, the
// K/V ring, TMEM map (S0 S1 | O0 O1 | P0 P1: the two halves of a tile still take turns on one 32-column P buffer, now from
// different warps), ones column, watchdog.  The arithmetic per score is the same instruction for instruction, so the output is
// bit-identical to window_attention_kernel's score-bound path (tests/test_gpu_attention_differential.py).
//
// A CTA whose 256 rows are not ALL within the bound does no work here: it sets exact_flags[blockIdx.x] and exits, and
// window_attention_kernel, launched behind this kernel on the same stream with AttnParams::only_flagged, does exactly those
// CTAs (exact online softmax per warp, as before) and returns at once from all others.
//
// Roles: warps 0-3 tile 0 / keys 0-63, warps 4-7 tile 1 / keys 0-63, warps 8-11 tile 0 / keys 64-127, warps 12-15 tile 1 / keys
// 64-127 (a warp reads the TMEM lanes 32 (warp % 4) .. +31: its rows), warp 16 TMA producer, warps 17-18 MMA issuers, warp 19 watchdog.
#include "attention_common.cuh"
#include "tensormap.h"

#include <atomic>
#include <cstddef>
#include <type_traits>

namespace mf {
namespace split {

constexpr int kD = 64, kBM = 128, kBN = 128, kQTiles = 2, kStages = 4;
constexpr int kTileBytes = kBM * kD * 2;
constexpr int kSoftmaxWarps = 16;
constexpr int kThreads = 640;
constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kColS = 0, kColO = 256, kColP = 416;
constexpr int kON = 80;
constexpr int kPH = 32;
constexpr float kScoreBoundMax = 32.0f;          // (attention.cu)
#ifndef MF_POLY_PAIRS_BOUND
#define MF_POLY_PAIRS_BOUND 7          // (attention.cu has the sweep; the two kernels must agree)
#endif

struct Smem {
    alignas(1024) uint8_t q[kQTiles][kTileBytes];
    alignas(1024) uint8_t k[kStages][kTileBytes];
    alignas(1024) uint8_t v[kStages][kTileBytes];
    alignas(1024) uint8_t ones[kTileBytes];
    alignas(8) uint64_t q_full;
    uint64_t k_full[kStages], k_empty[kStages], v_full[kStages], v_empty[kStages];
    uint64_t s_full[kQTiles], s_free[kQTiles], p_full[2][kQTiles], pv_done[2][kQTiles];   // [half][tile]
    uint64_t roles_done;
    uint32_t tmem_base;
    uint32_t zero;
};

constexpr uint32_t kIdescQK = ptx::idesc_bf16_f32(kBM, kBN, 0, 0);
constexpr uint32_t kIdescPV = ptx::idesc_bf16_f32(kBM, kON, 0, 1);

__device__ __forceinline__ void issue_qk(uint32_t tmem_s, uint32_t q, uint32_t k) {
    const uint64_t qd = ptx::smem_desc_sw128(q);
    const uint64_t kd = ptx::smem_desc_sw128(k);
#pragma unroll
    for (int i = 0; i < kD / 16; ++i) ptx::mma_ss(tmem_s, qd + 2 * i, kd + 2 * i, kIdescQK, i > 0);
}
__device__ __forceinline__ void issue_pv_half(uint32_t tmem_o, uint32_t tmem_p, uint32_t v_half, uint32_t ones_minus_v, bool accumulate) {
    const uint64_t vd = ptx::smem_desc_sw128(v_half, ones_minus_v);
#pragma unroll
    for (int i = 0; i < kBN / 32; ++i)
        ptx::mma_ts(tmem_o, tmem_p + 8 * i, vd + (2048 >> 4) * i, kIdescPV, (accumulate || i > 0) ? 1u : 0u);
}

__global__ void __launch_bounds__(kThreads, 1)
window_attention_split_kernel(const __grid_constant__ CUtensorMap map_q, const __grid_constant__ CUtensorMap map_k,
                              const __grid_constant__ CUtensorMap map_v, const AttnParams prm, uint32_t* __restrict__ exact_flags) {
    extern __shared__ uint8_t smem_raw[];
    Smem& sm = *reinterpret_cast<Smem*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    // (warp number through a shuffle: warp-uniform to the compiler, see attention.cu)
    const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;

    const int qb = blockIdx.x % prm.q_blocks;
    const int head = (blockIdx.x / prm.q_blocks) % prm.heads;
    const int seq = blockIdx.x / (prm.q_blocks * prm.heads);
    const int row0 = qb * (kQTiles * kBM);
    const bool tile1_live = row0 + kBM < prm.seq_len;
    const int n_kv = (prm.seq_len + kBN - 1) / kBN;

    if (warp == 16 && lane == 0) {
        ptx::prefetch_tensormap(&map_q);
        ptx::prefetch_tensormap(&map_k);
        ptx::prefetch_tensormap(&map_v);
        const uint32_t live = tile1_live ? 2 : 1;          // MMA issuers that release every K/V stage
        ptx::mbar_init(&sm.q_full, 1);
        for (int s = 0; s < kStages; ++s) {
            ptx::mbar_init(&sm.k_full[s], 1);
            ptx::mbar_init(&sm.k_empty[s], live);
            ptx::mbar_init(&sm.v_full[s], 1);
            ptx::mbar_init(&sm.v_empty[s], live);
        }
        for (int t = 0; t < kQTiles; ++t) {
            ptx::mbar_init(&sm.s_full[t], 1);
            ptx::mbar_init(&sm.s_free[t], 8);              // one arrival per softmax warp of the tile, both halves
            for (int h = 0; h < 2; ++h) {
                ptx::mbar_init(&sm.p_full[h][t], 4);       // the four warps of that half
                ptx::mbar_init(&sm.pv_done[h][t], 1);
            }
        }
        sm.zero = 0;
        ptx::mbar_init(&sm.roles_done, 19);
        ptx::fence_barrier_init();
    }
    {   // ones tile: logical (key r, column 0) = 1.0 under the 128-byte swizzle, everything else 0
        uint4* o4 = reinterpret_cast<uint4*>(sm.ones);
        for (int i = threadIdx.x; i < kTileBytes / 16; i += kThreads) {
            const int r = i >> 3, chunk = i & 7;
            o4[i] = make_uint4(chunk == (r & 7) ? 0x00003F80u : 0u, 0u, 0u, 0u);
        }
        ptx::fence_proxy_async();
    }
    if (warp == 17) ptx::tmem_alloc(&sm.tmem_base, kTmemCols);
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = __shfl_sync(0xffffffffu, sm.tmem_base, 0);
    const uint32_t sb = ptx::smem_u32(&sm);

    // ---- Q tiles, then the CTA-wide decision: are all of this CTA's rows within the score bound? ----
    if (warp == 16 && ptx::elect_one()) {
        const uint32_t a_q_full = sb + offsetof(Smem, q_full);
        ptx::mbar_arrive_expect_tx(a_q_full, (tile1_live ? 2 : 1) * kTileBytes);
        ptx::tma_load_4d(sb + offsetof(Smem, q), &map_q, a_q_full, 0, head, row0, seq);
        if (tile1_live) ptx::tma_load_4d(sb + offsetof(Smem, q) + kTileBytes, &map_q, a_q_full, 0, head, row0 + kBM, seq);
        // the first K/V stages go out before the decision (no wait needed: the ring is empty), so that it costs no load latency
        for (int j = 0; j < kStages && j < n_kv; ++j) {
            ptx::mbar_arrive_expect_tx(sb + offsetof(Smem, k_full) + 8 * j, kTileBytes);
            ptx::tma_load_4d(sb + offsetof(Smem, k) + kTileBytes * j, &map_k, sb + offsetof(Smem, k_full) + 8 * j, 0, head, j * kBN, seq);
            ptx::mbar_arrive_expect_tx(sb + offsetof(Smem, v_full) + 8 * j, kTileBytes);
            ptx::tma_load_4d(sb + offsetof(Smem, v) + kTileBytes * j, &map_v, sb + offsetof(Smem, v_full) + 8 * j, 0, head, j * kBN, seq);
        }
    }
    __syncwarp();
    const int tile = (warp >> 2) & 1, half = (warp >> 3) & 1;            // (softmax warps)
    const int row_in_tile = (warp & 3) * 32 + lane;
    float m_used = 0.f;
    int outside = 0;
    if (warp < kSoftmaxWarps && (tile == 0 || tile1_live)) {
        ptx::mbar_wait(sb + offsetof(Smem, q_full), 0);
        const uint4* q_row = reinterpret_cast<const uint4*>(sm.q[tile] + row_in_tile * (kD * 2));
        float qq = 0.f;
#pragma unroll
        for (int c = 0; c < 8; ++c) {                 // (same order of summation as attention.cu: the two kernels agree on every bound)
            const uint4 w = q_row[(c + lane) & 7];
            const uint32_t u[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const float lo = __uint_as_float(u[i] << 16), hi = __uint_as_float(u[i] & 0xffff0000u);
                qq = fmaf(lo, lo, fmaf(hi, hi, qq));
            }
        }
        const float kk = prm.key_norm2_max[static_cast<size_t>(seq) * prm.heads + head];
        const float bound = sqrtf(qq * kk) * fabsf(prm.scale_log2) * (1.0f + 0x1p-10f);
        outside = !(bound <= kScoreBoundMax);
        m_used = ceilf(bound);
    }
    if (__syncthreads_or(outside)) {
        // window_attention_kernel does this CTA.  Shared memory must outlive the loads in flight: the Q loads have landed (every
        // live softmax thread waited for them); the K/V stages sent ahead are waited for here.
        if (threadIdx.x == 0) exact_flags[blockIdx.x] = 1u;
        if (warp == 16)
            for (int j = 0; j < kStages && j < n_kv; ++j) {
                ptx::mbar_wait(sb + offsetof(Smem, k_full) + 8 * j, 0);
                ptx::mbar_wait(sb + offsetof(Smem, v_full) + 8 * j, 0);
            }
        ptx::tc_fence_before();
        __syncthreads();
        if (warp == 17) ptx::tmem_dealloc(tmem, kTmemCols);
        return;
    }

    // register split: 96/thread at launch (640 threads) -> 104 for the 16 softmax warps, 56 for the other four.  (setmaxnreg moves
    // registers inside the CTA's own allocation: 512 x 104 + 128 x 56 = 60416 <= 640 x 96; asking for more than the other warps
    // give up blocks the softmax warps for good.)
    if (warp >= kSoftmaxWarps) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        if (warp == 16) {
            // ===================== TMA producer (whole warp in the loop, one elected lane issues) =====================
            const bool leader = ptx::elect_one();
            for (int j = kStages; j < n_kv; ++j) {           // (stages 0 .. kStages-1 were sent before the decision)
                const int st = j % kStages;
                const uint32_t ph = (j / kStages) & 1;
                ptx::mbar_wait(sb + offsetof(Smem, k_empty) + 8 * st, ph ^ 1);
                if (leader) {
                    ptx::mbar_arrive_expect_tx(sb + offsetof(Smem, k_full) + 8 * st, kTileBytes);
                    ptx::tma_load_4d(sb + offsetof(Smem, k) + kTileBytes * st, &map_k, sb + offsetof(Smem, k_full) + 8 * st, 0, head, j * kBN, seq);
                }
                ptx::mbar_wait(sb + offsetof(Smem, v_empty) + 8 * st, ph ^ 1);
                if (leader) {
                    ptx::mbar_arrive_expect_tx(sb + offsetof(Smem, v_full) + 8 * st, kTileBytes);
                    ptx::tma_load_4d(sb + offsetof(Smem, v) + kTileBytes * st, &map_v, sb + offsetof(Smem, v_full) + 8 * st, 0, head, j * kBN, seq);
                }
            }
            __syncwarp();
        } else if (warp <= 18) {
            // ===================== MMA issuers (warp 17: Q tile 0, warp 18: Q tile 1; one elected lane issues) =====================
            const int t = warp - 17;
            if (t == 0 || tile1_live) {
                const bool leader = ptx::elect_one();
                const uint32_t t_s = tmem + kColS + t * kBN, t_o = tmem + kColO + t * kON, t_p = tmem + kColP + t * kPH;
                const uint32_t a_q = sb + offsetof(Smem, q) + kTileBytes * t, a_k = sb + offsetof(Smem, k), a_v = sb + offsetof(Smem, v);
                const uint32_t a_ones = sb + offsetof(Smem, ones);
                const uint32_t a_s_full = sb + offsetof(Smem, s_full) + 8 * t, a_s_free = sb + offsetof(Smem, s_free) + 8 * t;
                const uint32_t a_p_full = sb + offsetof(Smem, p_full) + 8 * t, a_pv_done = sb + offsetof(Smem, pv_done) + 8 * t;
                ptx::mbar_wait(sb + offsetof(Smem, q_full), 0);
                ptx::mbar_wait(sb + offsetof(Smem, k_full), 0);
                ptx::tc_fence_after();
                if (leader) {
                    issue_qk(t_s, a_q, a_k);
                    ptx::mma_commit(a_s_full);
                    ptx::mma_commit(sb + offsetof(Smem, k_empty));
                }
                for (int j = 0; j < n_kv; ++j) {
                    const int st = j % kStages;
                    if (j + 1 < n_kv) {
                        // S(j+1) as soon as both halves' warps hold S(j) in registers
                        const int st1 = (j + 1) % kStages;
                        ptx::mbar_wait(a_s_free, j & 1);
                        ptx::mbar_wait(sb + offsetof(Smem, k_full) + 8 * st1, ((j + 1) / kStages) & 1);
                        ptx::tc_fence_after();
                        if (leader) {
                            issue_qk(t_s, a_q, a_k + kTileBytes * st1);
                            ptx::mma_commit(a_s_full);
                            ptx::mma_commit(sb + offsetof(Smem, k_empty) + 8 * st1);
                        }
                    }
                    ptx::mbar_wait(sb + offsetof(Smem, v_full) + 8 * st, (j / kStages) & 1);
                    const uint32_t v_st = a_v + kTileBytes * st;
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        ptx::mbar_wait(a_p_full + 8 * kQTiles * h, j & 1);
                        ptx::tc_fence_after();
                        if (leader) {
                            issue_pv_half(t_o, t_p, v_st + h * (kTileBytes / 2), a_ones - v_st, j > 0 || h > 0);
                            ptx::mma_commit(a_pv_done + 8 * kQTiles * h);
                        }
                    }
                    if (leader) ptx::mma_commit(sb + offsetof(Smem, v_empty) + 8 * st);
                }
                __syncwarp();
            }
        } else if (lane == 0) {
            ptx::watchdog(&sm.roles_done);            // warp 19: traps if the 19 role warps do not finish within seconds
        }
        if (warp <= 18 && lane == 0) ptx::mbar_arrive(&sm.roles_done);
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 104;");
        // ===================== softmax warps: tile `tile`, keys 64 half .. 64 half + 63 of every KV tile =====================
        if (tile == 0 || tile1_live) {
            const uint32_t lane_addr = static_cast<uint32_t>((warp & 3) * 32) << 16;
            const uint32_t t_s = tmem + lane_addr + kColS + tile * kBN + 64 * half;
            const uint32_t t_o = tmem + lane_addr + kColO + tile * kON;
            const uint32_t t_p = tmem + lane_addr + kColP + tile * kPH;
            const uint64_t scale2 = ptx::pack2(prm.scale_log2, prm.scale_log2);
            const uint64_t neg_m2 = ptx::pack2(-m_used, -m_used);
            const uint64_t magic_minus_m2 = ptx::pack2(12582912.0f - m_used, 12582912.0f - m_used);       // (m_used is an integer)
            const uint32_t a_s_full = sb + offsetof(Smem, s_full) + 8 * tile, a_s_free = sb + offsetof(Smem, s_free) + 8 * tile;
            const uint32_t a_p_full = sb + offsetof(Smem, p_full) + 8 * tile + 8 * kQTiles * half;
            // the P buffer is free once the P V of the OTHER half, issued just before this half's, has completed
            const uint32_t a_prev_done = sb + offsetof(Smem, pv_done) + 8 * tile + 8 * kQTiles * (half ^ 1);
            // One KV tile.  `tail` = -1: every key exists; else the number (0, 1, 2) of this half's 32-key chunks that hold keys
            // (ragged last tile): those are masked and exponentiated as in attention.cu, the others stored as zeros.
            auto kv_tile = [&](const int j, auto tail) {
                constexpr bool kMasked = decltype(tail)::value >= 0;
                constexpr int kChunks = kMasked ? decltype(tail)::value : 2;
                ptx::mbar_wait(a_s_full, j & 1);
                ptx::tc_fence_after();
                uint32_t s[2][32];
#pragma unroll
                for (int c = 0; c < kChunks; ++c) ptx::tmem_ld32(t_s + 32 * c, s[c]);
                ptx::tc_wait_ld();
                ptx::tc_fence_before();
                __syncwarp();
#ifdef MF_TEST_PROTOCOL_BUG      // test builds only (tests/test_gpu_watchdog.py): CTA 0 never hands S back, so its pipeline stalls for good
                if (lane == 0 && blockIdx.x != 0) ptx::mbar_arrive(a_s_free);
#else
                if (lane == 0) ptx::mbar_arrive(a_s_free);               // S columns may be overwritten by S(j+1)
#endif
                if (kMasked) {
                    const int valid = prm.seq_len - j * kBN - 64 * half;       // keys of this half that exist
#pragma unroll
                    for (int c = 0; c < kChunks; ++c)
#pragma unroll
                        for (int i = 0; i < 32; ++i)
                            if (32 * c + i >= valid) s[c][i] = 0xff800000u;      // -inf
                }
#pragma unroll
                for (int c = 0; c < kChunks; ++c) {
#pragma unroll
                    for (int i = 0; i < 32; i += 2) {
                        constexpr int kPolyPairs = MF_POLY_PAIRS_BOUND;
                        const bool poly = ((((i >> 1) & 15) * kPolyPairs) & 15) < kPolyPairs;
                        if (poly && !kMasked) {
                            exp2_poly2_bounded(s[c][i], s[c][i + 1], scale2, magic_minus_m2);
                            continue;
                        }
                        ptx::ffma2(s[c][i], s[c][i + 1], scale2, neg_m2);
                        if (poly) {
                            exp2_poly2(s[c][i], s[c][i + 1]);
                        } else {
                            s[c][i] = __float_as_uint(ptx::ex2(__uint_as_float(s[c][i])));
                            s[c][i + 1] = __float_as_uint(ptx::ex2(__uint_as_float(s[c][i + 1])));
                        }
                    }
                }
                uint32_t pk[32];
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    pk[i] = 0 < kChunks ? ptx::pack_bf16(__uint_as_float(s[0][2 * i]), __uint_as_float(s[0][2 * i + 1])) : 0u;
                    pk[16 + i] = 1 < kChunks ? ptx::pack_bf16(__uint_as_float(s[1][2 * i]), __uint_as_float(s[1][2 * i + 1])) : 0u;
                }
                if (half == 1) ptx::mbar_wait(a_prev_done, j & 1);
                else if (j > 0) ptx::mbar_wait(a_prev_done, (j - 1) & 1);
                ptx::tc_fence_after();
                ptx::tmem_st32(t_p, pk);
                ptx::tc_wait_st();
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(a_p_full);
            };
            for (int j = 0; j + 1 < n_kv; ++j) kv_tile(j, std::integral_constant<int, -1>{});
            {
                // (a ragged last tile takes the masked instantiation in BOTH halves, even where a half's 64 keys all exist: its
                // FMA-pipe exponentials are then the clamped form attention.cu uses on that tile, bit for bit)
                const int valid = prm.seq_len - (n_kv - 1) * kBN - 64 * half;          // this half's keys in the last tile (may be <= 0)
                if (prm.seq_len % kBN == 0) kv_tile(n_kv - 1, std::integral_constant<int, -1>{});
                else if (valid > 32) kv_tile(n_kv - 1, std::integral_constant<int, 2>{});
                else if (valid > 0) kv_tile(n_kv - 1, std::integral_constant<int, 1>{});
                else kv_tile(n_kv - 1, std::integral_constant<int, 0>{});
            }
            // ---- epilogue: O / l -> bf16 -> global; this half's warps take output columns 32 half .. 32 half + 31 ----
            ptx::mbar_wait(sb + offsetof(Smem, pv_done) + 8 * tile + 8 * kQTiles, (n_kv - 1) & 1);
            ptx::tc_fence_after();
            const int row = row0 + tile * kBM + row_in_tile;
            uint32_t o[32];
            ptx::tmem_ld32(t_o + 32 * half, o);
            const float l = __uint_as_float(ptx::tmem_ld1(t_o + kD));           // row sum from the ones column
            ptx::tc_wait_ld();
            const float inv_l = 1.0f / l;
            if (row < prm.seq_len) {
                const size_t tok = static_cast<size_t>(seq) * prm.seq_len + row;
                uint4* dst = reinterpret_cast<uint4*>(prm.out + (tok * prm.heads + head) * kD) + 4 * half;
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    uint4 w;
                    w.x = ptx::pack_bf16(__uint_as_float(o[8 * i + 0]) * inv_l, __uint_as_float(o[8 * i + 1]) * inv_l);
                    w.y = ptx::pack_bf16(__uint_as_float(o[8 * i + 2]) * inv_l, __uint_as_float(o[8 * i + 3]) * inv_l);
                    w.z = ptx::pack_bf16(__uint_as_float(o[8 * i + 4]) * inv_l, __uint_as_float(o[8 * i + 5]) * inv_l);
                    w.w = ptx::pack_bf16(__uint_as_float(o[8 * i + 6]) * inv_l, __uint_as_float(o[8 * i + 7]) * inv_l);
                    dst[i] = w;
                }
                if (prm.lse && half == 0) {
                    const int win = seq / prm.lse_frames, frame = seq - win * prm.lse_frames;
                    prm.lse[(static_cast<size_t>(win) * prm.heads + head) * prm.lse_frames * prm.seq_len +
                            static_cast<size_t>(frame) * prm.seq_len + row] = (m_used + log2f(l)) * 0.6931471805599453f;
                }
            }
        }
        if (lane == 0) ptx::mbar_arrive(&sm.roles_done);
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 17) ptx::tmem_dealloc(tmem, kTmemCols);
}

}  // namespace split

mf_status launch_attention_split(const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv, long long grid,
                                 const AttnParams& prm, uint32_t* exact_flags, cudaStream_t stream) {
    using namespace split;
    const int smem = static_cast<int>(sizeof(Smem)) + 1024;
    {   // the opt-in shared-memory size is a per-device attribute of the kernel: set it once per device
        static std::atomic<bool> attr_set[64];
        int dev = 0;
        MF_CUDA_OK(cudaGetDevice(&dev));
        if (dev < 0 || dev >= 64 || !attr_set[dev].load(std::memory_order_acquire)) {
            MF_CUDA_OK(cudaFuncSetAttribute(window_attention_split_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            if (dev >= 0 && dev < 64) attr_set[dev].store(true, std::memory_order_release);
        }
    }
    window_attention_split_kernel<<<static_cast<unsigned>(grid), kThreads, smem, stream>>>(mq, mk, mv, prm, exact_flags);
    MF_CUDA_OK(cudaGetLastError());
    return MF_OK;
}

}  // namespace mf
