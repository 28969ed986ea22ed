// mf_window_attention: flash-style bf16 self-attention for sm_100a (BJ north_star, kernels 1 and 2).
//
// One CTA owns 256 query rows of one (sequence, head) as two 128-row tiles.  Roles:
//   warps 0-3  softmax warpgroup for Q tile 0 (one thread per query row, TMEM lane = row)
//   warps 4-7  softmax warpgroup for Q tile 1
//   warp  8    TMA producer: Q once, then K/V tiles (128 keys x 64, SWIZZLE_128B) through a ring
//   warp  9    tcgen05.mma issuer for Q tile 0 (the whole warp runs the loop, one elected lane issues)
//   warp 10    tcgen05.mma issuer for Q tile 1 (warp 11: the watchdog; it exists so setmaxnreg can move registers)
// TMEM (480 of 512 columns): S0 [0,128) S1 [128,256) O0 [256,336) O1 [336,416) P0 [416,448) P1 [448,480).
// Per KV tile j and Q tile t:  S_t(j) = Q_t K(j)^T  ->  softmax warpgroup t loads S_t(j) into registers and
// immediately hands the S columns back (s_free), so S_t(j+1) is computed while the warpgroup is still
// exponentiating tile j;  P_t(j) (bf16) goes to its own TMEM columns in two 64-key halves and
// O_t += P_t(j) V(j) reads it from there, half by half.  V is extended by a constant "ones" column (a second
// MN-major atom in shared memory), so column 64 of O accumulates l = sum_j p_j on the tensor core from the
// same bf16 weights: O/l is an exact convex combination of V rows whatever the rounding of P.
// The softmax warps therefore never wait for the tensor core in steady state: the exponent unit (MUFU, 16/clk/SM)
// is the binding resource at head_dim 64, and a fixed share of the exponentials is evaluated on the FMA pipe
// instead (Cody-Waite split + cubic, relative error 7.5e-5, invisible after rounding P to bf16).
// Online softmax in fp32 with lazy rescaling (O and l are rescaled only when the running maximum grew by more
// than 2^8); O is normalised by 1/l in the epilogue.  FRAME mode is GLOBAL mode on the same bytes viewed as
// [windows*W, P, H, D].
// Long sequences (32 KV tiles and more) first get max |k|^2 per (sequence, head) from key_norm_max_kernel; warps whose rows'
// Cauchy-Schwarz score bound is small subtract that bound instead of a running maximum ("Score bound" in the softmax code), and
// CTAs in which EVERY row is so bounded are done by window_attention_split_kernel (attention_split.cu: four softmax warps per
// scheduler), this kernel taking only the CTAs flagged by it (AttnParams::only_flagged).  Shorter sequences: attention_clc.cu.
#include "common.h"
#include "sm100_ptx.cuh"
#include "tensormap.h"
#include "attention_common.cuh"

#include <cuda_bf16.h>

#include <algorithm>
#include <atomic>
#include <cstddef>
#include <mutex>
#include <type_traits>

namespace mf {

constexpr int kD = 64;                 // head_dim
constexpr int kBM = 128;               // query rows per tile (UMMA M)
constexpr int kBN = 128;               // keys per KV tile (UMMA N of QK^T, K extent of PV)
constexpr int kQTiles = 2;             // Q tiles per CTA
constexpr int kStages = 4;             // K and V ring depth
constexpr int kTileBytes = kBM * kD * 2;           // 16 KB, also the K/V tile size
constexpr int kThreads = 384;          // 2 softmax warpgroups + 1 warpgroup holding the TMA and MMA warps
constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kColS = 0, kColO = 256, kColP = 416;
constexpr int kON = 80;                // PV accumulator columns: 64 outputs + column 64 = row sum l (+15 unused)
constexpr int kPH = 32;                // TMEM columns of one P half (64 keys, bf16)
constexpr float kRescaleThreshold = 8.0f;
constexpr float kScoreBoundMax = 32.0f;    // log2 units: the score-bound path is taken for rows with |q| max|k| scale log2(e) <= 32 (22 nats)
#ifndef MF_POLY_PAIRS_BOUND
#define MF_POLY_PAIRS_BOUND 7          // the same on the score-bound path (attention_split.cu: 4 .. 8 of 16 give 989 / 998 / 1014 / 1021 / 1022 TFLOP/s; this kernel alone: best at 6)
#endif
#ifndef MF_PERSISTENT_BELOW_TILES
#define MF_PERSISTENT_BELOW_TILES 32   // sequences of fewer KV tiles (S <= 3968) run on the persistent kernel (attention_clc.cu); with the score-bound path here, S = 6216 gains 4 % on this kernel, S = 1024 loses 19 %
#endif
constexpr int kPersistentBelowTiles = MF_PERSISTENT_BELOW_TILES;

struct AttnSmem {
    alignas(1024) uint8_t q[kQTiles][kTileBytes];
    alignas(1024) uint8_t k[kStages][kTileBytes];
    alignas(1024) uint8_t v[kStages][kTileBytes];
    alignas(1024) uint8_t ones[kTileBytes];          // [128 keys][64]: column 0 = 1.0, rest 0 (swizzled like V)
    alignas(8) uint64_t q_full;
    uint64_t k_full[kStages], k_empty[kStages], v_full[kStages], v_empty[kStages];
    uint64_t s_full[kQTiles], s_free[kQTiles], p_full[2][kQTiles], pv_done[2][kQTiles];   // [half][tile]
    uint64_t roles_done;   // arrivals: the 11 role warps when they leave their loops (watchdog, sm100_ptx.cuh)
    uint32_t tmem_base;
    uint32_t zero;     // always 0 (see the softmax loop)
};

constexpr uint32_t kIdescQK = ptx::idesc_bf16_f32(kBM, kBN, 0, 0);
constexpr uint32_t kIdescPV = ptx::idesc_bf16_f32(kBM, kON, 0, 1);      // V is MN-major ([keys][d], d contiguous)

// S[tile] = Q[tile] K^T : 4 MMAs of K=16 (32-byte steps inside the 128-byte swizzle atom)
__device__ __forceinline__ void issue_qk(uint32_t tmem_s, uint32_t q, uint32_t k) {          // q, k: shared-memory addresses
    const uint64_t qd = ptx::smem_desc_sw128(q);
    const uint64_t kd = ptx::smem_desc_sw128(k);
#pragma unroll
    for (int i = 0; i < kD / 16; ++i) ptx::mma_ss(tmem_s, qd + 2 * i, kd + 2 * i, kIdescQK, i > 0);
}
// O[tile] (+)= P_half[tile] V_half : 4 MMAs of K=16 keys; P slice = 8 TMEM columns, V slice = 16 rows = 2048 B
// v_half points at the first of the 64 key rows.  B = [V | ones]: atom 0 = the V rows, atom 1 (columns 64..79) =
// the same rows of the ones tile, LBO bytes further on.
__device__ __forceinline__ void issue_pv_half(uint32_t tmem_o, uint32_t tmem_p, uint32_t v_half, uint32_t ones_minus_v,
                                              bool accumulate) {
    const uint64_t vd = ptx::smem_desc_sw128(v_half, ones_minus_v);
#pragma unroll
    for (int i = 0; i < kBN / 32; ++i)
        ptx::mma_ts(tmem_o, tmem_p + 8 * i, vd + (2048 >> 4) * i, kIdescPV, (accumulate || i > 0) ? 1u : 0u);
}

__global__ void __launch_bounds__(kThreads, 1)
window_attention_kernel(const __grid_constant__ CUtensorMap map_q, const __grid_constant__ CUtensorMap map_k,
                        const __grid_constant__ CUtensorMap map_v, const AttnParams prm) {
    extern __shared__ uint8_t smem_raw[];
    AttnSmem& sm = *reinterpret_cast<AttnSmem*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    // The warp number passes through a shuffle so that the compiler knows it is warp-uniform: role dispatch, tile index, TMEM
    // and barrier addresses then live in uniform registers, and the single-lane issue of TMA / tcgen05 instructions needs no
    // per-instruction loop over "active lanes" (measured on the campus launch: MMA issuers +1.3 %, producer +1.0 %, softmax
    // warps +2.2 %).
    const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;
    if (prm.only_flagged != nullptr && prm.only_flagged[blockIdx.x] == 0u) return;      // done by window_attention_split_kernel

    // work item: q block fastest so that concurrently running CTAs share one head's K/V in L2
    const int qb = blockIdx.x % prm.q_blocks;
    const int head = (blockIdx.x / prm.q_blocks) % prm.heads;
    const int seq = blockIdx.x / (prm.q_blocks * prm.heads);
    const int row0 = qb * (kQTiles * kBM);
    const bool tile1_live = row0 + kBM < prm.seq_len;
    const int n_kv = (prm.seq_len + kBN - 1) / kBN;

    if (warp == 8 && lane == 0) {
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
            ptx::mbar_init(&sm.s_free[t], 4);              // one arrival per softmax warp
            for (int h = 0; h < 2; ++h) {
                ptx::mbar_init(&sm.p_full[h][t], 4);
                ptx::mbar_init(&sm.pv_done[h][t], 1);
            }
        }
        sm.zero = 0;
        ptx::mbar_init(&sm.roles_done, 11);
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
    if (warp == 9) ptx::tmem_alloc(&sm.tmem_base, kTmemCols);
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = __shfl_sync(0xffffffffu, sm.tmem_base, 0);       // (uniform, as above)

    // register split: 168/thread at launch -> 224 for the softmax warpgroups, 56 for the rest (232 / 40 measured 0.7 % slower, 216 / 72 and 208 / 88 slower still)
    if (warp >= 8) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        if (warp == 8) {
            // ===================== TMA producer (whole warp in the loop, one elected lane issues) =====================
            const bool leader = ptx::elect_one();
            const uint32_t sb = ptx::smem_u32(&sm);
            const uint32_t a_q_full = sb + offsetof(AttnSmem, q_full);
            if (leader) {
                ptx::mbar_arrive_expect_tx(a_q_full, (tile1_live ? 2 : 1) * kTileBytes);
                ptx::tma_load_4d(sb + offsetof(AttnSmem, q), &map_q, a_q_full, 0, head, row0, seq);
                if (tile1_live) ptx::tma_load_4d(sb + offsetof(AttnSmem, q) + kTileBytes, &map_q, a_q_full, 0, head, row0 + kBM, seq);
            }
            for (int j = 0; j < n_kv; ++j) {
                const int st = j % kStages;
                const uint32_t ph = (j / kStages) & 1;
                ptx::mbar_wait(sb + offsetof(AttnSmem, k_empty) + 8 * st, ph ^ 1);
                if (leader) {
                    ptx::mbar_arrive_expect_tx(sb + offsetof(AttnSmem, k_full) + 8 * st, kTileBytes);
                    ptx::tma_load_4d(sb + offsetof(AttnSmem, k) + kTileBytes * st, &map_k, sb + offsetof(AttnSmem, k_full) + 8 * st, 0, head, j * kBN, seq);
                }
                ptx::mbar_wait(sb + offsetof(AttnSmem, v_empty) + 8 * st, ph ^ 1);
                if (leader) {
                    ptx::mbar_arrive_expect_tx(sb + offsetof(AttnSmem, v_full) + 8 * st, kTileBytes);
                    ptx::tma_load_4d(sb + offsetof(AttnSmem, v) + kTileBytes * st, &map_v, sb + offsetof(AttnSmem, v_full) + 8 * st, 0, head, j * kBN, seq);
                }
            }
            __syncwarp();
        } else if (warp <= 10) {
            // ===================== MMA issuers (warp 9: Q tile 0, warp 10: Q tile 1) =====================
            // The whole warp runs the loop (warp-uniform control flow, so descriptors and addresses live in uniform registers);
            // one elected lane issues the MMAs and commits.
            const int t = warp - 9;
            if (t == 0 || tile1_live) {
                const bool leader = ptx::elect_one();
                const uint32_t t_s = tmem + kColS + t * kBN, t_o = tmem + kColO + t * kON, t_p = tmem + kColP + t * kPH;
                const uint32_t sb = ptx::smem_u32(&sm);
                const uint32_t a_q = sb + offsetof(AttnSmem, q) + kTileBytes * t, a_k = sb + offsetof(AttnSmem, k), a_v = sb + offsetof(AttnSmem, v);
                const uint32_t a_ones = sb + offsetof(AttnSmem, ones);
                const uint32_t a_s_full = sb + offsetof(AttnSmem, s_full) + 8 * t, a_s_free = sb + offsetof(AttnSmem, s_free) + 8 * t;
                const uint32_t a_p_full = sb + offsetof(AttnSmem, p_full) + 8 * t, a_pv_done = sb + offsetof(AttnSmem, pv_done) + 8 * t;
                ptx::mbar_wait(sb + offsetof(AttnSmem, q_full), 0);
                ptx::mbar_wait(sb + offsetof(AttnSmem, k_full), 0);
                ptx::tc_fence_after();
                if (leader) {
                    issue_qk(t_s, a_q, a_k);
                    ptx::mma_commit(a_s_full);
                    ptx::mma_commit(sb + offsetof(AttnSmem, k_empty));
                }
                for (int j = 0; j < n_kv; ++j) {
                    const int st = j % kStages;
                    if (j + 1 < n_kv) {
                        const int st1 = (j + 1) % kStages;
                        ptx::mbar_wait(a_s_free, j & 1);
                        ptx::mbar_wait(sb + offsetof(AttnSmem, k_full) + 8 * st1, ((j + 1) / kStages) & 1);
                        ptx::tc_fence_after();
                        if (leader) {
                            issue_qk(t_s, a_q, a_k + kTileBytes * st1);
                            ptx::mma_commit(a_s_full);
                            ptx::mma_commit(sb + offsetof(AttnSmem, k_empty) + 8 * st1);
                        }
                    }
                    ptx::mbar_wait(sb + offsetof(AttnSmem, v_full) + 8 * st, (j / kStages) & 1);
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
                    if (leader) ptx::mma_commit(sb + offsetof(AttnSmem, v_empty) + 8 * st);
                }
                __syncwarp();
            }
        } else if (lane == 0) {
            ptx::watchdog(&sm.roles_done);            // warp 11: traps if the 11 role warps do not finish within seconds
        }
        if (warp <= 10 && lane == 0) ptx::mbar_arrive(&sm.roles_done);
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 224;");
        // ===================== softmax warpgroups =====================
        const int tile = warp >> 2;                       // 0 or 1
        if (tile == 0 || tile1_live) {
            const int row_in_tile = (warp & 3) * 32 + lane;
            const uint32_t lane_addr = static_cast<uint32_t>((warp & 3) * 32) << 16;
            const uint32_t t_s = tmem + lane_addr + kColS + tile * kBN;
            const uint32_t t_o = tmem + lane_addr + kColO + tile * kON;
            const uint32_t t_p = tmem + lane_addr + kColP + tile * kPH;
            float m_used = -INFINITY;                     // running max in scaled log2 units
            const uint64_t scale2 = ptx::pack2(prm.scale_log2, prm.scale_log2);
            // barrier addresses = one opaque base register + constants (see smem_base_u32)
            const uint32_t sb = ptx::smem_base_u32(&sm);
            const uint32_t a_s_full = sb + offsetof(AttnSmem, s_full) + 8 * tile, a_s_free = sb + offsetof(AttnSmem, s_free) + 8 * tile;
            const uint32_t a_p_full0 = sb + offsetof(AttnSmem, p_full) + 8 * tile, a_p_full1 = a_p_full0 + 8 * kQTiles;
            const uint32_t a_pv_done0 = sb + offsetof(AttnSmem, pv_done) + 8 * tile, a_pv_done1 = a_pv_done0 + 8 * kQTiles;
            // One KV tile.  The loop below runs it without the tail-masking code (hundreds of selects that only a ragged LAST tile
            // needs: peeled off, the steady-state loop is one contiguous block of code); the last tile picks its instantiation:
            // `tail` = 0 for a full tile, else the number of 32-column chunks of S that hold keys.  The other chunks are neither
            // read nor exponentiated and their P is stored as zeros (at P = 777 the seventh tile of a frame holds 9 keys: a
            // quarter of the softmax work of a full tile; FRAME mode +5.5 %).  The MMA issuers do not know about it: narrowing
            // the tail's Q K^T and P V too was measured, and the extra selects and predicates in the issuing thread cost the
            // steady state 2 % (campus) to 4 % (suburban), for no gain on the tail.
            auto kv_tile = [&](const int j, auto tail, auto bounded_tag) {
                constexpr bool kBounded = decltype(bounded_tag)::value;          // m_used is the row's score bound: no maximum, no rescaling
                constexpr bool kMasked = decltype(tail)::value != 0;
                constexpr int kChunks = kMasked ? decltype(tail)::value : 4;
                ptx::mbar_wait(a_s_full, j & 1);
                ptx::tc_fence_after();
                uint32_t s[4][32];
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
                const int valid = prm.seq_len - j * kBN;  // keys of this tile that exist
                if (kMasked) {
#pragma unroll
                    for (int c = 0; c < kChunks; ++c)
#pragma unroll
                        for (int i = 0; i < 32; ++i)
                            if (32 * c + i >= valid) s[c][i] = 0xff800000u;      // -inf
                    // (MUFU lanes turn -inf into an exact 0; the polynomial lanes clamp to 2^-125.  Either way the key
                    // adds nothing to O: TMA zero-fills the V rows past the sequence end (FLOAT_OOB_FILL_NONE), and it
                    // adds at most 2^-125 per key to the row sum l >= 1.  Zeroing those words exactly was measured: a
                    // uniform branch with 96 selects on every tail tile costs 6 % in FRAME mode, for no change in O.)
                }
                if (!kBounded) {
                    float mx[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
                    for (int c = 0; c < kChunks; ++c)
#pragma unroll
                        for (int i = 0; i < 32; i += 8)
#pragma unroll
                            for (int a = 0; a < 4; ++a)
                                mx[a] = ptx::max3(mx[a], __uint_as_float(s[c][i + 2 * a]), __uint_as_float(s[c][i + 2 * a + 1]));
                    const float row_max = ptx::max3(fmaxf(mx[0], mx[1]), mx[2], mx[3]);
                    const float m_new = fmaxf(m_used, row_max * prm.scale_log2);
                    const bool grow = m_new > m_used + kRescaleThreshold;            // always true at j == 0
                    if (j == 0) {
                        m_used = m_new;
                    } else if (__any_sync(0xffffffffu, grow)) {
                        // O may only be touched once PV(j-1) has completed; PV(j) is not issued before p_full(j)
                        ptx::mbar_wait(a_pv_done1, (j - 1) & 1);
                        ptx::tc_fence_after();
                        const float alpha = grow ? ptx::ex2(m_used - m_new) : 1.0f;
                        if (grow) m_used = m_new;
                        const uint64_t alpha2 = ptx::pack2(alpha, alpha);
#pragma unroll
                        for (int c = 0; c < 2; ++c) {
                            uint32_t o[32];
                            ptx::tmem_ld32(t_o + 32 * c, o);
                            ptx::tc_wait_ld();
#pragma unroll
                            for (int i = 0; i < 32; i += 2) ptx::fmul2(o[i], o[i + 1], alpha2);
                            ptx::tmem_st32(t_o + 32 * c, o);
                        }
                        const float l_old = __uint_as_float(ptx::tmem_ld1(t_o + kD));
                        ptx::tc_wait_ld();
                        ptx::tmem_st1(t_o + kD, __float_as_uint(l_old * alpha));
                    }
                }
                const uint64_t neg_m2 = ptx::pack2(-m_used, -m_used);
                const uint64_t magic_minus_m2 = ptx::pack2(12582912.0f - m_used, 12582912.0f - m_used);       // (bound path: m_used is an integer)
                uint64_t scale_h = scale2;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
#pragma unroll
                    for (int c = 2 * h; c < 2 * h + 2 && c < kChunks; ++c) {
#pragma unroll
                        for (int i = 0; i < 32; i += 2) {
                            constexpr int kPolyPairs = kBounded ? MF_POLY_PAIRS_BOUND : MF_POLY_PAIRS;
                            const bool poly = ((((i >> 1) & 15) * kPolyPairs) & 15) < kPolyPairs;       // kPolyPairs of every 16 pairs, evenly spread
                            if (poly && kBounded && !kMasked) {           // straight from the raw scores (attention_common.cuh)
                                exp2_poly2_bounded(s[c][i], s[c][i + 1], scale_h, magic_minus_m2);
                                continue;
                            }
                            ptx::ffma2(s[c][i], s[c][i + 1], scale_h, neg_m2);
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
                        pk[i] = 2 * h < kChunks ? ptx::pack_bf16(__uint_as_float(s[2 * h][2 * i]), __uint_as_float(s[2 * h][2 * i + 1])) : 0u;
                        pk[16 + i] = 2 * h + 1 < kChunks ? ptx::pack_bf16(__uint_as_float(s[2 * h + 1][2 * i]), __uint_as_float(s[2 * h + 1][2 * i + 1])) : 0u;
                    }
                    // the P half buffer is free once the previous PV that read it has completed
                    if (h == 1) ptx::mbar_wait(a_pv_done0, j & 1);
                    else if (j > 0) ptx::mbar_wait(a_pv_done1, (j - 1) & 1);
                    ptx::tc_fence_after();
                    ptx::tmem_st32(t_p, pk);
                    ptx::tc_wait_st();
                    ptx::tc_fence_before();
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(h ? a_p_full1 : a_p_full0);
                    if (h == 0) {
                        // Keep the second half's exponentials behind the first half's store (ptxas would hoist them
                        // above it): their scale operand passes through an opaque shared-memory read of a zero word.
                        uint32_t z;
                        asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(z) : "r"(sb + static_cast<uint32_t>(offsetof(AttnSmem, zero))) : "memory");
                        scale_h = ptx::pack2(__uint_as_float(__float_as_uint(prm.scale_log2) | z),
                                             __uint_as_float(__float_as_uint(prm.scale_log2) | z));
                    }
                }
            };
            auto all_tiles = [&](auto bounded_tag) {
                for (int j = 0; j + 1 < n_kv; ++j) kv_tile(j, std::integral_constant<int, 0>{}, bounded_tag);
                const int tail_chunks = (prm.seq_len - (n_kv - 1) * kBN + 31) / 32;        // 1..4
                if (prm.seq_len % kBN == 0) kv_tile(n_kv - 1, std::integral_constant<int, 0>{}, bounded_tag);
                else if (tail_chunks == 1) kv_tile(n_kv - 1, std::integral_constant<int, 1>{}, bounded_tag);
                else if (tail_chunks == 2) kv_tile(n_kv - 1, std::integral_constant<int, 2>{}, bounded_tag);
                else kv_tile(n_kv - 1, std::integral_constant<int, 4>{}, bounded_tag);
            };
            // Score bound (Cauchy-Schwarz): every score of row i is at most |q_i| max_j |k_j|.  Softmax is invariant under the
            // choice of the subtracted constant, so when that bound is small enough that 2^(score - bound) stays far inside
            // the range of bf16 / fp32 (bound <= kScoreBoundMax: the largest weight of the row is then >= 2^-2*kScoreBoundMax),
            // the bound itself serves as the row's "maximum": no maximum over the scores, no rescaling of O, and nothing that an
            // exponential has to wait for (campus launch: +7.8 %).  The key norms come from a pass over K before this kernel
            // (key_norm_max_kernel); |q_i|^2 is summed from the row's 128 bytes in shared memory.  The decision is taken per
            // warp; rows with a larger bound (peaked logits), NaN or Inf anywhere in it take the exact online-softmax path.
            bool bounded = false;
            if (prm.key_norm2_max != nullptr) {
                ptx::mbar_wait(sb + offsetof(AttnSmem, q_full), 0);
                const uint4* q_row = reinterpret_cast<const uint4*>(sm.q[tile] + row_in_tile * (kD * 2));
                float qq = 0.f;
#pragma unroll
                for (int c = 0; c < 8; ++c) {             // (the swizzle permutes the row's eight 16-byte chunks: irrelevant to a sum)
                    const uint4 w = q_row[(c + lane) & 7];
                    const uint32_t u[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const float lo = __uint_as_float(u[i] << 16), hi = __uint_as_float(u[i] & 0xffff0000u);
                        qq = fmaf(lo, lo, fmaf(hi, hi, qq));
                    }
                }
                const float kk = prm.key_norm2_max[static_cast<size_t>(seq) * prm.heads + head];
                const float bound = sqrtf(qq * kk) * fabsf(prm.scale_log2) * (1.0f + 0x1p-10f);       // (slack: fp32 rounding of the sums and of S)
                bounded = __all_sync(0xffffffffu, bound <= kScoreBoundMax);
                if (bounded) m_used = ceilf(bound);         // an integer (exp2_poly2_bounded), at most kScoreBoundMax
            }
            if (bounded) all_tiles(std::true_type{});
            else all_tiles(std::false_type{});
            // ---- epilogue: O / l -> bf16 -> global ----
            ptx::mbar_wait(a_pv_done1, (n_kv - 1) & 1);
            ptx::tc_fence_after();
            const int row = row0 + tile * kBM + row_in_tile;
            uint32_t o[2][32];
            ptx::tmem_ld32(t_o, o[0]);
            ptx::tmem_ld32(t_o + 32, o[1]);
            const float l = __uint_as_float(ptx::tmem_ld1(t_o + kD));           // row sum from the ones column
            ptx::tc_wait_ld();
            const float inv_l = 1.0f / l;
            // Direct stores: a thread's own row is 128 contiguous bytes, but the rows of a warp are heads*128 bytes apart
            // (32 wavefronts per instruction, ~1 us per CTA).  That is 0.3 % of the 300-us CTAs this kernel is used for; the
            // short sequences, where it shows, go to the persistent kernel (attention_clc.cu), which stages the tile in
            // shared memory and sends it with one TMA store.  (A TMA-store epilogue here was measured: -0.45 % on the campus
            // window because the CTA has to outlive the TMA's read of shared memory, -0.6 % even as a branch never taken.)
            if (row < prm.seq_len) {
                const size_t tok = static_cast<size_t>(seq) * prm.seq_len + row;
                uint4* dst = reinterpret_cast<uint4*>(prm.out + (tok * prm.heads + head) * kD);
#pragma unroll
                for (int c = 0; c < 2; ++c)
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        uint4 w;
                        w.x = ptx::pack_bf16(__uint_as_float(o[c][8 * i + 0]) * inv_l, __uint_as_float(o[c][8 * i + 1]) * inv_l);
                        w.y = ptx::pack_bf16(__uint_as_float(o[c][8 * i + 2]) * inv_l, __uint_as_float(o[c][8 * i + 3]) * inv_l);
                        w.z = ptx::pack_bf16(__uint_as_float(o[c][8 * i + 4]) * inv_l, __uint_as_float(o[c][8 * i + 5]) * inv_l);
                        w.w = ptx::pack_bf16(__uint_as_float(o[c][8 * i + 6]) * inv_l, __uint_as_float(o[c][8 * i + 7]) * inv_l);
                        dst[4 * c + i] = w;
                    }
            }
            if (row < prm.seq_len) {
                if (prm.lse) {
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
    if (warp == 9) ptx::tmem_dealloc(tmem, kTmemCols);
}

// Pass over K before window_attention_kernel: out[sequence, head] = max over the tokens of |k|^2, as float bits (non-negative
// floats order like unsigned integers, so the maximum is an atomicMax and does not depend on the order of arrival; a NaN
// anywhere has the largest bits and survives: the attention kernel then takes its exact path).  K is [sequences, S, H, 64]
// bf16: a (token, head) row is eight 16-byte chunks, summed by eight neighbouring lanes.  HBM-bound: K is read once.
__global__ void __launch_bounds__(256)
key_norm_max_kernel(const uint4* __restrict__ k, uint32_t* __restrict__ out, long long rows_per_sequence, int heads) {
    extern __shared__ uint32_t head_max[];                 // [heads]
    for (int i = threadIdx.x; i < heads; i += blockDim.x) head_max[i] = 0u;
    __syncthreads();
    const uint4* base = k + static_cast<size_t>(blockIdx.y) * rows_per_sequence * 8;
    const long long chunks = rows_per_sequence * 8;         // (token, head) rows x 8
    const long long stride = static_cast<long long>(gridDim.x) * blockDim.x;
    constexpr int kUnroll = 4;
    for (long long g0 = static_cast<long long>(blockIdx.x) * blockDim.x + (threadIdx.x & ~31); g0 < chunks; g0 += kUnroll * stride) {
        uint4 w[kUnroll];
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) {
            const long long g = g0 + u * stride + (threadIdx.x & 31);
            w[u] = g < chunks ? __ldg(base + g) : make_uint4(0u, 0u, 0u, 0u);
        }
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) {
            const long long g = g0 + u * stride + (threadIdx.x & 31);
            const uint32_t x[4] = {w[u].x, w[u].y, w[u].z, w[u].w};
            float ss = 0.f;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const float lo = __uint_as_float(x[i] << 16), hi = __uint_as_float(x[i] & 0xffff0000u);
                ss = fmaf(lo, lo, fmaf(hi, hi, ss));
            }
            ss += __shfl_xor_sync(0xffffffffu, ss, 1);
            ss += __shfl_xor_sync(0xffffffffu, ss, 2);
            ss += __shfl_xor_sync(0xffffffffu, ss, 4);
            if ((threadIdx.x & 7) == 0 && g < chunks) atomicMax(&head_max[(g >> 3) % heads], __float_as_uint(ss));
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < heads; i += blockDim.x)
        if (head_max[i] != 0u) atomicMax(&out[static_cast<size_t>(blockIdx.y) * heads + i], head_max[i]);
}

}  // namespace mf

// ------------------------------------------------------------------------------------------------
// Host side: tensor maps (cached) + launch
// ------------------------------------------------------------------------------------------------
namespace mf {

// bf16 [sequences, seq_len, heads, 64] -> 4-D map (d, head, token, sequence), box = 64 x 1 x 128 x 1
static mf_status make_map(CUtensorMap* map, const void* base, int sequences, int seq_len, int heads) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return fail(MF_ERR_CUDA, "cuTensorMapEncodeTiled entry point not available");
    cuuint64_t dims[4] = {static_cast<cuuint64_t>(kD), static_cast<cuuint64_t>(heads), static_cast<cuuint64_t>(seq_len),
                          static_cast<cuuint64_t>(sequences)};
    cuuint64_t strides[3] = {static_cast<cuuint64_t>(kD) * 2, static_cast<cuuint64_t>(heads) * kD * 2,
                             static_cast<cuuint64_t>(seq_len) * heads * kD * 2};
    cuuint32_t box[4] = {kD, 1, kBM, 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(base), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(MF_ERR_CUDA, "cuTensorMapEncodeTiled failed (CUresult %d)", static_cast<int>(r));
    return MF_OK;
}

// Per-process tensor-map cache.  A map depends only on (base pointer, sequences, seq_len, heads): the
// layer stack of a window calls with the same q/k/v 24 times, a stream with the same static buffers for every window.
// Small direct-mapped table under a mutex; an entry is the encoded 128-byte map, so a hit is one compare and one copy.
struct MapKey {
    const void* base;
    int sequences, seq_len, heads;
    bool operator==(const MapKey& o) const { return base == o.base && sequences == o.sequences && seq_len == o.seq_len && heads == o.heads; }
};
static mf_status cached_map(CUtensorMap* out, const void* base, int sequences, int seq_len, int heads) {
    constexpr int kSlots = 64;
    static std::mutex mu;
    static MapKey keys[kSlots];
    static CUtensorMap maps[kSlots];
    static bool used[kSlots];
    const MapKey key{base, sequences, seq_len, heads};
    uint64_t h = reinterpret_cast<uintptr_t>(base) >> 8;
    h = (h ^ (h >> 17) ^ (static_cast<uint64_t>(seq_len) * 0x9E3779B97F4A7C15ull) ^ (static_cast<uint64_t>(sequences) << 7) ^ heads) % kSlots;
    {
        std::lock_guard<std::mutex> g(mu);
        if (used[h] && keys[h] == key) {
            *out = maps[h];
            return MF_OK;
        }
    }
    mf_status st = make_map(out, base, sequences, seq_len, heads);
    if (st != MF_OK) return st;
    std::lock_guard<std::mutex> g(mu);
    keys[h] = key;
    maps[h] = *out;
    used[h] = true;
    return MF_OK;
}

// Stream-ordered workspace for the score bound ([sequences, heads] floats): allocated and freed on the caller's stream from a
// pool of the library's own (cudaMallocFromPoolAsync: no synchronisation, safe with concurrent callers on other streams and
// inside stream capture, where it becomes a pair of graph nodes).  The pool keeps its memory between calls.
#ifndef MF_NO_SCORE_BOUND
static mf_status bound_workspace(uint32_t** p, size_t bytes, cudaStream_t stream) {
    static std::mutex mu;
    static cudaMemPool_t pools[64];
    static bool made[64];
    int dev = 0;
    MF_CUDA_OK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return fail(MF_ERR_UNSUPPORTED, "device ordinal %d", dev);
    cudaMemPool_t pool;
    {
        std::lock_guard<std::mutex> g(mu);
        if (!made[dev]) {
            cudaMemPoolProps props = {};
            props.allocType = cudaMemAllocationTypePinned;
            props.handleTypes = cudaMemHandleTypeNone;
            props.location.type = cudaMemLocationTypeDevice;
            props.location.id = dev;
            MF_CUDA_OK(cudaMemPoolCreate(&pools[dev], &props));
            uint64_t keep = ~0ull;
            MF_CUDA_OK(cudaMemPoolSetAttribute(pools[dev], cudaMemPoolAttrReleaseThreshold, &keep));
            made[dev] = true;
        }
        pool = pools[dev];
    }
    MF_CUDA_OK(cudaMallocFromPoolAsync(reinterpret_cast<void**>(p), bytes, pool, stream));
    return MF_OK;
}
#endif

}  // namespace mf

extern "C" mf_status mf_window_attention(const void* q, const void* k, const void* v, void* out, float* lse,
                                         int windows, int frames_per_window, int tokens_per_frame, int heads,
                                         int head_dim, mf_attn_mode mode, float softmax_scale, void* stream) {
    using namespace mf;
    if (!q || !k || !v || !out) return fail(MF_ERR_INVALID_ARG, "mf_window_attention: NULL tensor");
    if (windows < 1 || frames_per_window < 1 || tokens_per_frame < 1 || heads < 1)
        return fail(MF_ERR_INVALID_ARG, "mf_window_attention: non-positive dimension");
    if (mode != MF_ATTN_GLOBAL && mode != MF_ATTN_FRAME)
        return fail(MF_ERR_INVALID_ARG, "mf_window_attention: bad mode %d", static_cast<int>(mode));
    if (head_dim != kD && head_dim != 128)
        return fail(MF_ERR_UNSUPPORTED, "mf_window_attention: head_dim=%d (64 and 128 are built)", head_dim);
    if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(out))
        return fail(MF_ERR_ALIGNMENT, "mf_window_attention: q/k/v/out must be 16-byte aligned");
    if (out == q || out == k || out == v) return fail(MF_ERR_INVALID_ARG, "mf_window_attention: out aliases an input");
    mf_status st = require_sm100();
    if (st != MF_OK) return st;

    // FRAME mode == GLOBAL mode on [windows*W, P, H, D] (same bytes)
    const long long sequences_ll = mode == MF_ATTN_FRAME ? static_cast<long long>(windows) * frames_per_window : windows;
    const long long seq_len_ll = mode == MF_ATTN_FRAME ? tokens_per_frame
                                                       : static_cast<long long>(frames_per_window) * tokens_per_frame;
    if (seq_len_ll > (1 << 24) || sequences_ll > (1 << 24))
        return fail(MF_ERR_UNSUPPORTED, "mf_window_attention: sequence length / count too large");
    const int sequences = static_cast<int>(sequences_ll), seq_len = static_cast<int>(seq_len_ll);
    if (static_cast<long long>((seq_len + 255) / 256) * heads * sequences > 0x7fffffffLL)
        return fail(MF_ERR_UNSUPPORTED, "mf_window_attention: grid too large");
    if (validate_only()) return MF_OK;

    AttnParams prm;
    prm.seq_len = seq_len;
    prm.heads = heads;
    prm.q_blocks = (seq_len + kQTiles * kBM - 1) / (kQTiles * kBM);
    const float scale = softmax_scale > 0.f ? softmax_scale : 1.0f / sqrtf(static_cast<float>(head_dim));
    prm.scale_log2 = scale * 1.4426950408889634f;
    prm.out = static_cast<__nv_bfloat16*>(out);
    prm.lse = lse;
    prm.lse_frames = mode == MF_ATTN_FRAME ? frames_per_window : 1;
    prm.key_norm2_max = nullptr;
    prm.only_flagged = nullptr;
    if (head_dim == 128)       // re-tiled variant (attention_d128.cu); q_blocks is the same: 256 query rows per CTA
        return launch_attention_d128(q, k, v, sequences, seq_len, heads, prm, static_cast<cudaStream_t>(stream));

    CUtensorMap mq, mk, mv, mo;
    if ((st = cached_map(&mo, out, sequences, seq_len, heads)) != MF_OK) return st;
    if ((st = cached_map(&mq, q, sequences, seq_len, heads)) != MF_OK) return st;
    if ((st = cached_map(&mk, k, sequences, seq_len, heads)) != MF_OK) return st;
    if ((st = cached_map(&mv, v, sequences, seq_len, heads)) != MF_OK) return st;
    const long long grid = static_cast<long long>(prm.q_blocks) * heads * sequences;
    const int smem = static_cast<int>(sizeof(AttnSmem)) + 1024;
    // short items: persistent kernel (cluster launch control; its grid is 3-D, so heads and sequences must fit a grid dimension)
    if ((seq_len + kBN - 1) / kBN < kPersistentBelowTiles && heads <= 65535 && sequences <= 65535)
        return launch_attention_clc(mq, mk, mv, mo, sequences, seq_len, heads, prm, static_cast<cudaStream_t>(stream));
    {   // the opt-in shared-memory size is a per-device attribute of the kernel: set it once per device
        static std::atomic<bool> attr_set[64];
        int dev = 0;
        MF_CUDA_OK(cudaGetDevice(&dev));
        if (dev < 0 || dev >= 64 || !attr_set[dev].load(std::memory_order_acquire)) {
            MF_CUDA_OK(cudaFuncSetAttribute(window_attention_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            if (dev >= 0 && dev < 64) attr_set[dev].store(true, std::memory_order_release);
        }
    }
    cudaStream_t cs = static_cast<cudaStream_t>(stream);
    uint32_t* bound_ws = nullptr;
#ifndef MF_NO_SCORE_BOUND          // (test builds: tests/test_gpu_attention_differential.py compares the exact paths of the two kernels bit for bit)
    if (heads <= 4096 && sequences <= 65535) {
        // the score bound's pass over K (window_attention_kernel: "Score bound"); 0.3 % of the attention launch at S = 24864
        // scratch: [sequences, heads] key norms, then one flag per CTA of the attention grid (attention_split.cu)
        const size_t norm_words = static_cast<size_t>(sequences) * heads;
        const bool split = grid <= (1LL << 24);          // (64 MB of flags at most; larger grids run window_attention_kernel alone)
        const size_t ws_bytes = (norm_words + (split ? static_cast<size_t>(grid) : 0)) * sizeof(uint32_t);
        if ((st = bound_workspace(&bound_ws, ws_bytes, cs)) != MF_OK) return st;
        MF_CUDA_OK(cudaMemsetAsync(bound_ws, 0, ws_bytes, cs));
        const long long rows = static_cast<long long>(seq_len) * heads;
        const long long want = (rows * 8 + 256 * 4 - 1) / (256 * 4);
        const long long cap = (8LL * sm_count() + sequences - 1) / sequences;
        const unsigned gx = static_cast<unsigned>(std::max(1LL, std::min(want, cap)));
        key_norm_max_kernel<<<dim3(gx, static_cast<unsigned>(sequences)), 256, heads * sizeof(uint32_t), cs>>>(
            static_cast<const uint4*>(k), bound_ws, rows, heads);
        MF_CUDA_OK(cudaGetLastError());
        prm.key_norm2_max = reinterpret_cast<const float*>(bound_ws);
#ifndef MF_NO_SPLIT
        // CTAs whose rows are all within the bound: four softmax warps per scheduler (attention_split.cu); the others are flagged
        // there and done by the launch below, which returns at once from the rest
        if (split) {
            if ((st = launch_attention_split(mq, mk, mv, grid, prm, bound_ws + norm_words, cs)) != MF_OK) return st;
            prm.only_flagged = bound_ws + norm_words;
        }
#else
        (void)split;
#endif
    }
#endif
    window_attention_kernel<<<static_cast<unsigned>(grid), kThreads, smem, cs>>>(mq, mk, mv, prm);
    MF_CUDA_OK(cudaGetLastError());
    if (bound_ws) MF_CUDA_OK(cudaFreeAsync(bound_ws, cs));
    return MF_OK;
}

// ------------------------------------------------------------------------------------------------
// mf_window_attention_noalloc: the same attention for callers that cannot allocate (include/mf.h)
// ------------------------------------------------------------------------------------------------
namespace mf {

// The score bound's scratch ([sequences, heads] floats, see key_norm_max_kernel) as a fixed array in the library's own
// device image instead of a stream-ordered allocation: 64 Ki entries = 256 KB, held by every GPU that loads the library
// until the process exits.  In host code `g_bound_scratch` is only a stand-in for the symbol, not a device address: the
// address comes from cudaGetSymbolAddress, once per device, with that device current (static_bound_scratch below).
constexpr int kStaticBoundEntries = 65536;
static __device__ __align__(256) uint32_t g_bound_scratch[kStaticBoundEntries];

static mf_status static_bound_scratch(uint32_t** p) {
    static std::atomic<uint32_t*> addr[64];
    int dev = 0;
    MF_CUDA_OK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return fail(MF_ERR_UNSUPPORTED, "device ordinal %d", dev);
    uint32_t* a = addr[dev].load(std::memory_order_acquire);
    if (!a) {
        void* sym = nullptr;
        MF_CUDA_OK(cudaGetSymbolAddress(&sym, g_bound_scratch));          // (this device's copy of the array)
        if (!sym) return fail(MF_ERR_CUDA, "cudaGetSymbolAddress returned NULL");
        a = static_cast<uint32_t*>(sym);
        addr[dev].store(a, std::memory_order_release);
    }
    *p = a;
    return MF_OK;
}

}  // namespace mf

extern "C" mf_status mf_window_attention_noalloc(const void* q, const void* k, const void* v, void* out, float* lse,
                                                 int windows, int frames_per_window, int tokens_per_frame, int heads,
                                                 int head_dim, mf_attn_mode mode, float softmax_scale, void* stream) {
    using namespace mf;
    mf_status st;
    {   // every argument check of mf_window_attention, nothing enqueued
        const bool outer_dry_run = validate_only();
        validate_only() = true;
        st = mf_window_attention(q, k, v, out, lse, windows, frames_per_window, tokens_per_frame, heads, head_dim, mode,
                                 softmax_scale, stream);
        validate_only() = outer_dry_run;
        if (st != MF_OK || outer_dry_run) return st;
    }
    const int sequences = mode == MF_ATTN_FRAME ? windows * frames_per_window : windows;
    const int seq_len = mode == MF_ATTN_FRAME ? tokens_per_frame : frames_per_window * tokens_per_frame;
    // head_dim 128 and the short sequences of the persistent kernel use no scratch memory: mf_window_attention allocates
    // nothing on those paths and is the entry point for them as it stands
    if (head_dim == 128 || ((seq_len + kBN - 1) / kBN < kPersistentBelowTiles && heads <= 65535 && sequences <= 65535))
        return mf_window_attention(q, k, v, out, lse, windows, frames_per_window, tokens_per_frame, heads, head_dim, mode,
                                   softmax_scale, stream);
    // long sequences, head_dim 64: window_attention_kernel with the score bound in the static array
    const long long entries = static_cast<long long>(sequences) * heads;
    if (entries > kStaticBoundEntries || heads > 4096)
        return fail(MF_ERR_UNSUPPORTED, "mf_window_attention_noalloc: sequences x heads = %lld exceeds the static scratch (%d entries); "
                    "use mf_window_attention", entries, kStaticBoundEntries);
    uint32_t* scratch = nullptr;
    if ((st = static_bound_scratch(&scratch)) != MF_OK) return st;

    AttnParams prm;
    prm.seq_len = seq_len;
    prm.heads = heads;
    prm.q_blocks = (seq_len + kQTiles * kBM - 1) / (kQTiles * kBM);
    const float scale = softmax_scale > 0.f ? softmax_scale : 1.0f / sqrtf(static_cast<float>(head_dim));
    prm.scale_log2 = scale * 1.4426950408889634f;
    prm.out = static_cast<__nv_bfloat16*>(out);
    prm.lse = lse;
    prm.lse_frames = mode == MF_ATTN_FRAME ? frames_per_window : 1;
    prm.key_norm2_max = reinterpret_cast<const float*>(scratch);
    prm.only_flagged = nullptr;
    CUtensorMap mq, mk, mv;
    if ((st = cached_map(&mq, q, sequences, seq_len, heads)) != MF_OK) return st;
    if ((st = cached_map(&mk, k, sequences, seq_len, heads)) != MF_OK) return st;
    if ((st = cached_map(&mv, v, sequences, seq_len, heads)) != MF_OK) return st;
    const long long grid = static_cast<long long>(prm.q_blocks) * heads * sequences;
    const int smem = static_cast<int>(sizeof(AttnSmem)) + 1024;
    {   // (per-device kernel attribute, as in mf_window_attention)
        static std::atomic<bool> attr_set[64];
        int dev = 0;
        MF_CUDA_OK(cudaGetDevice(&dev));
        if (dev < 0 || dev >= 64 || !attr_set[dev].load(std::memory_order_acquire)) {
            MF_CUDA_OK(cudaFuncSetAttribute(window_attention_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            if (dev >= 0 && dev < 64) attr_set[dev].store(true, std::memory_order_release);
        }
    }
    cudaStream_t cs = static_cast<cudaStream_t>(stream);
    // the array keeps the previous call's maxima: the entries this call uses start at zero again
    MF_CUDA_OK(cudaMemsetAsync(scratch, 0, static_cast<size_t>(entries) * sizeof(uint32_t), cs));
    const long long rows = static_cast<long long>(seq_len) * heads;
    const long long want = (rows * 8 + 256 * 4 - 1) / (256 * 4);
    const long long cap = (8LL * sm_count() + sequences - 1) / sequences;
    const unsigned gx = static_cast<unsigned>(std::max(1LL, std::min(want, cap)));
    key_norm_max_kernel<<<dim3(gx, static_cast<unsigned>(sequences)), 256, heads * sizeof(uint32_t), cs>>>(
        static_cast<const uint4*>(k), scratch, rows, heads);
    MF_CUDA_OK(cudaGetLastError());
#ifndef MF_NO_SPLIT
    // where the array also holds one flag per CTA behind the norms, the score-bound CTAs run on attention_split.cu as in
    // mf_window_attention (same results bit for bit either way)
    if (entries + grid <= kStaticBoundEntries) {
        MF_CUDA_OK(cudaMemsetAsync(scratch + entries, 0, static_cast<size_t>(grid) * sizeof(uint32_t), cs));
        if ((st = launch_attention_split(mq, mk, mv, grid, prm, scratch + entries, cs)) != MF_OK) return st;
        prm.only_flagged = scratch + entries;
    }
#endif
    window_attention_kernel<<<static_cast<unsigned>(grid), kThreads, smem, cs>>>(mq, mk, mv, prm);
    MF_CUDA_OK(cudaGetLastError());
    return MF_OK;
}
