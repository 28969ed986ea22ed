// mf_window_attention at head_dim 128: the head_dim 64 kernel of attention.cu re-tiled.
//
// Same roles (384 threads: two softmax warpgroups, one thread per query row; TMA warp; one MMA issuer per Q tile) and the
// same algorithm (online softmax in log2 units, lazy rescaling, P in TMEM as the A operand of O += P V, row sum from a
// constant "ones" column of V), but S (2 x 128 columns), O with the ones column (2 x 144) and P would need 608 TMEM columns
// with 128-key tiles, so KV tiles hold 64 keys:
//   TMEM (480 of 512): S0 [0,64) S1 [64,128)  O0 [128,272) O1 [272,416)  P0 [416,448) P1 [448,480)
// and a whole P tile (64 keys, bf16) is published at once.  A row of Q/K/V is 256 bytes = two 128-byte swizzle atoms:
// every tile is stored as a low and a high 64-column half (two TMA boxes).  QK^T runs 8 K=16 steps, 4 in each half.  For
// O += P [V_lo | V_hi | ones] (M=128, N=144, MN-major B) the three 64-column atoms of a stage lie 8 KB apart (LBO), which is why
// every V stage carries its own copy of the ones tile.
// Per 64 keys and CTA the tensor pipe has 1088 clk of work (QK 512, PV 576) against 1024 clk on the exponent unit:
// at head_dim 128 the tensor core, not MUFU, is the first pipe to saturate.
#include "attention_common.cuh"
#include "tensormap.h"

#include <atomic>
#include <cstddef>
#include <type_traits>

namespace mf {
namespace d128 {

constexpr int kD = 128;                // head_dim
constexpr int kDH = 64;                // columns per swizzle atom (128 bytes of bf16)
constexpr int kBM = 128;               // query rows per tile (UMMA M)
constexpr int kBN = 64;                // keys per KV tile
constexpr int kQTiles = 2;
constexpr int kStages = 3;
constexpr int kQHalfBytes = kBM * kDH * 2;         // 16 KB
constexpr int kKVHalfBytes = kBN * kDH * 2;        // 8 KB
constexpr int kThreads = 384;
constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kColS = 0, kColO = 128, kColP = 416;
constexpr int kON = kD + 16;           // PV accumulator columns: 128 outputs + column 128 = row sum l (+15 unused)
constexpr int kPCols = kBN / 2;        // TMEM columns of one P tile (64 keys, bf16)
constexpr float kRescaleThreshold = 8.0f;
#ifndef MF_POLY_PAIRS_D128
#define MF_POLY_PAIRS_D128 0           // of every 16 score pairs, this many are exponentiated on the FMA pipe (measured: 0 is best here)
#endif
constexpr int kPolyPairs = MF_POLY_PAIRS_D128;

struct VStage {                        // the three MN atoms of the PV B operand, LBO = 8 KB apart
    uint8_t lo[kKVHalfBytes], hi[kKVHalfBytes], ones[kKVHalfBytes];
};

struct Smem {
    alignas(1024) uint8_t q[kQTiles][2][kQHalfBytes];        // [tile][lo/hi]
    alignas(1024) uint8_t k[kStages][2][kKVHalfBytes];
    alignas(1024) VStage v[kStages];
    alignas(8) uint64_t q_full;
    uint64_t k_full[kStages], k_empty[kStages], v_full[kStages], v_empty[kStages];
    uint64_t s_full[kQTiles], s_free[kQTiles], p_full[kQTiles], pv_done[kQTiles];
    uint64_t roles_done;   // arrivals: the 11 role warps when they leave their loops (watchdog, sm100_ptx.cuh)
    uint32_t tmem_base;
};

constexpr uint32_t kIdescQK = ptx::idesc_bf16_f32(kBM, kBN, 0, 0);
constexpr uint32_t kIdescPV = ptx::idesc_bf16_f32(kBM, kON, 0, 1);

// S[tile] = Q[tile] K^T: 8 MMAs of K=16, four in each 64-column half (32-byte steps inside the swizzle atom)
__device__ __forceinline__ void issue_qk(uint32_t tmem_s, const uint8_t (*q)[kQHalfBytes], const uint8_t (*k)[kKVHalfBytes]) {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const uint64_t qd = ptx::smem_desc_sw128(ptx::smem_u32(q[h]));
        const uint64_t kd = ptx::smem_desc_sw128(ptx::smem_u32(k[h]));
#pragma unroll
        for (int i = 0; i < kDH / 16; ++i) ptx::mma_ss(tmem_s, qd + 2 * i, kd + 2 * i, kIdescQK, (h | i) != 0);
    }
}
// O[tile] (+)= P[tile] [V | ones]: 4 MMAs of K=16 keys; P slice = 8 TMEM columns, V slice = 16 rows = 2048 B
__device__ __forceinline__ void issue_pv(uint32_t tmem_o, uint32_t tmem_p, const VStage& v, bool accumulate) {
    const uint64_t vd = ptx::smem_desc_sw128(ptx::smem_u32(v.lo), kKVHalfBytes);
#pragma unroll
    for (int i = 0; i < kBN / 16; ++i)
        ptx::mma_ts(tmem_o, tmem_p + 8 * i, vd + (2048 >> 4) * i, kIdescPV, (accumulate || i > 0) ? 1u : 0u);
}

__global__ void __launch_bounds__(kThreads, 1)
window_attention_d128_kernel(const __grid_constant__ CUtensorMap map_q, const __grid_constant__ CUtensorMap map_k,
                             const __grid_constant__ CUtensorMap map_v, const AttnParams prm) {
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
            ptx::mbar_init(&sm.p_full[t], 4);
            ptx::mbar_init(&sm.pv_done[t], 1);
        }
        ptx::mbar_init(&sm.roles_done, 11);
        ptx::fence_barrier_init();
    }
    {   // ones atoms: logical (key r, column 0) = 1.0 under the 128-byte swizzle, everything else 0
        for (int s = 0; s < kStages; ++s) {
            uint4* o4 = reinterpret_cast<uint4*>(sm.v[s].ones);
            for (int i = threadIdx.x; i < kKVHalfBytes / 16; i += kThreads) {
                const int r = i >> 3, chunk = i & 7;
                o4[i] = make_uint4(chunk == (r & 7) ? 0x00003F80u : 0u, 0u, 0u, 0u);
            }
        }
        ptx::fence_proxy_async();
    }
    if (warp == 9) ptx::tmem_alloc(&sm.tmem_base, kTmemCols);
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = __shfl_sync(0xffffffffu, sm.tmem_base, 0);       // (uniform, as above)

    if (warp >= 8) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        if (warp == 8) {
            // ===================== TMA producer (whole warp in the loop, one elected lane issues) =====================
            const bool leader = ptx::elect_one();
            if (leader) {
                ptx::mbar_arrive_expect_tx(&sm.q_full, (tile1_live ? 4 : 2) * kQHalfBytes);
                for (int t = 0; t < (tile1_live ? 2 : 1); ++t)
                    for (int h = 0; h < 2; ++h)
                        ptx::tma_load_4d(sm.q[t][h], &map_q, &sm.q_full, h * kDH, head, row0 + t * kBM, seq);
            }
            for (int j = 0; j < n_kv; ++j) {
                const int st = j % kStages;
                const uint32_t ph = (j / kStages) & 1;
                ptx::mbar_wait(&sm.k_empty[st], ph ^ 1);
                if (leader) {
                    ptx::mbar_arrive_expect_tx(&sm.k_full[st], 2 * kKVHalfBytes);
                    ptx::tma_load_4d(sm.k[st][0], &map_k, &sm.k_full[st], 0, head, j * kBN, seq);
                    ptx::tma_load_4d(sm.k[st][1], &map_k, &sm.k_full[st], kDH, head, j * kBN, seq);
                }
                ptx::mbar_wait(&sm.v_empty[st], ph ^ 1);
                if (leader) {
                    ptx::mbar_arrive_expect_tx(&sm.v_full[st], 2 * kKVHalfBytes);
                    ptx::tma_load_4d(sm.v[st].lo, &map_v, &sm.v_full[st], 0, head, j * kBN, seq);
                    ptx::tma_load_4d(sm.v[st].hi, &map_v, &sm.v_full[st], kDH, head, j * kBN, seq);
                }
            }
            __syncwarp();
        } else if (warp <= 10) {
            // ===================== MMA issuers (warp 9: Q tile 0, warp 10: Q tile 1; one elected lane issues) =====================
            const int t = warp - 9;
            if (t == 0 || tile1_live) {
                const bool leader = ptx::elect_one();
                const uint32_t t_s = tmem + kColS + t * kBN, t_o = tmem + kColO + t * kON, t_p = tmem + kColP + t * kPCols;
                ptx::mbar_wait(&sm.q_full, 0);
                ptx::mbar_wait(&sm.k_full[0], 0);
                ptx::tc_fence_after();
                if (leader) {
                    issue_qk(t_s, sm.q[t], sm.k[0]);
                    ptx::mma_commit(&sm.s_full[t]);
                    ptx::mma_commit(&sm.k_empty[0]);
                }
                for (int j = 0; j < n_kv; ++j) {
                    const int st = j % kStages;
                    if (j + 1 < n_kv) {
                        // S(j+1) as soon as the softmax warpgroup holds S(j) in registers
                        const int st1 = (j + 1) % kStages;
                        ptx::mbar_wait(&sm.s_free[t], j & 1);
                        ptx::mbar_wait(&sm.k_full[st1], ((j + 1) / kStages) & 1);
                        ptx::tc_fence_after();
                        if (leader) {
                            issue_qk(t_s, sm.q[t], sm.k[st1]);
                            ptx::mma_commit(&sm.s_full[t]);
                            ptx::mma_commit(&sm.k_empty[st1]);
                        }
                    }
                    ptx::mbar_wait(&sm.v_full[st], (j / kStages) & 1);
                    ptx::mbar_wait(&sm.p_full[t], j & 1);
                    ptx::tc_fence_after();
                    if (leader) {
                        issue_pv(t_o, t_p, sm.v[st], j > 0);
                        ptx::mma_commit(&sm.pv_done[t]);
                        ptx::mma_commit(&sm.v_empty[st]);
                    }
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
        const int tile = warp >> 2;
        if (tile == 0 || tile1_live) {
            const int row_in_tile = (warp & 3) * 32 + lane;
            const uint32_t lane_addr = static_cast<uint32_t>((warp & 3) * 32) << 16;
            const uint32_t t_s = tmem + lane_addr + kColS + tile * kBN;
            const uint32_t t_o = tmem + lane_addr + kColO + tile * kON;
            const uint32_t t_p = tmem + lane_addr + kColP + tile * kPCols;
            float m_used = -INFINITY;                     // running max in scaled log2 units
            const uint64_t scale2 = ptx::pack2(prm.scale_log2, prm.scale_log2);
            // barrier addresses = one opaque base register + constants (sm100_ptx.cuh: smem_base_u32)
            const uint32_t sb = ptx::smem_base_u32(&sm);
            const uint32_t a_s_full = sb + offsetof(Smem, s_full) + 8 * tile, a_s_free = sb + offsetof(Smem, s_free) + 8 * tile;
            const uint32_t a_p_full = sb + offsetof(Smem, p_full) + 8 * tile, a_pv_done = sb + offsetof(Smem, pv_done) + 8 * tile;
            // One KV tile; the ragged last tile is peeled off the loop (the steady-state loop holds no tail-masking code).
            auto kv_tile = [&](const int j, auto masked) {
                ptx::mbar_wait(a_s_full, j & 1);
                ptx::tc_fence_after();
                uint32_t s[2][32];
                ptx::tmem_ld32(t_s, s[0]);
                ptx::tmem_ld32(t_s + 32, s[1]);
                ptx::tc_wait_ld();
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(a_s_free);       // S columns may be overwritten by S(j+1)
                const int valid = prm.seq_len - j * kBN;  // keys of this tile that exist
                if (decltype(masked)::value) {
#pragma unroll
                    for (int c = 0; c < 2; ++c)
#pragma unroll
                        for (int i = 0; i < 32; ++i)
                            if (32 * c + i >= valid) s[c][i] = 0xff800000u;      // -inf
                }
                float mx[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
                for (int c = 0; c < 2; ++c)
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
                    ptx::mbar_wait(a_pv_done, (j - 1) & 1);
                    ptx::tc_fence_after();
                    const float alpha = grow ? ptx::ex2(m_used - m_new) : 1.0f;
                    if (grow) m_used = m_new;
                    const uint64_t alpha2 = ptx::pack2(alpha, alpha);
#pragma unroll
                    for (int c = 0; c < kD / 32; ++c) {
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
                const uint64_t neg_m2 = ptx::pack2(-m_used, -m_used);
#pragma unroll
                for (int c = 0; c < 2; ++c) {
#pragma unroll
                    for (int i = 0; i < 32; i += 2) {
                        ptx::ffma2(s[c][i], s[c][i + 1], scale2, neg_m2);
                        if (((((i >> 1) & 15) * kPolyPairs) & 15) < kPolyPairs) {       // kPolyPairs of every 16 pairs, evenly spread
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
                    pk[i] = ptx::pack_bf16(__uint_as_float(s[0][2 * i]), __uint_as_float(s[0][2 * i + 1]));
                    pk[16 + i] = ptx::pack_bf16(__uint_as_float(s[1][2 * i]), __uint_as_float(s[1][2 * i + 1]));
                }
                // the P buffer is free once PV(j-1), which read it, has completed
                if (j > 0) ptx::mbar_wait(a_pv_done, (j - 1) & 1);
                ptx::tc_fence_after();
                ptx::tmem_st32(t_p, pk);
                ptx::tc_wait_st();
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(a_p_full);
            };
            for (int j = 0; j + 1 < n_kv; ++j) kv_tile(j, std::false_type{});
            if (prm.seq_len % kBN != 0) kv_tile(n_kv - 1, std::true_type{});
            else kv_tile(n_kv - 1, std::false_type{});
            // ---- epilogue: O / l -> bf16 -> global ----
            ptx::mbar_wait(a_pv_done, (n_kv - 1) & 1);
            ptx::tc_fence_after();
            const int row = row0 + tile * kBM + row_in_tile;
            const float l = __uint_as_float(ptx::tmem_ld1(t_o + kD));           // row sum from the ones column
            ptx::tc_wait_ld();
            const float inv_l = 1.0f / l;
            const size_t tok = static_cast<size_t>(seq) * prm.seq_len + row;
            uint4* dst = reinterpret_cast<uint4*>(prm.out + (tok * prm.heads + head) * kD);
#pragma unroll
            for (int c = 0; c < kD / 32; ++c) {
                uint32_t o[32];
                ptx::tmem_ld32(t_o + 32 * c, o);
                ptx::tc_wait_ld();
                if (row < prm.seq_len) {
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        uint4 w;
                        w.x = ptx::pack_bf16(__uint_as_float(o[8 * i + 0]) * inv_l, __uint_as_float(o[8 * i + 1]) * inv_l);
                        w.y = ptx::pack_bf16(__uint_as_float(o[8 * i + 2]) * inv_l, __uint_as_float(o[8 * i + 3]) * inv_l);
                        w.z = ptx::pack_bf16(__uint_as_float(o[8 * i + 4]) * inv_l, __uint_as_float(o[8 * i + 5]) * inv_l);
                        w.w = ptx::pack_bf16(__uint_as_float(o[8 * i + 6]) * inv_l, __uint_as_float(o[8 * i + 7]) * inv_l);
                        dst[4 * c + i] = w;
                    }
                }
            }
            if (row < prm.seq_len && prm.lse) {
                const int win = seq / prm.lse_frames, frame = seq - win * prm.lse_frames;
                prm.lse[(static_cast<size_t>(win) * prm.heads + head) * prm.lse_frames * prm.seq_len +
                        static_cast<size_t>(frame) * prm.seq_len + row] = (m_used + log2f(l)) * 0.6931471805599453f;
            }
        }
        if (lane == 0) ptx::mbar_arrive(&sm.roles_done);
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 9) ptx::tmem_dealloc(tmem, kTmemCols);
}

// bf16 [sequences, seq_len, heads, 128] -> 4-D map (d, head, token, sequence), box = 64 x 1 x rows x 1
static mf_status make_map(CUtensorMap* map, const void* base, int sequences, int seq_len, int heads, int box_rows) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return fail(MF_ERR_CUDA, "cuTensorMapEncodeTiled entry point not available");
    cuuint64_t dims[4] = {static_cast<cuuint64_t>(kD), static_cast<cuuint64_t>(heads), static_cast<cuuint64_t>(seq_len),
                          static_cast<cuuint64_t>(sequences)};
    cuuint64_t strides[3] = {static_cast<cuuint64_t>(kD) * 2, static_cast<cuuint64_t>(heads) * kD * 2,
                             static_cast<cuuint64_t>(seq_len) * heads * kD * 2};
    cuuint32_t box[4] = {kDH, 1, static_cast<cuuint32_t>(box_rows), 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(base), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(MF_ERR_CUDA, "cuTensorMapEncodeTiled failed (CUresult %d)", static_cast<int>(r));
    return MF_OK;
}

}  // namespace d128

mf_status launch_attention_d128(const void* q, const void* k, const void* v, int sequences, int seq_len, int heads,
                                const AttnParams& prm_in, cudaStream_t stream) {
    using namespace d128;
    AttnParams prm = prm_in;
    prm.q_blocks = (seq_len + kQTiles * kBM - 1) / (kQTiles * kBM);
    CUtensorMap mq, mk, mv;
    mf_status st;
    if ((st = make_map(&mq, q, sequences, seq_len, heads, kBM)) != MF_OK) return st;
    if ((st = make_map(&mk, k, sequences, seq_len, heads, kBN)) != MF_OK) return st;
    if ((st = make_map(&mv, v, sequences, seq_len, heads, kBN)) != MF_OK) return st;
    const long long grid = static_cast<long long>(prm.q_blocks) * heads * sequences;
    if (grid > 0x7fffffffLL) return fail(MF_ERR_UNSUPPORTED, "mf_window_attention: grid too large");
    const int smem = static_cast<int>(sizeof(Smem)) + 1024;
    {
        static std::atomic<bool> attr_set[64];
        int dev = 0;
        MF_CUDA_OK(cudaGetDevice(&dev));
        if (dev < 0 || dev >= 64 || !attr_set[dev].load(std::memory_order_acquire)) {
            MF_CUDA_OK(cudaFuncSetAttribute(window_attention_d128_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            if (dev >= 0 && dev < 64) attr_set[dev].store(true, std::memory_order_release);
        }
    }
    window_attention_d128_kernel<<<static_cast<unsigned>(grid), kThreads, smem, stream>>>(mq, mk, mv, prm);
    MF_CUDA_OK(cudaGetLastError());
    return MF_OK;
}

}  // namespace mf
