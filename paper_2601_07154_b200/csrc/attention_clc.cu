// mf_window_attention, head_dim 64, short sequences (fewer than 32 KV tiles: FRAME mode, S <= 3968): the same tile pipeline as
// window_attention_kernel (attention.cu), made PERSISTENT with Blackwell's cluster launch control.
//
// A CTA of attention.cu lives for one work item (sequence, head, 256 query rows).  With 7 KV tiles per item (P = 777) its
// prologue (barrier init, TMEM allocation, the ones tile, first loads uncovered) and epilogue are a third of its life.  Here the
// grid is still one CTA per item, but a CTA that finishes an item does not exit: it asks the hardware for the coordinates of
// a CTA of the same grid that has not started yet (`clusterlaunchcontrol.try_cancel`, SASS UGETNEXTWORKID), cancels it and
// does that item itself, with TMEM, barriers and the ones tile already in place, the next item's Q tiles prefetched into a
// second Q slot and its first S tile issued before the current item's last P V.  So the work is handed out dynamically by the
// hardware CTA scheduler (a static round-robin was measured: SMs differ by 16 % in time per item and a fixed share per
// SM lost 8 % on the campus launch) and no global counter or workspace is needed behind the C ABI.
// The grid is 3-D (q block, head, sequence), so the cancelled CTA's %ctaid is the work item, no division.
// Roles and TMEM map as in attention.cu; differences: barrier phases run across items (counters instead of the tile index),
// Q is double-buffered, `o_free` lets the MMA issuer overwrite O only after the previous item's epilogue has read it, the
// 128 x 64 output tile leaves through one TMA store staged in the item's Q tile (the Q slot is released once the store has
// read it), and the idle warp 11 is the watchdog (sm100_ptx.cuh).
#include "attention_common.cuh"
#include "tensormap.h"

#include <atomic>
#include <cstddef>
#include <type_traits>

namespace mf {
namespace clc {

constexpr int kD = 64;                 // head_dim
constexpr int kBM = 128;               // query rows per tile (UMMA M)
constexpr int kBN = 128;               // keys per KV tile
constexpr int kQTiles = 2;             // Q tiles per CTA
constexpr int kQSlots = 2;             // Q double buffer (the next item's Q is prefetched)
constexpr int kStages = 4;             // K and V ring depth
constexpr int kItemSlots = 4;          // cluster-launch-control responses in flight
constexpr int kTileBytes = kBM * kD * 2;
constexpr int kThreads = 384;
constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kColS = 0, kColO = 256, kColP = 416;
constexpr int kON = 80;                // PV accumulator columns: 64 outputs + column 64 = row sum l (+15 unused)
constexpr int kPH = 32;                // TMEM columns of one P half (64 keys, bf16)
constexpr float kRescaleThreshold = 8.0f;
constexpr int kPolyPairs = MF_POLY_PAIRS;          // (attention_common.cuh)

struct Smem {
    alignas(1024) uint8_t q[kQSlots][kQTiles][kTileBytes];
    alignas(1024) uint8_t k[kStages][kTileBytes];
    alignas(1024) uint8_t v[kStages][kTileBytes];
    alignas(1024) uint8_t ones[kTileBytes];          // [128 keys][64]: column 0 = 1.0, rest 0 (swizzled like V)
    alignas(16) uint32_t next_item[kItemSlots][4];   // try_cancel responses (opaque 16 bytes each)
    alignas(8) uint64_t item_ready[kItemSlots];      // complete_tx of the response
    uint64_t q_full[kQSlots], q_empty[kQSlots];
    uint64_t k_full[kStages], k_empty[kStages], v_full[kStages], v_empty[kStages];
    uint64_t s_full[kQTiles], s_free[kQTiles], p_full[2][kQTiles], pv_done[2][kQTiles], o_free[kQTiles];   // [half][tile]
    uint64_t roles_done;
    uint32_t tmem_base;
    uint32_t zero;     // always 0 (see the softmax loop)
};

constexpr uint32_t kIdescQK = ptx::idesc_bf16_f32(kBM, kBN, 0, 0);
constexpr uint32_t kIdescPV = ptx::idesc_bf16_f32(kBM, kON, 0, 1);

__device__ __forceinline__ void issue_qk(uint32_t tmem_s, const uint8_t* q, const uint8_t* k) {
    const uint64_t qd = ptx::smem_desc_sw128(ptx::smem_u32(q));
    const uint64_t kd = ptx::smem_desc_sw128(ptx::smem_u32(k));
#pragma unroll
    for (int i = 0; i < kD / 16; ++i) ptx::mma_ss(tmem_s, qd + 2 * i, kd + 2 * i, kIdescQK, i > 0);
}
__device__ __forceinline__ void issue_pv_half(uint32_t tmem_o, uint32_t tmem_p, const uint8_t* v_half, uint32_t ones_minus_v,
                                              bool accumulate) {
    const uint64_t vd = ptx::smem_desc_sw128(ptx::smem_u32(v_half), ones_minus_v);
#pragma unroll
    for (int i = 0; i < kBN / 32; ++i)
        ptx::mma_ts(tmem_o, tmem_p + 8 * i, vd + (2048 >> 4) * i, kIdescPV, (accumulate || i > 0) ? 1u : 0u);
}

// A work item = the coordinates of one CTA of the grid: (q block, head, sequence).
struct Item {
    int qb, head, seq;
    bool valid;
    __device__ __forceinline__ int row0() const { return qb * (kQTiles * kBM); }
    __device__ __forceinline__ bool tile1_live(const AttnParams& prm) const { return row0() + kBM < prm.seq_len; }
};
__device__ __forceinline__ Item own_item() {
    Item it;
    it.qb = blockIdx.x; it.head = blockIdx.y; it.seq = blockIdx.z; it.valid = true;
    return it;
}
// Item number qi >= 1 of this CTA (called by whole warps): wait for the response to the query the producer sent while item qi-1 began, decode it.
// (Slot reuse: the query for item qi+4 is sent when the producer starts item qi+3, which needs the Q slot of item qi+1
// released, i.e. every role well past reading the response for item qi.)
__device__ __forceinline__ Item fetch_item(Smem& sm, int qi) {
    const int slot = (qi - 1) % kItemSlots;               // item 0 is the CTA's own: responses are numbered from item 1
    ptx::mbar_wait(&sm.item_ready[slot], ((qi - 1) / kItemSlots) & 1);
    Item it;
    uint32_t valid, x, y, z;
    asm volatile(
        "{\n\t.reg .pred p1;\n\t.reg .b128 res;\n\t"
        "ld.shared.b128 res, [%4];\n\t"
        "clusterlaunchcontrol.query_cancel.is_canceled.pred.b128 p1, res;\n\t"
        "selp.u32 %3, 1, 0, p1;\n\t"
        "@p1 clusterlaunchcontrol.query_cancel.get_first_ctaid.v4.b32.b128 {%0, %1, %2, _}, res;\n\t}"
        : "=r"(x), "=r"(y), "=r"(z), "=r"(valid) : "r"(ptx::smem_u32(sm.next_item[slot])) : "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");         // the slot is rewritten by the async proxy later
    // (every lane of the calling warp read the same 16 bytes; the shuffles tell the compiler so)
    it.valid = __shfl_sync(0xffffffffu, valid, 0) != 0;
    it.qb = static_cast<int>(__shfl_sync(0xffffffffu, x, 0));
    it.head = static_cast<int>(__shfl_sync(0xffffffffu, y, 0));
    it.seq = static_cast<int>(__shfl_sync(0xffffffffu, z, 0));
    return it;
}
// Ask the hardware for one more not-yet-started CTA of this grid; the 16-byte answer lands in next_item[slot].
__device__ __forceinline__ void query_item(Smem& sm, int qi) {
    const int slot = (qi - 1) % kItemSlots;
    ptx::mbar_arrive_expect_tx(&sm.item_ready[slot], 16);
    asm volatile("clusterlaunchcontrol.try_cancel.async.shared::cta.mbarrier::complete_tx::bytes.b128 [%0], [%1];"
                 :: "r"(ptx::smem_u32(sm.next_item[slot])), "r"(ptx::smem_u32(&sm.item_ready[slot])) : "memory");
}

__global__ void __launch_bounds__(kThreads, 1)
window_attention_clc_kernel(const __grid_constant__ CUtensorMap map_q, const __grid_constant__ CUtensorMap map_k,
                            const __grid_constant__ CUtensorMap map_v, const __grid_constant__ CUtensorMap map_o,
                            const AttnParams prm) {
    extern __shared__ uint8_t smem_raw[];
    Smem& sm = *reinterpret_cast<Smem*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    // (warp number through a shuffle: warp-uniform to the compiler, see attention.cu)
    const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;

    if (warp == 8 && lane == 0) {
        ptx::prefetch_tensormap(&map_q);
        ptx::prefetch_tensormap(&map_k);
        ptx::prefetch_tensormap(&map_v);
        ptx::prefetch_tensormap(&map_o);
        for (int s = 0; s < kItemSlots; ++s) ptx::mbar_init(&sm.item_ready[s], 1);
        for (int s = 0; s < kQSlots; ++s) {
            ptx::mbar_init(&sm.q_full[s], 1);
            ptx::mbar_init(&sm.q_empty[s], 2 * kQTiles);   // per Q tile: its MMA issuer (last Q K^T issued) and its output store (staging read)
        }
        for (int s = 0; s < kStages; ++s) {
            ptx::mbar_init(&sm.k_full[s], 1);
            ptx::mbar_init(&sm.k_empty[s], kQTiles);       // both MMA issuers release every K/V stage
            ptx::mbar_init(&sm.v_full[s], 1);
            ptx::mbar_init(&sm.v_empty[s], kQTiles);
        }
        for (int t = 0; t < kQTiles; ++t) {
            ptx::mbar_init(&sm.s_full[t], 1);
            ptx::mbar_init(&sm.s_free[t], 4);              // one arrival per softmax warp
            ptx::mbar_init(&sm.o_free[t], 4);
            for (int h = 0; h < 2; ++h) {
                ptx::mbar_init(&sm.p_full[h][t], 4);
                ptx::mbar_init(&sm.pv_done[h][t], 1);
            }
        }
        ptx::mbar_init(&sm.roles_done, 11);
        sm.zero = 0;
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
    // All 512 columns are allocated, so the allocation starts at column 0, lane 0: TMEM addresses below are compile-time
    // constants (one register less in every role).  Anything else is a protocol error.
    if (sm.tmem_base != 0u) __trap();
    constexpr uint32_t tmem = 0u;
    const int n_kv = (prm.seq_len + kBN - 1) / kBN;

    // register split: 168/thread at launch -> 224 for the softmax warpgroups, 56 for the rest
    if (warp >= 8) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        if (warp == 8) {
            // ===================== TMA producer and work scheduler (whole warp in the loop, one elected lane issues) =====================
            {
                const bool leader = ptx::elect_one();
                uint32_t kv = 0;                            // K/V tiles loaded so far (ring position)
                Item it = own_item();
                for (int qi = 0; it.valid; ++qi) {
                    if (leader) query_item(sm, qi + 1);     // the item after this one, while this one is being loaded
                    const int slot = qi & 1, use = qi >> 1;
                    if (use > 0) ptx::mbar_wait(&sm.q_empty[slot], (use - 1) & 1);
                    // a dead second tile re-reads the first one (in bounds, never used); no output store will read its staging
                    // buffer, so the producer makes that arrival on the Q slot itself
                    const bool dead1 = !it.tile1_live(prm);
                    if (leader) {
                        ptx::mbar_arrive_expect_tx(&sm.q_full[slot], kQTiles * kTileBytes);
                        ptx::tma_load_4d(sm.q[slot][0], &map_q, &sm.q_full[slot], 0, it.head, it.row0(), it.seq);
                        ptx::tma_load_4d(sm.q[slot][1], &map_q, &sm.q_full[slot], 0, it.head, dead1 ? it.row0() : it.row0() + kBM, it.seq);
                        if (dead1) ptx::mbar_arrive(&sm.q_empty[slot]);
                    }
                    for (int j = 0; j < n_kv; ++j, ++kv) {
                        const int st = kv % kStages;
                        const uint32_t ph = (kv / kStages) & 1;
                        ptx::mbar_wait(&sm.k_empty[st], ph ^ 1);
                        if (leader) {
                            ptx::mbar_arrive_expect_tx(&sm.k_full[st], kTileBytes);
                            ptx::tma_load_4d(sm.k[st], &map_k, &sm.k_full[st], 0, it.head, j * kBN, it.seq);
                        }
                        ptx::mbar_wait(&sm.v_empty[st], ph ^ 1);
                        if (leader) {
                            ptx::mbar_arrive_expect_tx(&sm.v_full[st], kTileBytes);
                            ptx::tma_load_4d(sm.v[st], &map_v, &sm.v_full[st], 0, it.head, j * kBN, it.seq);
                        }
                    }
                    it = fetch_item(sm, qi + 1);
                }
                __syncwarp();
            }
        } else if (warp <= 10) {
            // ===================== MMA issuers (warp 9: Q tile 0, warp 10: Q tile 1) =====================
            // (the whole warp runs the loop, one elected lane issues the MMAs, commits and arrives)
            const int t = warp - 9;
            {
                const bool leader = ptx::elect_one();
                const uint32_t t_s = tmem + kColS + t * kBN, t_o = tmem + kColO + t * kON, t_p = tmem + kColP + t * kPH;
                uint32_t kv = 0;                            // ring position of the tile whose P V comes next
                uint32_t ns = 0;                            // S tiles issued so far (= phase counter of s_full / s_free)
                uint32_t np = 0;                            // KV tiles whose P V has been issued (= phase of p_full / pv_done)
                uint32_t live_items = 0;                    // items of this tile slot finished (= phase of o_free)
                bool have_s = false;                        // S(0) of the current item was issued ahead, during the previous item
                auto issue_s = [&](int slot, uint32_t kvi) {
                    const int st = kvi % kStages;
                    if (ns > 0) ptx::mbar_wait(&sm.s_free[t], (ns - 1) & 1);      // the softmax warps hold the previous S in registers
                    ptx::mbar_wait(&sm.k_full[st], (kvi / kStages) & 1);
                    ptx::tc_fence_after();
                    if (leader) {
                        issue_qk(t_s, sm.q[slot][t], sm.k[st]);
                        ptx::mma_commit(&sm.s_full[t]);
                        ptx::mma_commit(&sm.k_empty[st]);
                    }
                    ++ns;
                };
                Item it = own_item();
                for (int qi = 0; it.valid; ++qi) {
                    const int slot = qi & 1;
                    const bool live = t == 0 || it.tile1_live(prm);
                    if (!live) {
                        // Nothing to compute for this tile slot, but it stays a link of the flow control: it releases the Q slot
                        // and every K/V stage of the item only after it has seen them filled.  (Parity waits tell only
                        // neighbouring phases apart: an issuer that skipped these waits would later take a stage's previous fill
                        // for the one it is waiting for, and one that only watched, with the producer making its arrivals, could
                        // be lapped by the producer.  Both were tried; both deadlock on long runs of such items.)
                        ptx::mbar_wait(&sm.q_full[slot], (qi >> 1) & 1);
                        if (leader) ptx::mbar_arrive(&sm.q_empty[slot]);
                        for (int j = 0; j < n_kv; ++j, ++kv) {
                            const int st = kv % kStages;
                            const uint32_t ph = (kv / kStages) & 1;
                            ptx::mbar_wait(&sm.k_full[st], ph);
                            if (leader) ptx::mbar_arrive(&sm.k_empty[st]);
                            ptx::mbar_wait(&sm.v_full[st], ph);
                            if (leader) ptx::mbar_arrive(&sm.v_empty[st]);
                        }
                        have_s = false;
                        it = fetch_item(sm, qi + 1);
                        continue;
                    }
                    Item next = it;
                    if (!have_s) {
                        ptx::mbar_wait(&sm.q_full[slot], (qi >> 1) & 1);
                        issue_s(slot, kv);
                    }
                    have_s = false;
                    for (int j = 0; j < n_kv; ++j, ++kv, ++np) {
                        const int st = kv % kStages;
                        if (j + 1 < n_kv) {
                            issue_s(slot, kv + 1);          // S(j+1) as soon as the softmax warpgroup holds S(j) in registers
                        } else {
                            if (leader) ptx::mma_commit(&sm.q_empty[slot]);             // every Q K^T of this item has been issued
                            next = fetch_item(sm, qi + 1);  // (asked for when this item began: long since answered)
                            // The next item's S(0), ahead of this item's last P V -- but only if its Q tiles have landed: this
                            // thread must never BLOCK on the future while it still owes the present its P V.  (With one KV tile
                            // per item the next-but-one Q load waits for this item's output store, which waits for the softmax
                            // warps, which wait for this P V: a blocking wait here deadlocked S <= 128 launches of more than
                            // 148 items; found by differential fuzzing against attention.cu, ended by the watchdog.)
                            // (one decision for the warp: all lanes must have seen the phase complete)
                            if (next.valid && (t == 0 || next.tile1_live(prm)) &&
                                __all_sync(0xffffffffu, ptx::mbar_try_wait(&sm.q_full[slot ^ 1], ((qi + 1) >> 1) & 1))) {
                                issue_s(slot ^ 1, kv + 1);
                                have_s = true;
                            }
                        }
                        ptx::mbar_wait(&sm.v_full[st], (kv / kStages) & 1);
                        if (j == 0 && live_items > 0) ptx::mbar_wait(&sm.o_free[t], (live_items - 1) & 1);   // previous item's O has been read
                        const uint32_t ones_minus_v = ptx::smem_u32(sm.ones) - ptx::smem_u32(sm.v[st]);
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            ptx::mbar_wait(&sm.p_full[h][t], np & 1);
                            ptx::tc_fence_after();
                            if (leader) {
                                issue_pv_half(t_o, t_p, sm.v[st] + h * (kTileBytes / 2), ones_minus_v, j > 0 || h > 0);
                                ptx::mma_commit(&sm.pv_done[h][t]);
                            }
                        }
                        if (leader) ptx::mma_commit(&sm.v_empty[st]);
                    }
                    ++live_items;
                    it = next;
                }
                __syncwarp();
            }
        } else if (lane == 0) {
            ptx::watchdog_progress(&sm.roles_done, sm.k_full);                // warp 11: traps if the 11 role warps do not finish within seconds
        }
        if (warp <= 10 && lane == 0) ptx::mbar_arrive(&sm.roles_done);
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 224;");
        // ===================== softmax warpgroups =====================
        const int tile = warp >> 2;                       // 0 or 1
        const int row_in_tile = (warp & 3) * 32 + lane;
        const uint32_t lane_addr = static_cast<uint32_t>((warp & 3) * 32) << 16;
        const uint32_t t_s = tmem + lane_addr + kColS + tile * kBN;
        const uint32_t t_o = tmem + lane_addr + kColO + tile * kON;
        const uint32_t t_p = tmem + lane_addr + kColP + tile * kPH;
        const uint64_t scale2 = ptx::pack2(prm.scale_log2, prm.scale_log2);
        // barrier addresses = one opaque base register + constants (sm100_ptx.cuh: smem_base_u32)
        const uint32_t sb = ptx::smem_base_u32(&sm);
        const uint32_t a_s_full = sb + offsetof(Smem, s_full) + 8 * tile, a_s_free = sb + offsetof(Smem, s_free) + 8 * tile;
        const uint32_t a_p_full0 = sb + offsetof(Smem, p_full) + 8 * tile, a_p_full1 = a_p_full0 + 8 * kQTiles;
        const uint32_t a_pv_done0 = sb + offsetof(Smem, pv_done) + 8 * tile, a_pv_done1 = a_pv_done0 + 8 * kQTiles;
        uint32_t ns = 0;                                  // KV tiles consumed by this warpgroup (phase counter, runs across items)
        int store_pending = -1;                           // (thread row_in_tile == 0) Q slot whose output store is still reading shared memory
        Item it = own_item();
        for (int qi = 0; it.valid; ++qi) {
            const int slot = qi & 1;
            if (tile == 1 && !it.tile1_live(prm)) {
                if (store_pending >= 0) {                 // (the producer may be waiting for this Q slot before it can go on)
                    ptx::tma_store_wait_read();
                    ptx::mbar_arrive(&sm.q_empty[store_pending]);
                    store_pending = -1;
                }
                it = fetch_item(sm, qi + 1);
                continue;
            }
            float m_used = -INFINITY;                     // running max in scaled log2 units
            // One KV tile.  The loop below runs it without the tail-masking code (only a ragged LAST tile needs it: peeled off, the
            // steady-state loop is one contiguous block of code); the last tile picks its instantiation: `tail` = 0 for a full
            // tile, else the number of 32-column chunks of S that hold keys; the other chunks are neither read nor exponentiated
            // and their P is stored as zeros (attention.cu has the measurements).
            auto kv_tile = [&](const int j, auto tail) {
                constexpr bool kMasked = decltype(tail)::value != 0;
                constexpr int kChunks = kMasked ? decltype(tail)::value : 4;
                ptx::mbar_wait(a_s_full, ns & 1);
                ptx::tc_fence_after();
                uint32_t s[4][32];
#pragma unroll
                for (int c = 0; c < kChunks; ++c) ptx::tmem_ld32(t_s + 32 * c, s[c]);
                ptx::tc_wait_ld();
                ptx::tc_fence_before();
                __syncwarp();
#ifdef MF_TEST_PROTOCOL_BUG      // test builds only (tests/test_gpu_watchdog.py): CTA (0,0,0) never hands S back, so its pipeline stalls for good
                if (lane == 0 && (blockIdx.x | blockIdx.y | blockIdx.z) != 0) ptx::mbar_arrive(a_s_free);
#else
                if (lane == 0) ptx::mbar_arrive(a_s_free);               // S columns may be overwritten by the next S
#endif
                const int valid = prm.seq_len - j * kBN;  // keys of this tile that exist
                if (kMasked) {
#pragma unroll
                    for (int c = 0; c < kChunks; ++c)
#pragma unroll
                        for (int i = 0; i < 32; ++i)
                            if (32 * c + i >= valid) s[c][i] = 0xff800000u;      // -inf
                }
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
                    ptx::mbar_wait(a_pv_done1, (ns - 1) & 1);
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
                const uint64_t neg_m2 = ptx::pack2(-m_used, -m_used);
                uint64_t scale_h = scale2;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
#pragma unroll
                    for (int c = 2 * h; c < 2 * h + 2 && c < kChunks; ++c) {
#pragma unroll
                        for (int i = 0; i < 32; i += 2) {
                            ptx::ffma2(s[c][i], s[c][i + 1], scale_h, neg_m2);
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
                        pk[i] = 2 * h < kChunks ? ptx::pack_bf16(__uint_as_float(s[2 * h][2 * i]), __uint_as_float(s[2 * h][2 * i + 1])) : 0u;
                        pk[16 + i] = 2 * h + 1 < kChunks ? ptx::pack_bf16(__uint_as_float(s[2 * h + 1][2 * i]), __uint_as_float(s[2 * h + 1][2 * i + 1])) : 0u;
                    }
                    // the P half buffer is free once the previous PV that read it has completed
                    if (h == 1) ptx::mbar_wait(a_pv_done0, ns & 1);
                    else if (ns > 0) ptx::mbar_wait(a_pv_done1, (ns - 1) & 1);
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
                        asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(z) : "r"(sb + static_cast<uint32_t>(offsetof(Smem, zero))) : "memory");
                        scale_h = ptx::pack2(__uint_as_float(__float_as_uint(prm.scale_log2) | z),
                                             __uint_as_float(__float_as_uint(prm.scale_log2) | z));
                    }
                }
                if (j == 0 && store_pending >= 0) {
                    // the previous item's TMA store has read its staging buffer (that item's Q tile) by now: release the Q slot
                    ptx::tma_store_wait_read();
                    ptx::mbar_arrive(&sm.q_empty[store_pending]);
                    store_pending = -1;
                }
            };
            for (int j = 0; j + 1 < n_kv; ++j, ++ns) kv_tile(j, std::integral_constant<int, 0>{});
            const int tail_chunks = (prm.seq_len - (n_kv - 1) * kBN + 31) / 32;        // 1..4
            if (prm.seq_len % kBN == 0) kv_tile(n_kv - 1, std::integral_constant<int, 0>{});
            else if (tail_chunks == 1) kv_tile(n_kv - 1, std::integral_constant<int, 1>{});
            else if (tail_chunks == 2) kv_tile(n_kv - 1, std::integral_constant<int, 2>{});
            else kv_tile(n_kv - 1, std::integral_constant<int, 4>{});
            ++ns;
            // ---- epilogue: O / l -> bf16 -> shared memory (this item's Q tile) -> one TMA store ----
            ptx::mbar_wait(a_pv_done1, (ns - 1) & 1);
            ptx::tc_fence_after();
            const int row = it.row0() + tile * kBM + row_in_tile;
            uint32_t o[2][32];
            ptx::tmem_ld32(t_o, o[0]);
            ptx::tmem_ld32(t_o + 32, o[1]);
            const float l = __uint_as_float(ptx::tmem_ld1(t_o + kD));           // row sum from the ones column
            ptx::tc_wait_ld();
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&sm.o_free[tile]);                   // the next item's P V may overwrite O
            const float inv_l = 1.0f / l;
            {
                uint4* stage = reinterpret_cast<uint4*>(sm.q[slot][tile]) + row_in_tile * 8;     // 8 chunks of 16 bytes per row
#pragma unroll
                for (int c = 0; c < 2; ++c)
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        uint4 w;
                        w.x = ptx::pack_bf16(__uint_as_float(o[c][8 * i + 0]) * inv_l, __uint_as_float(o[c][8 * i + 1]) * inv_l);
                        w.y = ptx::pack_bf16(__uint_as_float(o[c][8 * i + 2]) * inv_l, __uint_as_float(o[c][8 * i + 3]) * inv_l);
                        w.z = ptx::pack_bf16(__uint_as_float(o[c][8 * i + 4]) * inv_l, __uint_as_float(o[c][8 * i + 5]) * inv_l);
                        w.w = ptx::pack_bf16(__uint_as_float(o[c][8 * i + 6]) * inv_l, __uint_as_float(o[c][8 * i + 7]) * inv_l);
                        stage[(4 * c + i) ^ (row_in_tile & 7)] = w;
                    }
                ptx::fence_proxy_async();                         // generic-proxy writes -> visible to the TMA (async proxy)
                asm volatile("bar.sync %0, 128;" :: "r"(1 + tile) : "memory");      // the tile's four softmax warps
                if (row_in_tile == 0) {
                    ptx::tma_store_4d(&map_o, sm.q[slot][tile], 0, it.head, it.row0() + tile * kBM, it.seq);
                    ptx::tma_store_commit();
                    store_pending = slot;                 // waited for (and the Q slot released) after the next item's first tile
                }
            }
            if (row < prm.seq_len && prm.lse) {
                const int win = it.seq / prm.lse_frames, frame = it.seq - win * prm.lse_frames;
                prm.lse[(static_cast<size_t>(win) * prm.heads + it.head) * prm.lse_frames * prm.seq_len +
                        static_cast<size_t>(frame) * prm.seq_len + row] = (m_used + log2f(l)) * 0.6931471805599453f;
            }
            it = fetch_item(sm, qi + 1);
        }
        if (store_pending >= 0) ptx::tma_store_wait_read();       // shared memory must outlive the last store's read
        if (lane == 0) ptx::mbar_arrive(&sm.roles_done);
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 9) ptx::tmem_dealloc(tmem, kTmemCols);
}

}  // namespace clc

mf_status launch_attention_clc(const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv, const CUtensorMap& mo,
                               int sequences, int seq_len, int heads, const AttnParams& prm, cudaStream_t stream) {
    using namespace clc;
    if (heads > 65535 || sequences > 65535)       // (the caller keeps such launches on the 1-D grid of attention.cu)
        return fail(MF_ERR_INVALID_ARG, "launch_attention_clc: heads and sequences must fit a grid dimension");
    const int smem = static_cast<int>(sizeof(Smem)) + 1024;
    {   // the opt-in shared-memory size is a per-device attribute of the kernel: set it once per device
        static std::atomic<bool> attr_set[64];
        int dev = 0;
        MF_CUDA_OK(cudaGetDevice(&dev));
        if (dev < 0 || dev >= 64 || !attr_set[dev].load(std::memory_order_acquire)) {
            MF_CUDA_OK(cudaFuncSetAttribute(window_attention_clc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
            if (dev >= 0 && dev < 64) attr_set[dev].store(true, std::memory_order_release);
        }
    }
    const dim3 grid(static_cast<unsigned>(prm.q_blocks), static_cast<unsigned>(heads), static_cast<unsigned>(sequences));
    window_attention_clc_kernel<<<grid, kThreads, smem, stream>>>(mq, mk, mv, mo, prm);
    MF_CUDA_OK(cudaGetLastError());
    return MF_OK;
}

}  // namespace mf
