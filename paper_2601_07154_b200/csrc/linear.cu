// mf_linear: out = act(x w^T + bias) (+ residual), bf16 in / fp32 accumulate / bf16 out, for sm_100a
// (the QKV projection, output projection and MLP around the window attention; reading E1-E4).
//
// Persistent kernel, 320 threads per CTA, one CTA per SM, CTAs working in PAIRS (cluster of 2, tcgen05 cta_group::2) on
// 256 x 256 output tiles (a 1-CTA 128 x 256 instantiation remains for single-band problems and MF_LINEAR_CTAS=1):
//   warp 0     TMA producer: this CTA's 128 rows of x and its HALF of the w tile (128 output columns) per 64-wide k step,
//              SWIZZLE_128B, 6-stage ring (32 KB per stage); both CTAs' loads complete on the leader's mbarrier
//   warp 1     leader CTA only: one thread issues tcgen05.mma.cta_group::2, M = 256, N = 256, 4 x K=16 per stage; the MMA
//              reads both CTAs' shared memory and accumulates rows 0-127 in the leader's TMEM, 128-255 in the peer's;
//              tcgen05.commit ... multicast::cluster frees the stage / publishes the accumulator in both CTAs.  Two
//              accumulators (2 x 256 columns) so the epilogue of tile i overlaps the main loop of tile i+1
//   warps 2-9  epilogue (both CTAs, own 128 rows): tcgen05.ld 64 columns per pass (TMEM lane = output row; two warps per
//              lane quarter, half of the columns each), + bias, GELU, + residual, round to bf16, staged through a swizzled
//              per-warp buffer so that global stores and residual loads are 4 rows x 128 B per warp instruction
// Output tiles are visited n-fastest, so the CTAs running together share one band of x rows in L2 while w (a few
// MB) stays L2-resident.  Columns may be split over up to three output tensors (q | k | v): n_split columns each.
#include "common.h"
#include "sm100_ptx.cuh"
#include "tensormap.h"

#include <cuda_bf16.h>

#include <atomic>
#include <cstdlib>

namespace mf {

constexpr int kGM = 128, kGN = 256, kGK = 64;
constexpr int kEpiWarps = 8;               // two per TMEM lane quarter: each takes half of the tile's 256 columns
constexpr int kGThreads = (4 + kEpiWarps) * 32;   // warpgroup 0: TMA producer, MMA issuer and two idle warps; warpgroups 1-2: the epilogue warps
// (A CTA of 10 warps is allocated as 12 anyway, which capped the kernel at 168 registers per thread and made ptxas spill the
// epilogue's residual prefetch: the spill store then waited for the loads in front of every tile.  With 12 warps setmaxnreg
// moves warpgroup 0's registers to the epilogue warps: 56 / 224.)
constexpr int kATile = kGM * kGK * 2;      // 16 KB

// kCtas = 1: one CTA per 128 x 256 output tile.  kCtas = 2: a CTA pair (cluster of 2, tcgen05 cta_group::2) per 256 x 256
// tile: each CTA holds its 128 rows of x and HALF of the w tile (128 of the 256 output columns), the leader issues
// M = 256 MMAs that read both CTAs' shared memory and accumulate into both CTAs' TMEM.  A stage is 32 KB instead of
// 48 KB, so the same shared memory holds 6 stages: the ring covers 3072 instead of 2048 tensor clocks of load latency.
template <int kCtas>
struct GemmSmem {
    static constexpr int kStages = kCtas == 2 ? 6 : 4;
    static constexpr int kBTile = (kGN / kCtas) * kGK * 2;      // 32 KB, or 16 KB per CTA of a pair
    static constexpr int kGStages = kStages;
    alignas(1024) uint8_t a[kStages][kATile];
    alignas(1024) uint8_t b[kStages][kBTile];
    alignas(16) uint8_t stage[kEpiWarps][32 * 128];      // per epilogue warp: 32 rows x 64 bf16, XOR-swizzled 16-byte chunks
    alignas(8) uint64_t full[kGStages];
    uint64_t empty[kGStages], acc_full[2], acc_empty[2];
    uint32_t tmem_base;
};

struct GemmParams {
    int M, N, K, n_split;
    int m_tiles, n_tiles;       // m_tiles counts 128-row (kCtas = 1) or 256-row (kCtas = 2) bands
    const float* bias;
    const __nv_bfloat16* residual;
    __nv_bfloat16* out[3];
    int act;
};

constexpr uint32_t kIdescGemm = ptx::idesc_bf16_f32(kGM, kGN, 0, 0);
constexpr uint32_t kIdescGemmPair = ptx::idesc_bf16_f32(2 * kGM, kGN, 0, 0);

// Reading E3 (exact erf GELU).  erf by Abramowitz & Stegun 7.1.26 (|error| <= 1.5e-7, far below the bf16 output's 2^-9):
// erf(x) = 1 - (a1 t + ... + a5 t^5) exp(-x^2), t = 1 / (1 + p x), x >= 0; odd in x.
__device__ __forceinline__ float gelu_erf(float v) {
    const float x = fabsf(v) * 0.70710678118654752f;
    float t;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(t) : "f"(fmaf(0.3275911f, x, 1.0f)));
    float poly = fmaf(1.061405429f, t, -1.453152027f);
    poly = fmaf(poly, t, 1.421413741f);
    poly = fmaf(poly, t, -0.284496736f);
    poly = fmaf(poly, t, 0.254829592f);
    const float e = ptx::ex2(-x * x * 1.4426950408889634f);
    const float erf_abs = fmaf(-poly * t, e, 1.0f);
    return 0.5f * v * (1.0f + copysignf(erf_abs, v));
}

// The same for two values with packed f32x2 instructions (the same operations in the same order per element, so the result is
// the scalar form's bit for bit): 13 packed + 4 logic + 4 MUFU instructions per pair instead of 32 + 4.
__device__ __forceinline__ void gelu_erf2(float& v0, float& v1) {
    const uint64_t v = ptx::pack2(v0, v1);
    const uint64_t ax = ptx::pack2(fabsf(v0), fabsf(v1));
    uint64_t x, d, poly, arg, pt, ea, r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(x) : "l"(ax), "l"(ptx::pack2(0.70710678118654752f, 0.70710678118654752f)));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(ptx::pack2(0.3275911f, 0.3275911f)), "l"(x), "l"(ptx::pack2(1.0f, 1.0f)));
    float d0, d1, t0, t1;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(d0), "=f"(d1) : "l"(d));
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(t0) : "f"(d0));
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(t1) : "f"(d1));
    const uint64_t t = ptx::pack2(t0, t1);
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(poly) : "l"(ptx::pack2(1.061405429f, 1.061405429f)), "l"(t), "l"(ptx::pack2(-1.453152027f, -1.453152027f)));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(poly) : "l"(poly), "l"(t), "l"(ptx::pack2(1.421413741f, 1.421413741f)));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(poly) : "l"(poly), "l"(t), "l"(ptx::pack2(-0.284496736f, -0.284496736f)));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(poly) : "l"(poly), "l"(t), "l"(ptx::pack2(0.254829592f, 0.254829592f)));
    // (-x * x) * log2(e), then e = 2^that
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(arg) : "l"(x ^ 0x8000000080000000ull), "l"(x));
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(arg) : "l"(arg), "l"(ptx::pack2(1.4426950408889634f, 1.4426950408889634f)));
    float a0, a1;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a0), "=f"(a1) : "l"(arg));
    const uint64_t e = ptx::pack2(ptx::ex2(a0), ptx::ex2(a1));
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(pt) : "l"(poly ^ 0x8000000080000000ull), "l"(t));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(ea) : "l"(pt), "l"(e), "l"(ptx::pack2(1.0f, 1.0f)));
    // copysign(erf_abs, v); 0.5 v (1 + that)
    const uint64_t cs = (ea & 0x7fffffff7fffffffull) | (v & 0x8000000080000000ull);
    uint64_t one_cs, hv;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(one_cs) : "l"(ptx::pack2(1.0f, 1.0f)), "l"(cs));
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(hv) : "l"(ptx::pack2(0.5f, 0.5f)), "l"(v));
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(hv), "l"(one_cs));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(v0), "=f"(v1) : "l"(r));
}

__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* m, uint64_t* bar, int c0, int c1) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
                 :: "r"(ptx::smem_u32(smem_dst)), "l"(reinterpret_cast<uint64_t>(m)), "r"(ptx::smem_u32(bar)), "r"(c0), "r"(c1)
                 : "memory");
}

template <int kCtas>
__global__ void __launch_bounds__(kGThreads, 1)
linear_kernel(const __grid_constant__ CUtensorMap map_x, const __grid_constant__ CUtensorMap map_w, const GemmParams prm) {
    using Smem = GemmSmem<kCtas>;
    constexpr int kGStages = Smem::kStages;
    constexpr int kBTile = Smem::kBTile;
    extern __shared__ uint8_t smem_raw[];
    Smem& sm = *reinterpret_cast<Smem*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    // (warp number and cluster rank through a shuffle: warp-uniform to the compiler, so the role loops keep their addresses and
    // descriptors in uniform registers and the single-lane TMA / MMA issue needs no per-instruction active-lane loop; attention.cu)
    const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;
    const int n_tiles_total = prm.m_tiles * prm.n_tiles;
    const int k_steps = prm.K / kGK;
    const int rank = kCtas == 2 ? __shfl_sync(0xffffffffu, static_cast<int>(ptx::cluster_ctarank()), 0) : 0;     // 0 = leader of the pair
    const int tile0 = blockIdx.x / kCtas, tile_step = gridDim.x / kCtas;

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tensormap(&map_x);
        ptx::prefetch_tensormap(&map_w);
        for (int s = 0; s < kGStages; ++s) {
            ptx::mbar_init(&sm.full[s], 1);
            ptx::mbar_init(&sm.empty[s], 1);
        }
        for (int b = 0; b < 2; ++b) {
            ptx::mbar_init(&sm.acc_full[b], 1);
            ptx::mbar_init(&sm.acc_empty[b], kEpiWarps * kCtas);   // one arrival per epilogue warp (of both CTAs of a pair)
        }
        ptx::fence_barrier_init();
    }
    if (warp == 1) {
        if (kCtas == 2) ptx::tmem_alloc_pair(&sm.tmem_base, 512);
        else ptx::tmem_alloc(&sm.tmem_base, 512);
    }
    ptx::tc_fence_before();
    if (kCtas == 2) ptx::cluster_sync();
    else __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = __shfl_sync(0xffffffffu, sm.tmem_base, 0);

    if (warp < 4) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
    if (warp == 0) {
        // ===================== TMA producer (whole warp in the loop, one elected lane issues) =====================
        {
            const bool leader = ptx::elect_one();
            int it = 0;
            for (int tile = tile0; tile < n_tiles_total; tile += tile_step) {
                const int mt = tile / prm.n_tiles, nt = tile - mt * prm.n_tiles;
                for (int ks = 0; ks < k_steps; ++ks, ++it) {
                    const int st = it % kGStages;
                    ptx::mbar_wait(&sm.empty[st], ((it / kGStages) & 1) ^ 1);
                    if (!leader) continue;
                    if (kCtas == 1) {
                        ptx::mbar_arrive_expect_tx(&sm.full[st], kATile + kBTile);
                        tma_load_2d(sm.a[st], &map_x, &sm.full[st], ks * kGK, mt * kGM);
                        tma_load_2d(sm.b[st], &map_w, &sm.full[st], ks * kGK, nt * kGN);
                    } else {
                        // Both CTAs' loads complete on the LEADER's barrier (the MMA issuer waits there): the leader arrives
                        // once expecting the bytes of both, the peer only contributes bytes.  The peer cannot run a phase
                        // ahead: it refills a stage only after the leader's MMAs on it have completed (multicast commit).
                        const uint32_t lead_full = ptx::mapa(&sm.full[st], 0);
                        if (rank == 0) ptx::mbar_arrive_expect_tx(&sm.full[st], 2 * (kATile + kBTile));
                        ptx::tma_load_2d_pair(sm.a[st], &map_x, lead_full, ks * kGK, mt * (2 * kGM) + rank * kGM);
                        ptx::tma_load_2d_pair(sm.b[st], &map_w, lead_full, ks * kGK, nt * kGN + rank * (kGN / 2));
                    }
                }
            }
            __syncwarp();
        }
    } else if (warp == 1) {
        // ===================== MMA issuer (whole warp in the loop, one elected lane issues) =====================
        if (rank == 0) {
            const bool leader = ptx::elect_one();
            int it = 0, local = 0;
            for (int tile = tile0; tile < n_tiles_total; tile += tile_step, ++local) {
                const int buf = local & 1;
                ptx::mbar_wait(&sm.acc_empty[buf], ((local >> 1) & 1) ^ 1);     // epilogue has drained this accumulator
                ptx::tc_fence_after();
                const uint32_t d = tmem + buf * kGN;
                for (int ks = 0; ks < k_steps; ++ks, ++it) {
                    const int st = it % kGStages;
                    ptx::mbar_wait(&sm.full[st], (it / kGStages) & 1);
                    ptx::tc_fence_after();
                    if (!leader) continue;
                    const uint64_t ad = ptx::smem_desc_sw128(ptx::smem_u32(sm.a[st]));
                    const uint64_t bd = ptx::smem_desc_sw128(ptx::smem_u32(sm.b[st]));
#pragma unroll
                    for (int i = 0; i < kGK / 16; ++i) {
                        if (kCtas == 2) ptx::mma_ss_pair(d, ad + 2 * i, bd + 2 * i, kIdescGemmPair, (ks > 0 || i > 0) ? 1u : 0u);
                        else ptx::mma_ss(d, ad + 2 * i, bd + 2 * i, kIdescGemm, (ks > 0 || i > 0) ? 1u : 0u);
                    }
                    if (kCtas == 2) ptx::mma_commit_pair(&sm.empty[st], 3);        // frees the stage in both CTAs
                    else ptx::mma_commit(&sm.empty[st]);
                }
                if (leader) {
                    if (kCtas == 2) ptx::mma_commit_pair(&sm.acc_full[buf], 3);
                    else ptx::mma_commit(&sm.acc_full[buf]);
                }
            }
            __syncwarp();
        }
    }
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 224;");
        // ===================== epilogue warps =====================
        // A thread owns one output row (TMEM lane) and 64 consecutive columns per pass.  Rows are 2-8 KB apart in
        // global memory, so the 32 x 128 B block of a pass goes through a per-warp, XOR-swizzled staging buffer: global
        // accesses are then 4 rows x 128 B per warp instruction (4 wavefronts instead of 32), for the stores and for
        // the residual loads alike.
        const int quarter = warp & 3;                      // TMEM lanes 32*quarter .. +31
        const int chalf = (warp - 4) >> 2;                 // columns [128*chalf, 128*chalf + 128) of the tile
        const uint32_t lane_addr = static_cast<uint32_t>(quarter * 32) << 16;
        uint4* stage = reinterpret_cast<uint4*>(sm.stage[warp - 4]);      // [32 rows][8 chunks of 16 B]
        const int crow = lane >> 3, cchunk = lane & 7;     // coalesced phase: this lane's row (of 4) and 16-byte chunk
        int local = 0;
        // Residual: the 32 x 128 B block of ONE pass is in flight in registers at a time (coalesced loads), issued a whole pass
        // ahead: pass 1's while pass 0 is computed, the next tile's pass 0 while pass 1 is.
        uint4 rres[8];
        auto load_residual = [&](int t, int g) {
            const int t_mt = t / prm.n_tiles, t_nt = t - t_mt * prm.n_tiles;
            const int t_row0 = t_mt * (kCtas * kGM) + rank * kGM + quarter * 32;
            const int t_n0 = t_nt * kGN + 128 * chalf;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int r = t_row0 + 4 * i + crow;
                rres[i] = r < prm.M ? __ldg(reinterpret_cast<const uint4*>(prm.residual + static_cast<size_t>(r) * prm.N + t_n0 + 64 * g + 8 * cchunk))
                                    : make_uint4(0u, 0u, 0u, 0u);
            }
        };
        if (prm.residual && tile0 < n_tiles_total) load_residual(tile0, 0);
        for (int tile = tile0; tile < n_tiles_total; tile += tile_step, ++local) {
            const int buf = local & 1;
            const int mt = tile / prm.n_tiles, nt = tile - mt * prm.n_tiles;
            const int row0 = mt * (kCtas * kGM) + rank * kGM + quarter * 32;      // first of this warp's 32 rows
            const int n0 = nt * kGN + 128 * chalf;         // first of this warp's 128 columns
            const int which = n0 / prm.n_split, c0 = n0 - which * prm.n_split;
            __nv_bfloat16* dst = prm.out[which] + c0;
            ptx::mbar_wait(&sm.acc_full[buf], (local >> 1) & 1);
            ptx::tc_fence_after();
#pragma unroll
            for (int g = 0; g < 2; ++g) {
                uint32_t acc[2][32];
                ptx::tmem_ld32(tmem + lane_addr + buf * kGN + 128 * chalf + 64 * g, acc[0]);
                ptx::tmem_ld32(tmem + lane_addr + buf * kGN + 128 * chalf + 64 * g + 32, acc[1]);
                uint4 myres[8];                            // this thread's own row of the residual (8 x 8 bf16)
                if (prm.residual) {
                    __syncwarp();
#pragma unroll
                    for (int i = 0; i < 8; ++i) stage[(4 * i + crow) * 8 + (cchunk ^ ((4 * i + crow) & 7))] = rres[i];
                    __syncwarp();
#pragma unroll
                    for (int j = 0; j < 8; ++j) myres[j] = stage[lane * 8 + (j ^ (lane & 7))];
                    __syncwarp();
                    if (g == 0) load_residual(tile, 1);
                    else if (tile + tile_step < n_tiles_total) load_residual(tile + tile_step, 0);
                }
                ptx::tc_wait_ld();
                if (g == 1) {                              // the accumulator is in registers: hand it back to the MMA issuer
                    ptx::tc_fence_before();
                    __syncwarp();
                    if (lane == 0) {
                        if (kCtas == 2 && rank != 0) ptx::mbar_arrive_cluster(ptx::mapa(&sm.acc_empty[buf], 0));
                        else ptx::mbar_arrive(&sm.acc_empty[buf]);
                    }
                }
#pragma unroll
                for (int j = 0; j < 8; ++j) {              // 8 columns per step
                    float vals[8];
#pragma unroll
                    for (int i = 0; i < 8; ++i) vals[i] = __uint_as_float(acc[j >> 2][8 * (j & 3) + i]);
                    if (prm.bias) {
                        const float4 b0 = __ldg(reinterpret_cast<const float4*>(prm.bias + n0 + 64 * g + 8 * j));
                        const float4 b1 = __ldg(reinterpret_cast<const float4*>(prm.bias + n0 + 64 * g + 8 * j + 4));
                        vals[0] += b0.x; vals[1] += b0.y; vals[2] += b0.z; vals[3] += b0.w;
                        vals[4] += b1.x; vals[5] += b1.y; vals[6] += b1.z; vals[7] += b1.w;
                    }
                    if (prm.act == MF_ACT_GELU) {
#pragma unroll
                        for (int i = 0; i < 8; i += 2) gelu_erf2(vals[i], vals[i + 1]);
                    }
                    if (prm.residual) {
                        const uint32_t rr[4] = {myres[j].x, myres[j].y, myres[j].z, myres[j].w};
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            vals[2 * i] += __uint_as_float(rr[i] << 16);
                            vals[2 * i + 1] += __uint_as_float(rr[i] & 0xffff0000u);
                        }
                    }
                    uint4 o;
                    o.x = ptx::pack_bf16(vals[0], vals[1]);
                    o.y = ptx::pack_bf16(vals[2], vals[3]);
                    o.z = ptx::pack_bf16(vals[4], vals[5]);
                    o.w = ptx::pack_bf16(vals[6], vals[7]);
                    stage[lane * 8 + (j ^ (lane & 7))] = o;
                }
                __syncwarp();
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const int r = 4 * i + crow;
                    if (row0 + r < prm.M)
                        *reinterpret_cast<uint4*>(dst + static_cast<size_t>(row0 + r) * prm.n_split + 64 * g + 8 * cchunk) =
                            stage[r * 8 + (cchunk ^ (r & 7))];
                }
                __syncwarp();
            }
        }
    }
    ptx::tc_fence_before();
    if (kCtas == 2) ptx::cluster_sync();                   // the peer may still be arriving on this CTA's barriers / reading TMEM
    else __syncthreads();
    if (warp == 1) {
        if (kCtas == 2) ptx::tmem_dealloc_pair(tmem, 512);
        else ptx::tmem_dealloc(tmem, 512);
    }
}

}  // namespace mf

// ------------------------------------------------------------------------------------------------
// LayerNorm (reading E4): one warp per row, bf16 in/out, fp32 statistics (two-pass over registers)
// ------------------------------------------------------------------------------------------------
namespace mf {

template <int VEC>      // d = 32 * 8 * VEC channels: each lane holds VEC 16-byte chunks
__global__ void __launch_bounds__(256)
layernorm_kernel(const __nv_bfloat16* __restrict__ x, const float* __restrict__ gamma, const float* __restrict__ beta,
                 float eps, __nv_bfloat16* __restrict__ out, int M) {
    const int row = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (row >= M) return;
    constexpr int d = 32 * 8 * VEC;
    const uint4* src = reinterpret_cast<const uint4*>(x + static_cast<size_t>(row) * d);
    float v[8 * VEC];
    float sum = 0.f;
#pragma unroll
    for (int c = 0; c < VEC; ++c) {
        const uint4 u = __ldg(src + c * 32 + lane);
        const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            v[8 * c + 2 * i] = __uint_as_float(w[i] << 16);
            v[8 * c + 2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
            sum += v[8 * c + 2 * i] + v[8 * c + 2 * i + 1];
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
    const float mean = sum * (1.0f / d);
    float sq = 0.f;
#pragma unroll
    for (int i = 0; i < 8 * VEC; ++i) {
        v[i] -= mean;
        sq = fmaf(v[i], v[i], sq);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sq += __shfl_xor_sync(0xffffffffu, sq, o);
    const float rstd = rsqrtf(sq * (1.0f / d) + eps);
    uint4* dst = reinterpret_cast<uint4*>(out + static_cast<size_t>(row) * d);
#pragma unroll
    for (int c = 0; c < VEC; ++c) {
        const int ch = (c * 32 + lane) * 8;
        const float4 g0 = __ldg(reinterpret_cast<const float4*>(gamma + ch)), g1 = __ldg(reinterpret_cast<const float4*>(gamma + ch + 4));
        const float4 b0 = __ldg(reinterpret_cast<const float4*>(beta + ch)), b1 = __ldg(reinterpret_cast<const float4*>(beta + ch + 4));
        const float g[8] = {g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w};
        const float b[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
        float y[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) y[i] = fmaf(v[8 * c + i] * rstd, g[i], b[i]);
        uint4 o;
        o.x = ptx::pack_bf16(y[0], y[1]);
        o.y = ptx::pack_bf16(y[2], y[3]);
        o.z = ptx::pack_bf16(y[4], y[5]);
        o.w = ptx::pack_bf16(y[6], y[7]);
        dst[c * 32 + lane] = o;
    }
}

// bf16 [rows, K] row-major -> 2-D map (k, row), box = 64 x box_rows, SWIZZLE_128B, zero OOB fill
static mf_status make_map_2d(CUtensorMap* map, const void* base, long long rows, int K, int box_rows) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return fail(MF_ERR_CUDA, "cuTensorMapEncodeTiled entry point not available");
    cuuint64_t dims[2] = {static_cast<cuuint64_t>(K), static_cast<cuuint64_t>(rows)};
    cuuint64_t strides[1] = {static_cast<cuuint64_t>(K) * 2};
    cuuint32_t box[2] = {static_cast<cuuint32_t>(kGK), static_cast<cuuint32_t>(box_rows)};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(MF_ERR_CUDA, "cuTensorMapEncodeTiled failed (CUresult %d)", static_cast<int>(r));
    return MF_OK;
}

}  // namespace mf

namespace mf {
// the opt-in shared-memory size is a per-device attribute of each kernel instantiation: set it once per device
template <typename K>
static cudaError_t ensure_smem(K kernel, int smem, int slot) {
    static std::atomic<bool> done[2][64];
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64 || !done[slot][dev].load(std::memory_order_acquire)) {
        e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) done[slot][dev].store(true, std::memory_order_release);
    }
    return cudaSuccess;
}
}  // namespace mf

extern "C" mf_status mf_linear(const void* x, const void* w, const float* bias, const void* residual, void* out0,
                               void* out1, void* out2, int M, int N, int K, int n_split, mf_activation act,
                               void* stream) {
    using namespace mf;
    if (!x || !w || !out0) return fail(MF_ERR_INVALID_ARG, "mf_linear: NULL tensor");
    if (M < 1 || N < 1 || K < 1 || n_split < 1) return fail(MF_ERR_INVALID_ARG, "mf_linear: non-positive dimension");
    if (act != MF_ACT_NONE && act != MF_ACT_GELU) return fail(MF_ERR_INVALID_ARG, "mf_linear: bad activation %d", static_cast<int>(act));
    if (N % n_split != 0 || N / n_split > 3) return fail(MF_ERR_INVALID_ARG, "mf_linear: N must be 1..3 x n_split");
    const int parts = N / n_split;
    if ((parts > 1 && !out1) || (parts > 2 && !out2)) return fail(MF_ERR_INVALID_ARG, "mf_linear: missing output tensor");
    if (residual && parts != 1) return fail(MF_ERR_INVALID_ARG, "mf_linear: residual needs a single output");
    if (K % kGK != 0 || n_split % kGN != 0)
        return fail(MF_ERR_UNSUPPORTED, "mf_linear: K %% 64 == 0 and n_split %% 256 == 0 required (K=%d, n_split=%d)", K, n_split);
    if (!aligned16(x) || !aligned16(w) || !aligned16(out0) || (out1 && !aligned16(out1)) || (out2 && !aligned16(out2)) ||
        (bias && !aligned16(bias)) || (residual && !aligned16(residual)))
        return fail(MF_ERR_ALIGNMENT, "mf_linear: tensors must be 16-byte aligned");
    if (out0 == x || out1 == x || out2 == x) return fail(MF_ERR_INVALID_ARG, "mf_linear: output aliases x");
    mf_status st = require_sm100();
    if (st != MF_OK) return st;
    CUtensorMap mx, mw;
    // CTA pairs (256 x 256 tiles) unless the problem is a single 128-row band or MF_LINEAR_CTAS=1 asks for the 1-CTA kernel
    static const int forced = [] { const char* e = getenv("MF_LINEAR_CTAS"); return e ? atoi(e) : 0; }();
    const int ctas = forced == 1 ? 1 : (forced == 2 ? 2 : (M > kGM ? 2 : 1));
    if ((st = make_map_2d(&mx, x, M, K, kGM)) != MF_OK) return st;
    if ((st = make_map_2d(&mw, w, N, K, kGN / ctas)) != MF_OK) return st;
    GemmParams prm;
    prm.M = M; prm.N = N; prm.K = K; prm.n_split = n_split;
    prm.m_tiles = (M + ctas * kGM - 1) / (ctas * kGM);
    prm.n_tiles = N / kGN;
    prm.bias = bias;
    prm.residual = static_cast<const __nv_bfloat16*>(residual);
    prm.out[0] = static_cast<__nv_bfloat16*>(out0);
    prm.out[1] = static_cast<__nv_bfloat16*>(out1);
    prm.out[2] = static_cast<__nv_bfloat16*>(out2);
    prm.act = act;
    const long long tiles = static_cast<long long>(prm.m_tiles) * prm.n_tiles;
    if (tiles > 0x7fffffffLL) return fail(MF_ERR_UNSUPPORTED, "mf_linear: too many tiles");
    cudaStream_t cs = static_cast<cudaStream_t>(stream);
    if (ctas == 1) {
        const int grid = static_cast<int>(tiles < sm_count() ? tiles : sm_count());
        const int smem = static_cast<int>(sizeof(GemmSmem<1>)) + 1024;
        MF_CUDA_OK(ensure_smem(linear_kernel<1>, smem, 0));
        linear_kernel<1><<<grid, kGThreads, smem, cs>>>(mx, mw, prm);
    } else {
        const int pairs = static_cast<int>(tiles < sm_count() / 2 ? tiles : sm_count() / 2);
        const int smem = static_cast<int>(sizeof(GemmSmem<2>)) + 1024;
        MF_CUDA_OK(ensure_smem(linear_kernel<2>, smem, 1));
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(2 * pairs);
        cfg.blockDim = dim3(kGThreads);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = cs;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 2;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        MF_CUDA_OK(cudaLaunchKernelEx(&cfg, linear_kernel<2>, mx, mw, prm));
    }
    MF_CUDA_OK(cudaGetLastError());
    return MF_OK;
}

extern "C" mf_status mf_layernorm(const void* x, const float* gamma, const float* beta, float eps, void* out, int M,
                                  int d, void* stream) {
    using namespace mf;
    if (!x || !gamma || !beta || !out) return fail(MF_ERR_INVALID_ARG, "mf_layernorm: NULL tensor");
    if (M < 1 || d < 1 || !(eps >= 0.f)) return fail(MF_ERR_INVALID_ARG, "mf_layernorm: bad dimension or eps");
    if (!aligned16(x) || !aligned16(out) || !aligned16(gamma) || !aligned16(beta))
        return fail(MF_ERR_ALIGNMENT, "mf_layernorm: tensors must be 16-byte aligned");
    mf_status st = require_sm100();
    if (st != MF_OK) return st;
    const unsigned grid = static_cast<unsigned>((static_cast<long long>(M) * 32 + 255) / 256);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const __nv_bfloat16* xi = static_cast<const __nv_bfloat16*>(x);
    __nv_bfloat16* xo = static_cast<__nv_bfloat16*>(out);
    switch (d) {
        case 256: layernorm_kernel<1><<<grid, 256, 0, s>>>(xi, gamma, beta, eps, xo, M); break;
        case 512: layernorm_kernel<2><<<grid, 256, 0, s>>>(xi, gamma, beta, eps, xo, M); break;
        case 768: layernorm_kernel<3><<<grid, 256, 0, s>>>(xi, gamma, beta, eps, xo, M); break;
        case 1024: layernorm_kernel<4><<<grid, 256, 0, s>>>(xi, gamma, beta, eps, xo, M); break;
        default: return fail(MF_ERR_UNSUPPORTED, "mf_layernorm: d=%d (256, 512, 768, 1024 are built)", d);
    }
    MF_CUDA_OK(cudaGetLastError());
    return MF_OK;
}

// ------------------------------------------------------------------------------------------------
// One transformer block (reading E1, E2, E5): host-side sequencing of the seven launches
// ------------------------------------------------------------------------------------------------
static size_t block_tokens_bytes(long long tokens, int width) { return (static_cast<size_t>(tokens) * width * 2 + 255) / 256 * 256; }

extern "C" size_t mf_block_workspace_size(int windows, int frames_per_window, int tokens_per_frame, int d_model, int d_hidden) {
    if (windows < 1 || frames_per_window < 1 || tokens_per_frame < 1 || d_model < 1 || d_hidden < 1) return 0;
    const long long tokens = static_cast<long long>(windows) * frames_per_window * tokens_per_frame;
    return 6 * block_tokens_bytes(tokens, d_model) + block_tokens_bytes(tokens, d_hidden);     // a, q, k, v, o, h | u
}

extern "C" mf_status mf_block_forward(const void* x, const mf_block_weights* wt, void* y, int windows, int frames_per_window,
                                      int tokens_per_frame, int heads, int head_dim, int d_hidden, mf_attn_mode mode,
                                      float ln_eps, void* workspace, size_t workspace_bytes, void* stream) {
    using namespace mf;
    if (!x || !wt || !y) return fail(MF_ERR_INVALID_ARG, "mf_block_forward: NULL tensor");
    if (windows < 1 || frames_per_window < 1 || tokens_per_frame < 1 || heads < 1 || head_dim < 1 || d_hidden < 1)
        return fail(MF_ERR_INVALID_ARG, "mf_block_forward: non-positive dimension");
    if (!wt->ln1_gamma || !wt->ln1_beta || !wt->w_qkv || !wt->w_o || !wt->ln2_gamma || !wt->ln2_beta || !wt->w_1 || !wt->w_2)
        return fail(MF_ERR_INVALID_ARG, "mf_block_forward: NULL weight");
    const int d = heads * head_dim;
    const long long tokens_ll = static_cast<long long>(windows) * frames_per_window * tokens_per_frame;
    if (tokens_ll > 0x7fffffffLL) return fail(MF_ERR_UNSUPPORTED, "mf_block_forward: too many tokens");
    const int tokens = static_cast<int>(tokens_ll);
    const size_t need = mf_block_workspace_size(windows, frames_per_window, tokens_per_frame, d, d_hidden);
    if (!workspace || workspace_bytes < need || !aligned16(workspace))
        return fail(MF_ERR_WORKSPACE, "mf_block_forward: workspace needs %zu bytes (got %zu)", need, workspace_bytes);
    char* base = static_cast<char*>(workspace);
    const size_t td = block_tokens_bytes(tokens, d);
    void *a = base, *q = base + td, *k = base + 2 * td, *v = base + 3 * td, *o = base + 4 * td, *h = base + 5 * td, *u = base + 6 * td;
    mf_status st;
    if ((st = mf_layernorm(x, wt->ln1_gamma, wt->ln1_beta, ln_eps, a, tokens, d, stream)) != MF_OK) return st;
    if ((st = mf_linear(a, wt->w_qkv, wt->b_qkv, nullptr, q, k, v, tokens, 3 * d, d, d, MF_ACT_NONE, stream)) != MF_OK) return st;
    if ((st = mf_window_attention(q, k, v, o, nullptr, windows, frames_per_window, tokens_per_frame, heads, head_dim, mode, 0.f,
                                  stream)) != MF_OK) return st;
    if ((st = mf_linear(o, wt->w_o, wt->b_o, x, h, nullptr, nullptr, tokens, d, d, d, MF_ACT_NONE, stream)) != MF_OK) return st;
    if ((st = mf_layernorm(h, wt->ln2_gamma, wt->ln2_beta, ln_eps, a, tokens, d, stream)) != MF_OK) return st;
    if ((st = mf_linear(a, wt->w_1, wt->b_1, nullptr, u, nullptr, nullptr, tokens, d_hidden, d, d_hidden, MF_ACT_GELU, stream)) != MF_OK)
        return st;
    return mf_linear(u, wt->w_2, wt->b_2, h, y, nullptr, nullptr, tokens, d, d_hidden, d, MF_ACT_NONE, stream);
}
