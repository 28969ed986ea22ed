// mf_motion_focus: Eq. 1-7 + motion-guided depth, four launches on the caller's stream:
//   1. points_kernel   Eq. 1,3,4,6 per rendered frame in fp64 (bit-exact rules of common.h);
//                      (u_i, v_i, sigma_i) rounded once to fp32, focus_uv / focus_index written.
//   2. tables_kernel   separable factors of Eq. 7: Ex[f][i][x], EyT[f][y][i] evaluated in fp64,
//                      stored fp32.  Each point's factors are normalised to peak 1 over the image
//                      and carry a relative weight w_i <= 1, so far-off-image points cannot
//                      underflow the whole map (the common factor cancels in M = U/Z).
//   3. norm_kernel     Z per frame: MAX by an exact branch-and-bound over 32x32 tiles (a tile is
//                      evaluated only if its separable upper bound can beat the best centre
//                      value), SUM in closed form from the tables.  Moves no image bytes.
//   4. render_kernel   the HBM-bound pass: read depth (128-bit), U = sum_i Ex_i[x] EyT[y][i],
//                      write M = U/Z and G = M*D (128-bit, streaming stores).  12 B/pixel.
#include "common.h"

#include <cfloat>
#include <cmath>

namespace mf {

constexpr int kMaxPoints = 32;
constexpr int kTile = 32;                 // branch-and-bound tile edge (pixels)

struct FrameMeta {
    int n_valid;
    float inv_z;        // 1/Z' of the rescaled map
    float out_scale;    // exp(cmax): only applied for MF_NORM_NONE
    int pad;
};

struct Workspace {
    float4* pts;        // [count][kMaxPoints]  (u, v, sigma, 0), valid points first
    FrameMeta* meta;    // [count]
    float* ex;          // [count][npad][width]
    float* eyt;         // [count][height][npad]
};

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
static inline int pad_points(int n) { return (n + 7) / 8 * 8; }

static size_t carve(void* base, int count, int width, int height, int n_points, Workspace* ws) {
    const int npad = pad_points(n_points);
    size_t off = 0;
    char* b = static_cast<char*>(base);
    size_t s_pts = align_up(sizeof(float4) * kMaxPoints * static_cast<size_t>(count), 256);
    size_t s_meta = align_up(sizeof(FrameMeta) * static_cast<size_t>(count), 256);
    size_t s_ex = align_up(sizeof(float) * static_cast<size_t>(count) * npad * width, 256);
    size_t s_ey = align_up(sizeof(float) * static_cast<size_t>(count) * npad * height, 256);
    if (ws) {
        ws->pts = reinterpret_cast<float4*>(b + off);
    }
    off += s_pts;
    if (ws) ws->meta = reinterpret_cast<FrameMeta*>(b + off);
    off += s_meta;
    if (ws) ws->ex = reinterpret_cast<float*>(b + off);
    off += s_ex;
    if (ws) ws->eyt = reinterpret_cast<float*>(b + off);
    off += s_ey;
    return off;
}

// ------------------------------------------------------------------------------------------------
// 1. points (fp64, one warp per rendered frame, one lane per trailing point)
// ------------------------------------------------------------------------------------------------
struct PointParams {
    double fx, fy, cx, cy, eps_z, sigma;
    int n_points, vec, mag, pts, width, height, render_begin, count;
};

__device__ __forceinline__ void load_centre(const double* __restrict__ m, double p[3]) {
    // Eq. 1: p = -R^T t
#pragma unroll
    for (int c = 0; c < 3; ++c) p[c] = -dot3(m[c], m[4 + c], m[8 + c], m[3], m[7], m[11]);
}

__device__ __forceinline__ double norm3(const double a[3]) {
    return __dsqrt_rn(dadd(dadd(dmul(a[0], a[0]), dmul(a[1], a[1])), dmul(a[2], a[2])));
}

__global__ void __launch_bounds__(128)
points_kernel(const double* __restrict__ w2c, PointParams pp, float4* __restrict__ pts, FrameMeta* __restrict__ meta,
              float* __restrict__ focus_uv, int32_t* __restrict__ focus_index) {
    // one warp per rendered frame; lane = slot in the trailing window (oldest first), n_points <= 32
    const int f = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (f >= pp.count) return;
    const int t = pp.render_begin + f;
    const int i = t - pp.n_points + 1 + lane;
    const int need = pp.vec == MF_VEC_ACCEL ? 2 : 1;
    bool valid = lane < pp.n_points && i >= need;
    double u = 0.0, v = 0.0, sig = 0.0;
    if (valid) {
        double p0[3], p1[3], aw[3];
        load_centre(w2c + static_cast<size_t>(i) * 16, p0);
        load_centre(w2c + static_cast<size_t>(i - 1) * 16, p1);
        if (pp.vec == MF_VEC_ACCEL) {
            double p2[3];
            load_centre(w2c + static_cast<size_t>(i - 2) * 16, p2);
#pragma unroll
            for (int c = 0; c < 3; ++c) aw[c] = dsub(dsub(p0[c], p1[c]), dsub(p1[c], p2[c]));   // Eq. 2-3
        } else {
#pragma unroll
            for (int c = 0; c < 3; ++c) aw[c] = dsub(p0[c], p1[c]);
        }
        const double s = norm3(aw);
        if (s < 1e-12) valid = false;
        const double* r = w2c + static_cast<size_t>(pp.pts == MF_PTS_CURRENT_FRAME ? t : i) * 16;
        double ac[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) ac[c] = dot3(r[4 * c], r[4 * c + 1], r[4 * c + 2], aw[0], aw[1], aw[2]);   // Eq. 4
        const double nc = norm3(ac);
        if (fabs(ac[2]) <= dmul(pp.eps_z, nc)) valid = false;
        u = dadd(pp.cx, dmul(pp.fx, ddiv(ac[0], ac[2])));                                                // Eq. 6
        v = dadd(pp.cy, dmul(pp.fy, ddiv(ac[1], ac[2])));
        sig = pp.mag == MF_MAG_RAW ? dmul(pp.sigma, s) : pp.sigma;
        if (sig < 1e-3) sig = 1e-3;
    }
    const unsigned mask = __ballot_sync(0xffffffffu, valid);
    if (valid)
        pts[static_cast<size_t>(f) * kMaxPoints + __popc(mask & ((1u << lane) - 1u))] =
            make_float4(__double2float_rn(u), __double2float_rn(v), __double2float_rn(sig), 0.f);
    if (lane == 0) meta[f].n_valid = __popc(mask);
    if (lane == pp.n_points - 1) {                      // the frame's own point (i == t)
        int index = -1;
        float fu = __int_as_float(0x7fc00000), fv = __int_as_float(0x7fc00000);
        if (valid) {
            fu = __double2float_rn(u);
            fv = __double2float_rn(v);
            if (isfinite(u) && isfinite(v)) {
                const double x = floor(dadd(u, 0.5));
                const double y = floor(dadd(v, 0.5));
                if (x >= 0.0 && x < static_cast<double>(pp.width) && y >= 0.0 && y < static_cast<double>(pp.height))
                    index = static_cast<int>(y) * pp.width + static_cast<int>(x);
            }
        }
        if (focus_uv) {
            focus_uv[2 * f] = fu;
            focus_uv[2 * f + 1] = fv;
        }
        if (focus_index) focus_index[f] = index;
    }
}

// ------------------------------------------------------------------------------------------------
// 2. separable tables (fp64 evaluation, fp32 storage).  grid = (npad, count), one (frame, slot) each.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double nearest_in_range(double u, int hi) {
    // integer coordinate in [0, hi] nearest to u
    double r = rint(u);
    r = r < 0.0 ? 0.0 : r;
    r = r > static_cast<double>(hi) ? static_cast<double>(hi) : r;
    return r;
}

// log of point j's peak value over the image's pixel grid; -inf if the point is unusable
__device__ __forceinline__ double log_peak(float4 p, int width, int height, double* dxmin, double* dymin) {
    const double u = p.x, v = p.y, s = p.z;
    if (!isfinite(u) || !isfinite(v) || !(s > 0.0) || !isfinite(s)) {
        *dxmin = 0.0;
        *dymin = 0.0;
        return -INFINITY;
    }
    *dxmin = nearest_in_range(u, width - 1) - u;
    *dymin = nearest_in_range(v, height - 1) - v;
    return -((*dxmin) * (*dxmin) + (*dymin) * (*dymin)) / (2.0 * s * s);
}

__global__ void __launch_bounds__(256)
tables_kernel(const float4* __restrict__ pts, FrameMeta* __restrict__ meta, float* __restrict__ ex,
              float* __restrict__ eyt, int npad, int width, int height) {
    const int j = blockIdx.x, f = blockIdx.y;
    const int n_valid = meta[f].n_valid;
    const float4* fp = pts + static_cast<size_t>(f) * kMaxPoints;
    // common factor exp(cmax) pulled out of every point of this frame (cancels in U/Z)
    double cmax = -INFINITY, dx0 = 0.0, dy0 = 0.0, lw_j = -INFINITY;
    for (int k = 0; k < n_valid; ++k) {
        double a, b;
        const double lw = log_peak(fp[k], width, height, &a, &b);
        cmax = lw > cmax ? lw : cmax;
        if (k == j) {
            lw_j = lw;
            dx0 = a;
            dy0 = b;
        }
    }
    const bool frame_empty = !(cmax > -700.0);          // fp64 Eq. 7 underflows to 0 everywhere
    if (j == 0 && threadIdx.x == 0) {
        meta[f].out_scale = frame_empty ? 0.f : static_cast<float>(exp(cmax));
        meta[f].pad = frame_empty ? 1 : 0;
    }
    float* exr = ex + (static_cast<size_t>(f) * npad + j) * width;
    float* eyc = eyt + static_cast<size_t>(f) * height * npad + j;
    const bool live = j < n_valid && !frame_empty && lw_j > -INFINITY;
    if (!live) {
        for (int x = threadIdx.x; x < width; x += blockDim.x) exr[x] = 0.f;
        for (int y = threadIdx.x; y < height; y += blockDim.x) eyc[static_cast<size_t>(y) * npad] = 0.f;
        return;
    }
    const double u = fp[j].x, v = fp[j].y, s = fp[j].z;
    const double inv = 1.0 / (2.0 * s * s);
    const double w = exp(lw_j - cmax);
    for (int x = threadIdx.x; x < width; x += blockDim.x) {
        const double d = static_cast<double>(x) - u;
        exr[x] = static_cast<float>(exp(-(d * d - dx0 * dx0) * inv));
    }
    for (int y = threadIdx.x; y < height; y += blockDim.x) {
        const double d = static_cast<double>(y) - v;
        eyc[static_cast<size_t>(y) * npad] = static_cast<float>(w * exp(-(d * d - dy0 * dy0) * inv));
    }
}

// ------------------------------------------------------------------------------------------------
// 3. per-frame normaliser.  grid = count, 256 threads, dynamic smem = npad*(TC+TR) floats.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

__device__ __forceinline__ int clamp_round(float u, int lo, int hi) {
    return static_cast<int>(fminf(fmaxf(rintf(u), static_cast<float>(lo)), static_cast<float>(hi)));
}

// U'(x,y) with the SAME fma chain as render_kernel (so that max M == Zmax * inv_z)
__device__ __forceinline__ float eval_pixel(const float* __restrict__ exf, const float* __restrict__ eyrow,
                                            int npad, int width, int x) {
    float acc = 0.f;
    for (int k = 0; k < npad; ++k) acc = fmaf(exf[static_cast<size_t>(k) * width + x], eyrow[k], acc);
    return acc;
}

__global__ void __launch_bounds__(256)
norm_kernel(const float4* __restrict__ pts, FrameMeta* __restrict__ meta, const float* __restrict__ ex,
            const float* __restrict__ eyt, int npad, int width, int height, int norm) {
    extern __shared__ float sm_f[];
    __shared__ float s_red[8];
    __shared__ double s_dred[8];
    const int f = blockIdx.x;
    const int n_valid = meta[f].n_valid;
    const float* exf = ex + static_cast<size_t>(f) * npad * width;
    const float* eyf = eyt + static_cast<size_t>(f) * height * npad;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (n_valid == 0 || meta[f].pad != 0) {
        if (threadIdx.x == 0) meta[f].inv_z = 0.f;
        return;
    }
    if (norm == MF_NORM_NONE) {
        if (threadIdx.x == 0) meta[f].inv_z = meta[f].out_scale;
        return;
    }
    if (norm == MF_NORM_SUM) {
        // sum_xy U' = sum_j (sum_x Ex_j)(sum_y Ey_j), closed form from the tables, fp64
        double total = 0.0;
        for (int j = 0; j < n_valid; ++j) {
            double sx = 0.0, sy = 0.0;
            for (int x = threadIdx.x; x < width; x += blockDim.x) sx += exf[static_cast<size_t>(j) * width + x];
            for (int y = threadIdx.x; y < height; y += blockDim.x) sy += eyf[static_cast<size_t>(y) * npad + j];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                sx += __shfl_xor_sync(0xffffffffu, sx, o);
                sy += __shfl_xor_sync(0xffffffffu, sy, o);
            }
            __syncthreads();
            if (lane == 0) s_dred[warp] = sx;
            __syncthreads();
            double bx = 0.0;
            for (int w = 0; w < 8; ++w) bx += s_dred[w];
            __syncthreads();
            if (lane == 0) s_dred[warp] = sy;
            __syncthreads();
            double by = 0.0;
            for (int w = 0; w < 8; ++w) by += s_dred[w];
            total += bx * by;
        }
        if (threadIdx.x == 0) meta[f].inv_z = total > 0.0 ? static_cast<float>(1.0 / total) : 0.f;
        return;
    }
    // ---- MF_NORM_MAX ----
    const int tc = (width + kTile - 1) / kTile, tr = (height + kTile - 1) / kTile;
    float* mx = sm_f;                       // [npad][tc] max over the tile's columns of Ex_j
    float* my = sm_f + npad * tc;           // [npad][tr]
    const float4* fp = pts + static_cast<size_t>(f) * kMaxPoints;
    for (int i = threadIdx.x; i < npad * tc; i += blockDim.x) {
        const int j = i / tc, c = i % tc;
        float val = 0.f;
        if (j < n_valid) {
            const int x0 = c * kTile, x1 = min(x0 + kTile, width) - 1;
            val = exf[static_cast<size_t>(j) * width + clamp_round(fp[j].x, x0, x1)];
        }
        mx[i] = val;
    }
    for (int i = threadIdx.x; i < npad * tr; i += blockDim.x) {
        const int j = i / tr, r = i % tr;
        float val = 0.f;
        if (j < n_valid) {
            const int y0 = r * kTile, y1 = min(y0 + kTile, height) - 1;
            val = eyf[static_cast<size_t>(clamp_round(fp[j].y, y0, y1)) * npad + j];
        }
        my[i] = val;
    }
    // lower bound: the map at the pixel nearest to each centre
    float best = 0.f;
    if (warp == 0) {
        if (lane < n_valid) {
            const int x = clamp_round(fp[lane].x, 0, width - 1), y = clamp_round(fp[lane].y, 0, height - 1);
            best = eval_pixel(exf, eyf + static_cast<size_t>(y) * npad, npad, width, x);
        }
        best = warp_max(best);
        if (lane == 0) s_red[0] = best;
    }
    __syncthreads();
    best = s_red[0];
    __syncthreads();
    // each lane bounds one tile; surviving tiles are then evaluated by the whole warp
    const int n_tiles = tc * tr;
    for (int base = warp * 32; base < n_tiles; base += 8 * 32) {
        const int mine = base + lane;
        float ub = 0.f;
        if (mine < n_tiles) {
            const int c = mine % tc, r = mine / tc;
            for (int k = 0; k < npad; ++k) ub = fmaf(mx[k * tc + c], my[k * tr + r], ub);
        } else {
            ub = -1.f;
        }
        unsigned surv = __ballot_sync(0xffffffffu, ub * 1.00001f >= best);
        while (surv) {
            const int src = __ffs(surv) - 1;
            surv &= surv - 1;
            if (__shfl_sync(0xffffffffu, ub, src) * 1.00001f < best) continue;     // best may have grown
            const int tile = base + src;
            const int c = tile % tc, r = tile / tc;
            const int x = min(c * kTile + lane, width - 1);                         // duplicates are harmless for a max
            const int y0 = r * kTile, y1 = min(y0 + kTile, height);
            float local = 0.f;
            float e[kMaxPoints];
#pragma unroll
            for (int k = 0; k < kMaxPoints; ++k) e[k] = k < npad ? exf[static_cast<size_t>(k) * width + x] : 0.f;
            for (int y = y0; y < y1; ++y) {
                const float4* row = reinterpret_cast<const float4*>(eyf + static_cast<size_t>(y) * npad);
                float acc = 0.f;
#pragma unroll
                for (int q = 0; q < kMaxPoints / 4; ++q) {
                    if (4 * q < npad) {
                        const float4 w = __ldg(row + q);
                        acc = fmaf(e[4 * q + 0], w.x, acc);
                        acc = fmaf(e[4 * q + 1], w.y, acc);
                        acc = fmaf(e[4 * q + 2], w.z, acc);
                        acc = fmaf(e[4 * q + 3], w.w, acc);
                    }
                }
                local = fmaxf(local, acc);
            }
            best = fmaxf(best, warp_max(local));
        }
    }
    if (lane == 0) s_red[warp] = best;
    __syncthreads();
    if (threadIdx.x == 0) {
        float z = 0.f;
        for (int w = 0; w < 8; ++w) z = fmaxf(z, s_red[w]);
        meta[f].inv_z = z > 0.f ? 1.0f / z : 0.f;
    }
}

// ------------------------------------------------------------------------------------------------
// 4. render: the streaming pass.  One thread owns 4 adjacent columns (one 128-bit access per image
//    row) over kRowsPerThread rows; the 4*NP column factors stay in registers, the NP row factors
//    of each row are a broadcast 128-bit read of EyT (L1-resident).  Algorithmic HBM traffic is
//    12 B/pixel with depth and guided depth, 4 B/pixel map-only.
// ------------------------------------------------------------------------------------------------
constexpr int kRowsPerThread = 32;
constexpr int kRenderThreads = 256;

__device__ __forceinline__ float4 ld_stream(const float4* p) {
    float4 r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::128B.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ void st_stream(float4* p, float4 v) {
    asm volatile("st.global.cs.v4.f32 [%0], {%1,%2,%3,%4};" :: "l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

template <int NP, bool HAS_DEPTH, bool HAS_G>
__global__ void __launch_bounds__(kRenderThreads)
render_kernel(const float* __restrict__ ex, const float* __restrict__ eyt, const FrameMeta* __restrict__ meta,
              const float* __restrict__ depth, float* __restrict__ focus_map, float* __restrict__ guided,
              int width, int height, int blocks_per_frame) {
    const int f = blockIdx.x / blocks_per_frame;
    const int b = blockIdx.x - f * blocks_per_frame;
    const int wq = width >> 2;
    const int idx = b * kRenderThreads + threadIdx.x;
    const int rb = idx / wq;
    const int x = (idx - rb * wq) << 2;
    const int y0 = rb * kRowsPerThread;
    if (y0 >= height) return;
    const int y1 = min(y0 + kRowsPerThread, height);
    const float scale = meta[f].inv_z;

    float4 e[NP];
    const float* exf = ex + static_cast<size_t>(f) * NP * width + x;
#pragma unroll
    for (int j = 0; j < NP; ++j) e[j] = __ldg(reinterpret_cast<const float4*>(exf + static_cast<size_t>(j) * width));

    const size_t img = static_cast<size_t>(f) * height * width + x;
    const float4* eyrow = reinterpret_cast<const float4*>(eyt + (static_cast<size_t>(f) * height + y0) * NP);
    constexpr int U = 4;
    for (int y = y0; y < y1; y += U) {
        float4 d[U];
        if (HAS_DEPTH) {
#pragma unroll
            for (int r = 0; r < U; ++r)
                if (y + r < y1) d[r] = ld_stream(reinterpret_cast<const float4*>(depth + img + static_cast<size_t>(y + r) * width));
        }
#pragma unroll
        for (int r = 0; r < U; ++r) {
            if (y + r < y1) {
                float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                for (int q = 0; q < NP / 4; ++q) {
                    const float4 w = __ldg(eyrow + (y - y0 + r) * (NP / 4) + q);
                    const float wy[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        acc.x = fmaf(e[4 * q + k].x, wy[k], acc.x);
                        acc.y = fmaf(e[4 * q + k].y, wy[k], acc.y);
                        acc.z = fmaf(e[4 * q + k].z, wy[k], acc.z);
                        acc.w = fmaf(e[4 * q + k].w, wy[k], acc.w);
                    }
                }
                const float4 m = make_float4(acc.x * scale, acc.y * scale, acc.z * scale, acc.w * scale);
                const size_t o = img + static_cast<size_t>(y + r) * width;
                st_stream(reinterpret_cast<float4*>(focus_map + o), m);
                if (HAS_G)
                    st_stream(reinterpret_cast<float4*>(guided + o),
                              make_float4(m.x * d[r].x, m.y * d[r].y, m.z * d[r].z, m.w * d[r].w));
            }
        }
    }
}

template <int NP>
static void launch_render(const Workspace& ws, const float* depth, float* focus_map, float* guided, int count,
                          int width, int height, cudaStream_t stream) {
    const int row_blocks = (height + kRowsPerThread - 1) / kRowsPerThread;
    const long long threads = static_cast<long long>(width / 4) * row_blocks;
    const int bpf = static_cast<int>((threads + kRenderThreads - 1) / kRenderThreads);
    const unsigned grid = static_cast<unsigned>(bpf) * static_cast<unsigned>(count);
    if (guided)
        render_kernel<NP, true, true><<<grid, kRenderThreads, 0, stream>>>(ws.ex, ws.eyt, ws.meta, depth, focus_map,
                                                                            guided, width, height, bpf);
    else
        render_kernel<NP, false, false><<<grid, kRenderThreads, 0, stream>>>(ws.ex, ws.eyt, ws.meta, depth, focus_map,
                                                                              guided, width, height, bpf);
}

}  // namespace mf

extern "C" size_t mf_motion_focus_workspace_size(int count, int width, int height, int n_points) {
    if (count < 1 || width < 1 || height < 1 || n_points < 1 || n_points > mf::kMaxPoints) return 0;
    return mf::carve(nullptr, count, width, height, n_points, nullptr);
}

extern "C" mf_status mf_motion_focus(const double* global_w2c, mf_intrinsics K, int num_frames, int render_begin,
                                     int render_end, int width, int height, const float* depth,
                                     const mf_focus_params* params, float* focus_map, float* guided_depth,
                                     float* focus_uv, int32_t* focus_index, void* workspace, size_t workspace_bytes,
                                     void* stream) {
    using namespace mf;
    if (!global_w2c || !params) return fail(MF_ERR_INVALID_ARG, "mf_motion_focus: NULL poses or params");
    if (num_frames < 1 || render_begin < 0 || render_end > num_frames || render_end <= render_begin)
        return fail(MF_ERR_INVALID_ARG, "mf_motion_focus: bad frame range [%d,%d) of %d", render_begin, render_end,
                    num_frames);
    if (width < 1 || height < 1) return fail(MF_ERR_INVALID_ARG, "mf_motion_focus: bad image size %dx%d", width, height);
    if (params->n_points < 1 || !(params->sigma > 0.f) || !(params->eps_z >= 0.0))
        return fail(MF_ERR_INVALID_ARG, "mf_motion_focus: need n_points>=1, sigma>0, eps_z>=0");
    if (params->n_points > kMaxPoints)
        return fail(MF_ERR_UNSUPPORTED, "mf_motion_focus: n_points=%d > %d", params->n_points, kMaxPoints);
    if (params->vec < 0 || params->vec > 1 || params->mag < 0 || params->mag > 1 || params->norm < 0 ||
        params->norm > 2 || params->pts < 0 || params->pts > 1)
        return fail(MF_ERR_INVALID_ARG, "mf_motion_focus: bad enum in params");
    if (guided_depth && (!depth || !focus_map))
        return fail(MF_ERR_INVALID_ARG, "mf_motion_focus: guided_depth requires depth and focus_map");
    if (focus_map && (width % 4 != 0 || !aligned16(focus_map) || (depth && !aligned16(depth)) ||
                      (guided_depth && !aligned16(guided_depth))))
        return fail(MF_ERR_ALIGNMENT, "mf_motion_focus: width %% 4 == 0 and 16-byte aligned images required");
    const int count = render_end - render_begin;
    const size_t need = carve(nullptr, count, width, height, params->n_points, nullptr);
    if (!workspace || workspace_bytes < need || !aligned16(workspace))
        return fail(MF_ERR_WORKSPACE, "mf_motion_focus: workspace needs %zu bytes (got %zu)", need, workspace_bytes);
    mf_status st = require_sm100();
    if (st != MF_OK) return st;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    Workspace ws;
    carve(workspace, count, width, height, params->n_points, &ws);
    const int npad = pad_points(params->n_points);

    PointParams pp;
    pp.fx = K.fx; pp.fy = K.fy; pp.cx = K.cx; pp.cy = K.cy;
    pp.eps_z = params->eps_z;
    pp.sigma = static_cast<double>(params->sigma);
    pp.n_points = params->n_points; pp.vec = params->vec; pp.mag = params->mag; pp.pts = params->pts;
    pp.width = width; pp.height = height; pp.render_begin = render_begin; pp.count = count;
    points_kernel<<<(count + 3) / 4, 128, 0, s>>>(global_w2c, pp, ws.pts, ws.meta, focus_uv, focus_index);
    MF_CUDA_OK(cudaGetLastError());
    if (!focus_map) return MF_OK;

    tables_kernel<<<dim3(npad, count), 256, 0, s>>>(ws.pts, ws.meta, ws.ex, ws.eyt, npad, width, height);
    MF_CUDA_OK(cudaGetLastError());
    const int tc = (width + kTile - 1) / kTile, tr = (height + kTile - 1) / kTile;
    const size_t smem = sizeof(float) * npad * static_cast<size_t>(tc + tr);
    if (smem > 200 * 1024) return fail(MF_ERR_UNSUPPORTED, "mf_motion_focus: image too large for the bound tables");
    if (smem > 48 * 1024)
        MF_CUDA_OK(cudaFuncSetAttribute(norm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem)));
    norm_kernel<<<count, 256, smem, s>>>(ws.pts, ws.meta, ws.ex, ws.eyt, npad, width, height, params->norm);
    MF_CUDA_OK(cudaGetLastError());
    switch (npad) {
        case 8: launch_render<8>(ws, depth, focus_map, guided_depth, count, width, height, s); break;
        case 16: launch_render<16>(ws, depth, focus_map, guided_depth, count, width, height, s); break;
        case 24: launch_render<24>(ws, depth, focus_map, guided_depth, count, width, height, s); break;
        default: launch_render<32>(ws, depth, focus_map, guided_depth, count, width, height, s); break;
    }
    MF_CUDA_OK(cudaGetLastError());
    return MF_OK;
}
