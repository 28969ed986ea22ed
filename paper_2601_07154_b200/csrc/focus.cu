// mf_motion_focus: Eq. 1-7 + motion-guided depth, three launches on the caller's stream (the second and
// third by programmatic dependent launch):
//   1. tables_kernel   warp 0 of every CTA: Eq. 1,3,4,6 for the frame's trailing points in fp64 (bit-exact rules of
//                      common.h), (u_i, v_i, sigma_i) rounded once to fp32; CTA 0 of the frame publishes them with
//                      focus_uv / focus_index.  Then the separable factors of Eq. 7, Ex[f][i][x] and EyT[f][y][i],
//                      argument in fp64, stored fp32.  Each point's factors are normalised to peak 1 over the image
//                      and carry a relative weight w_i <= 1, so far-off-image points cannot underflow the whole map
//                      (the common factor cancels in M = U/Z).  Factors below 1e-15 of their peak are stored as 0.
//   2. norm_kernel     Z per frame: MAX by an exact branch-and-bound over 32x32 tiles (a tile is evaluated only if
//                      its separable upper bound can beat the best centre value), SUM in closed form from the
//                      tables; also the bounding box outside which every factor is < 1e-13.  Moves no image bytes.
//   3. render_kernel   the HBM-bound pass: read depth (128-bit), U = sum_i Ex_i[x] EyT[y][i] inside the bounding
//                      box and exact zeros outside it, write M = U/Z and G = M*D (128-bit, streaming stores).
//                      12 B/pixel.
// (points_kernel alone runs when no map is requested.)
#include "common.h"

#include <algorithm>
#include <cfloat>
#include <climits>
#include <cmath>

namespace mf {

// Programmatic dependent launch: a kernel launched with launch_pdl() may start while its predecessor on the stream is
// still running; it must call pdl_wait() before touching anything the predecessor wrote.  pdl_trigger() lets the
// successor's CTAs be scheduled early (they then sit in pdl_wait()).  This hides launch latency between the short,
// dependent kernels of one call.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... KArgs, typename... Args>
static cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

constexpr int kMaxPoints = 32;
constexpr int kTile = 32;                 // branch-and-bound tile edge (pixels)
#ifndef MF_NORM_BLOCKS
#define MF_NORM_BLOCKS 8
#endif
constexpr int kNormBlocks = MF_NORM_BLOCKS;            // CTAs per frame in norm_kernel (MF_NORM_MAX tiles are dealt round-robin)
constexpr double kTruncate = 34.5;         // separable factors below e^-34.5 = 1e-15 of their peak are stored as 0
constexpr float kCullBelow = 1e-13f;      // a column factor below this adds < 1e-13 of the map's peak (S8(c)-D3 allows 1e-12)

struct FrameMeta {
    int n_valid;
    float inv_z;        // 1/Z' of the rescaled map (MF_NORM_SUM, MF_NORM_NONE)
    float out_scale;    // exp(cmax): only applied for MF_NORM_NONE
    int pad;            // 1: the whole frame underflows in fp64 (renders as zero)
    unsigned zmax_bits; // MF_NORM_MAX: bit pattern of Z' = max U' (>= 0, so unsigned order == float order)
    int reserved[3];
};

struct Workspace {
    float4* pts;        // [count][kMaxPoints]  (u, v, sigma, 0), valid points first
    FrameMeta* meta;    // [count]
    float* ex;          // [count][npad][width]
    float* eyt;         // [count][height][npad]
    uint32_t* colmask;  // [count][ceil(width/32)]  bit j: point j matters somewhere in this 32-column strip
    uint32_t* rowmask;  // [count][ceil(height/32)]
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
    const size_t tc = (width + kTile - 1) / kTile, tr = (height + kTile - 1) / kTile;
    if (ws) ws->colmask = reinterpret_cast<uint32_t*>(b + off);
    off += align_up(sizeof(uint32_t) * tc * static_cast<size_t>(count), 256);
    if (ws) ws->rowmask = reinterpret_cast<uint32_t*>(b + off);
    off += align_up(sizeof(uint32_t) * tr * static_cast<size_t>(count), 256);
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

// Eq. 1-6 for rendered frame f by one full warp; lane = slot in the trailing window (oldest first), n_points <= 32.
// The valid points are compacted into spts[0..n_valid) (shared memory, (u, v, sigma, 0) rounded once to fp32);
// with `write` they, n_valid, focus_uv and focus_index also go to global memory.  Returns n_valid.
__device__ __forceinline__ int frame_points_warp(const double* __restrict__ w2c, const PointParams& pp, int f, int lane,
                                                 float4* spts, bool write, float4* __restrict__ pts,
                                                 FrameMeta* __restrict__ meta, float* __restrict__ focus_uv,
                                                 int32_t* __restrict__ focus_index) {
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
    const int n_valid = __popc(mask);
    if (valid) {
        const float4 q = make_float4(__double2float_rn(u), __double2float_rn(v), __double2float_rn(sig), 0.f);
        const int slot = __popc(mask & ((1u << lane) - 1u));
        spts[slot] = q;
        if (write) pts[static_cast<size_t>(f) * kMaxPoints + slot] = q;
    }
    __syncwarp();
    if (!write) return n_valid;
    if (lane == 0) {
        meta[f].n_valid = n_valid;
        meta[f].zmax_bits = 0u;
    }
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
    return n_valid;
}

// points only (focus_map == NULL): one warp per rendered frame
__global__ void __launch_bounds__(128)
points_kernel(const double* __restrict__ w2c, PointParams pp, float4* __restrict__ pts, FrameMeta* __restrict__ meta,
              float* __restrict__ focus_uv, int32_t* __restrict__ focus_index) {
    __shared__ float4 spts[4][kMaxPoints];
    const int f = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (f >= pp.count) return;
    frame_points_warp(w2c, pp, f, threadIdx.x & 31, spts[threadIdx.x >> 5], true, pts, meta, focus_uv, focus_index);
}

// ------------------------------------------------------------------------------------------------
// 2. separable tables (fp64 evaluation, fp32 storage).
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

__device__ __forceinline__ int warp_min_i(int v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = min(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ int warp_max_i(int v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = max(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

struct TablePoint {     // per-point constants of the separable factors (fp64)
    double u, v, inv, dx0sq, dy0sq, lw;     // lw = log of the point's weight relative to the frame's strongest point (<= 0)
    int live;
};

// e^-a for 0 <= a <= 40 from an fp64 argument: a*log2(e) = k + r in fp64, 2^-r by ex2.approx on |r| <= 0.5 (fp32,
// ~2 ulp), 2^-k exactly through the exponent field.  Relative error ~3e-7; exactly 1 at a == 0.
__device__ __forceinline__ float exp_neg(double a) {
    const double t = a * 1.4426950408889634;
    const double k = rint(t);
    const float r = static_cast<float>(t - k);
    float p;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(p) : "f"(-r));
    return p * __int_as_float((127 - static_cast<int>(k)) << 23);
}
constexpr int kTableItems = 8;              // table entries per thread

// grid = (chunks, count): a CTA fills kTableItems*256 consecutive entries of the frame's [Ex | EyT] tables, so every
// store is coalesced; the per-point constants are recomputed by warp 0 of every CTA (15 lanes of fp64, ~1 us).
__global__ void __launch_bounds__(256)
tables_kernel(const double* __restrict__ w2c, PointParams pp, float4* __restrict__ pts, FrameMeta* __restrict__ meta,
              float* __restrict__ focus_uv, int32_t* __restrict__ focus_index, float* __restrict__ ex,
              float* __restrict__ eyt, int npad, int width, int height) {
    __shared__ TablePoint tp[kMaxPoints];
    __shared__ float4 spts[kMaxPoints];
    pdl_trigger();
    const int f = blockIdx.y;
    const int lane = threadIdx.x & 31;
    if (threadIdx.x < 32) {
        // the frame's motion points (every CTA recomputes them; CTA 0 of the frame publishes them)
        const int n_valid = frame_points_warp(w2c, pp, f, lane, spts, blockIdx.x == 0, pts, meta, focus_uv, focus_index);
        // common factor exp(cmax) pulled out of every point of this frame (cancels in U/Z)
        double dx0 = 0.0, dy0 = 0.0, lw = -INFINITY;
        float4 p = make_float4(0.f, 0.f, 1.f, 0.f);
        if (lane < n_valid) {
            p = spts[lane];
            lw = log_peak(p, width, height, &dx0, &dy0);
        }
        double cmax = lw;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) cmax = fmax(cmax, __shfl_xor_sync(0xffffffffu, cmax, o));
        const bool frame_empty = !(cmax > -700.0);      // fp64 Eq. 7 underflows to 0 everywhere
        if (blockIdx.x == 0 && lane == 0) {
            meta[f].out_scale = frame_empty ? 0.f : static_cast<float>(exp(cmax));
            meta[f].pad = frame_empty ? 1 : 0;
        }
        TablePoint t;
        const double sg = p.z;
        t.u = p.x; t.v = p.y; t.inv = 1.0 / (2.0 * sg * sg);
        t.dx0sq = dx0 * dx0; t.dy0sq = dy0 * dy0;
        t.live = lane < n_valid && !frame_empty && lw > -INFINITY;
        t.lw = t.live ? lw - cmax : 0.0;
        tp[lane] = t;
    }
    __syncthreads();
    const int n_ex = npad * width, n_all = n_ex + npad * height;
    float* exf = ex + static_cast<size_t>(f) * n_ex;
    float* eyf = eyt + static_cast<size_t>(f) * height * npad;
#pragma unroll
    for (int it = 0; it < kTableItems; ++it) {
        const int idx = (blockIdx.x * kTableItems + it) * 256 + threadIdx.x;
        if (idx < n_ex) {
            const int j = idx / width, x = idx - j * width;
            const TablePoint& t = tp[j];
            const double d = static_cast<double>(x) - t.u;
            const double a = (d * d - t.dx0sq) * t.inv;
            const float val = (!t.live || a > kTruncate) ? 0.f : exp_neg(a);
            exf[idx] = val;
        } else if (idx < n_all) {
            const int i = idx - n_ex;
            const int y = i / npad, j = i - y * npad;
            const TablePoint& t = tp[j];
            const double d = static_cast<double>(y) - t.v;
            const double a = (d * d - t.dy0sq) * t.inv - t.lw;                // the weight folded into the exponent
            const float val = (!t.live || a > kTruncate) ? 0.f : exp_neg(a);
            eyf[i] = val;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// 3. per-frame normaliser.  grid = (kNormBlocks, count), 256 threads, dynamic smem = npad*(TC+TR) floats.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

__device__ __forceinline__ int clamp_round(float u, int lo, int hi) {
    return static_cast<int>(fminf(fmaxf(rintf(u), static_cast<float>(lo)), static_cast<float>(hi)));
}

constexpr int kMaxSurvivors = 256;

// Largest U'(x,y) over one kTile x kTile tile, lane = column, with the SAME fma chain (k ascending) as render_kernel.
// The tile's row factors (contiguous in EyT) are staged in shared memory by the warp: every global load of the tile
// is in flight at once.
__device__ __forceinline__ float eval_tile(const float* __restrict__ exf, const float* __restrict__ eyf, float* buf, int npad,
                                           int width, int height, int tile, int tc, int lane) {
    const int c = tile % tc, r = tile / tc;
    const int x = min(c * kTile + lane, width - 1);                         // duplicates are harmless for a max
    const int y0 = r * kTile, rows = min(y0 + kTile, height) - y0;
    float e[kMaxPoints];
#pragma unroll
    for (int k = 0; k < kMaxPoints; ++k) e[k] = k < npad ? __ldg(exf + static_cast<size_t>(k) * width + x) : 0.f;
    const float4* src = reinterpret_cast<const float4*>(eyf + static_cast<size_t>(y0) * npad);
    const int n4 = rows * npad / 4;
    float4 stage[kTile * kMaxPoints / 4 / 32];
#pragma unroll
    for (int u = 0; u < kTile * kMaxPoints / 4 / 32; ++u)
        if (u * 32 + lane < n4) stage[u] = __ldg(src + u * 32 + lane);
    __syncwarp();                                                           // previous tile's readers are done
#pragma unroll
    for (int u = 0; u < kTile * kMaxPoints / 4 / 32; ++u)
        if (u * 32 + lane < n4) reinterpret_cast<float4*>(buf)[u * 32 + lane] = stage[u];
    __syncwarp();
    float local = 0.f;
    for (int y = 0; y < rows; ++y) {
        const float* row = buf + y * npad;
        float acc = 0.f;
#pragma unroll
        for (int k = 0; k < kMaxPoints; ++k)
            if (k < npad) acc = fmaf(e[k], row[k], acc);
        local = fmaxf(local, acc);
    }
    return local;
}

__global__ void __launch_bounds__(256)
norm_kernel(const float4* __restrict__ pts, FrameMeta* __restrict__ meta, const float* __restrict__ ex,
            const float* __restrict__ eyt, uint32_t* __restrict__ colmask, uint32_t* __restrict__ rowmask, int npad,
            int width, int height, int norm) {
    extern __shared__ float sm_f[];
    __shared__ double s_dred[8];
    __shared__ float4 s_pts[kMaxPoints];
    __shared__ unsigned s_best;             // bit pattern of a lower bound of the frame's maximum
    __shared__ unsigned s_exact;            // bit pattern of the largest exactly evaluated pixel of this CTA
    __shared__ int s_count;
    __shared__ int s_list[kMaxSurvivors];
    pdl_wait();                             // tables_kernel's output
    pdl_trigger();
    const int f = blockIdx.y, part = blockIdx.x;
    const int n_valid = meta[f].n_valid;
    const bool empty = n_valid == 0 || meta[f].pad != 0;
    if (part != 0 && (norm != MF_NORM_MAX || empty)) return;
    const float* exf = ex + static_cast<size_t>(f) * npad * width;
    const float* eyf = eyt + static_cast<size_t>(f) * height * npad;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (empty) {                            // renders as zeros: render_kernel never reads the masks when the scale is 0
        if (threadIdx.x == 0) meta[f].inv_z = 0.f;
        return;
    }
    // Every step below issues all of its (independent) global loads before using any of them: the kernel is a chain
    // of memory latencies, not of arithmetic.
    const int tc = (width + kTile - 1) / kTile, tr = (height + kTile - 1) / kTile;
    float* mx = sm_f;                       // [npad][tc] largest Ex_j over the tile's columns (Ex_j is unimodal)
    float* my = sm_f + npad * tc;           // [npad][tr]
    float* centre = my + npad * tr;         // [kMaxPoints] map value at each centre's pixel
    float* tile_buf = centre + kMaxPoints;  // [8 warps][kTile rows][npad] staged row factors
    if (threadIdx.x < kMaxPoints) {
        s_pts[threadIdx.x] = threadIdx.x < n_valid ? pts[static_cast<size_t>(f) * kMaxPoints + threadIdx.x]
                                                   : make_float4(0.f, 0.f, 1.f, 0.f);
        centre[threadIdx.x] = 0.f;
    }
    if (threadIdx.x == 0) {
        s_best = 0u;
        s_exact = 0u;
        s_count = 0;
    }
    __syncthreads();
    constexpr int kPer = 8;                 // table entries per thread and pass
    for (int base = 0; base < npad * tc; base += kPer * 256) {
        float val[kPer];
#pragma unroll
        for (int u = 0; u < kPer; ++u) {
            const int i = base + u * 256 + threadIdx.x;
            const int j = i / tc, c = i - j * tc;
            val[u] = 0.f;
            if (i < npad * tc && j < n_valid) {
                const int x0 = c * kTile, x1 = min(x0 + kTile, width) - 1;
                val[u] = __ldg(exf + static_cast<size_t>(j) * width + clamp_round(s_pts[j].x, x0, x1));
            }
        }
#pragma unroll
        for (int u = 0; u < kPer; ++u) {
            const int i = base + u * 256 + threadIdx.x;
            if (i < npad * tc) mx[i] = val[u];
        }
    }
    for (int base = 0; base < npad * tr; base += kPer * 256) {
        float val[kPer];
#pragma unroll
        for (int u = 0; u < kPer; ++u) {
            const int i = base + u * 256 + threadIdx.x;
            const int j = i / tr, r = i - j * tr;
            val[u] = 0.f;
            if (i < npad * tr && j < n_valid) {
                const int y0 = r * kTile, y1 = min(y0 + kTile, height) - 1;
                val[u] = __ldg(eyf + static_cast<size_t>(clamp_round(s_pts[j].y, y0, y1)) * npad + j);
            }
        }
#pragma unroll
        for (int u = 0; u < kPer; ++u) {
            const int i = base + u * 256 + threadIdx.x;
            if (i < npad * tr) my[i] = val[u];
        }
    }
    if (norm == MF_NORM_MAX) {
        // lower bound: the map at the pixel nearest to each centre; one (centre p, term k) product per thread, summed
        // over k in any order (a bound, not the result: the tile holding that pixel is evaluated exactly below)
        for (int base = 0; base < n_valid * npad; base += 256) {
            const int i = base + threadIdx.x;
            float term = 0.f;
            if (i < n_valid * npad) {
                const int p = i / npad, k = i - p * npad;
                const int x = clamp_round(s_pts[p].x, 0, width - 1), y = clamp_round(s_pts[p].y, 0, height - 1);
                term = __ldg(exf + static_cast<size_t>(k) * width + x) * __ldg(eyf + static_cast<size_t>(y) * npad + k);
            }
            // npad is 8, 16, 24 or 32: groups of 8 lanes never straddle two centres
            term += __shfl_xor_sync(0xffffffffu, term, 1);
            term += __shfl_xor_sync(0xffffffffu, term, 2);
            term += __shfl_xor_sync(0xffffffffu, term, 4);
            if ((lane & 7) == 0 && i < n_valid * npad) atomicAdd(&centre[i / npad], term);
        }
    }
    __syncthreads();
    if (part == 0) {
        // which points matter in which 32-pixel column / row strip: render_kernel skips the others (and writes exact
        // zeros where none matters).  A factor below kCullBelow adds less than that fraction of the map's peak.
        for (int i = threadIdx.x; i < tc + tr; i += blockDim.x) {
            const bool col = i < tc;
            const int t = col ? i : i - tc;
            uint32_t m = 0u;
            for (int j = 0; j < n_valid; ++j)
                if ((col ? mx[j * tc + t] : my[j * tr + t]) >= kCullBelow) m |= 1u << j;
            (col ? colmask + static_cast<size_t>(f) * tc : rowmask + static_cast<size_t>(f) * tr)[t] = m;
        }
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
    // ---- MF_NORM_MAX: exact branch and bound ----
    if (threadIdx.x < n_valid) atomicMax(&s_best, __float_as_uint(fmaxf(centre[threadIdx.x], 0.f) * 0.9999f));
    __syncthreads();
    const float best = __uint_as_float(s_best);
    float exact = 0.f;
    // tile t belongs to warp (t mod 8*kNormBlocks) of the frame: neighbouring (surviving) tiles go to different warps
    const int kWarpsPerFrame = 8 * static_cast<int>(gridDim.x);
    const int gw = part * 8 + warp;
    const int n_tiles = tc * tr;
    for (int i = lane; i * kWarpsPerFrame + gw < n_tiles; i += 32) {
        const int tile = i * kWarpsPerFrame + gw;
        const int c = tile % tc, r = tile / tc;
        float ub = 0.f;
        for (int k = 0; k < npad; ++k) ub = fmaf(mx[k * tc + c], my[k * tr + r], ub);
        if (ub * 1.00001f >= best) {
            const int slot = atomicAdd(&s_count, 1);
            if (slot < kMaxSurvivors) s_list[slot] = tile;
        }
    }
    __syncthreads();
    const int n_surv = s_count;
    if (n_surv > kMaxSurvivors) {
        // more survivors than the list holds (huge sigma): fall back to this CTA's whole share of the tiles, i.e. the
        // SAME partition as the scan above (tile = i * kWarpsPerFrame + gw), so that a CTA that overflowed and one that
        // did not still cover every surviving tile between them
        for (int i = 0; i * kWarpsPerFrame + gw < n_tiles; ++i)
            exact = fmaxf(exact, warp_max(eval_tile(exf, eyf, tile_buf + warp * (kTile * npad), npad, width, height,
                                                    i * kWarpsPerFrame + gw, tc, lane)));
    } else {
        for (int i = warp; i < n_surv; i += 8)
            exact = fmaxf(exact, warp_max(eval_tile(exf, eyf, tile_buf + warp * (kTile * npad), npad, width, height,
                                                    s_list[i], tc, lane)));
    }
    // only exactly evaluated pixels may set Z (the bound above is 0.9999 x an approximately summed value); the tile
    // holding the true maximum always survives: its bound is >= the map's value there >= every centre value >= best
    if (lane == 0) atomicMax(&s_exact, __float_as_uint(exact));
    __syncthreads();
    if (threadIdx.x == 0 && s_exact != 0u) atomicMax(&meta[f].zmax_bits, s_exact);      // order-independent: deterministic
}

// ------------------------------------------------------------------------------------------------
// 4. render: the streaming pass.  One thread owns 4 adjacent columns (one 128-bit access per image
//    row) over kRowsPerThread rows; the 4*NP column factors stay in registers, the NP row factors
//    of each row are a broadcast 128-bit read of EyT (L1-resident).  Algorithmic HBM traffic is
//    12 B/pixel with depth and guided depth, 4 B/pixel map-only.
// ------------------------------------------------------------------------------------------------
#ifndef MF_RENDER_ROWS
#define MF_RENDER_ROWS 32
#endif
#ifndef MF_RENDER_THREADS
#define MF_RENDER_THREADS 128          // (256 until the end of round 2.  Alone at full clock 128 is worth +5 % at 960x544, +1 % at 1080p, -0.5 % at 4K;
#endif                                 //  behind the attention stack, at its power-capped 1.48 GHz: +16 % at 1080p, +11 % at 4K: smaller CTAs, finer tail)
#ifndef MF_RENDER_U
#define MF_RENDER_U 4
#endif
#ifndef MF_RENDER_MINB
#define MF_RENDER_MINB 1
#endif
constexpr int kRowsPerThread = MF_RENDER_ROWS;
constexpr int kStageRows = 2 * MF_RENDER_ROWS;   // row factors staged per warp in render_kernel
constexpr int kRenderThreads = MF_RENDER_THREADS;

__device__ __forceinline__ float4 ld_stream(const float4* p) {
    float4 r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::128B.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ void st_stream(float4* p, float4 v) {
    asm volatile("st.global.cs.v4.f32 [%0], {%1,%2,%3,%4};" :: "l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

// rows [ya, yb) of this thread's 4 columns where the map is identically zero: M = 0 and G = 0 (reading G1: the guided depth
// is 0 wherever the map is 0, whatever the depth holds there, so the depth is not read)
template <bool HAS_DEPTH, bool HAS_G, bool LOWRES>
__device__ __forceinline__ void stream_zero_rows(const float* __restrict__ depth, float* __restrict__ focus_map,
                                                 float* __restrict__ guided, size_t img, int width, int ya, int yb) {
    constexpr int U = 8;
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int y = ya; y < yb; y += U) {
#pragma unroll
        for (int r = 0; r < U; ++r) {
            if (y + r < yb) {
                const size_t o = img + static_cast<size_t>(y + r) * width;
                st_stream(reinterpret_cast<float4*>(focus_map + o), zero);
                if (HAS_G) st_stream(reinterpret_cast<float4*>(guided + o), zero);
            }
        }
    }
}

// Bilinear taps of reading F1 (half-pixel centres, edge clamp) for output index o of n_out from n_in samples, in exact
// integer arithmetic: src = max(0, ((2o+1) n_in - n_out) / (2 n_out)).
// Sizes are < 2^15 (checked by the caller), so the numerator fits 32 bits; inv_den = 1 / (2 n_out).
__device__ __forceinline__ void bilinear_taps(int o, int n_out, int n_in, float inv_den, int& i0, int& i1, float& lam) {
    const int num = (2 * o + 1) * n_in - n_out;
    if (num <= 0) {
        i0 = 0;
        lam = 0.f;
    } else {
        i0 = min(num / (2 * n_out), n_in - 1);
        lam = static_cast<float>(num - i0 * 2 * n_out) * inv_den;
    }
    i1 = min(i0 + 1, n_in - 1);
}

template <int NP, bool HAS_DEPTH, bool HAS_G, bool LOWRES>
__global__ void __launch_bounds__(kRenderThreads, LOWRES ? 2 : MF_RENDER_MINB)
render_kernel(const float* __restrict__ ex, const float* __restrict__ eyt, const FrameMeta* __restrict__ meta,
              const uint32_t* __restrict__ colmask, const uint32_t* __restrict__ rowmask,
              const float* __restrict__ depth, float* __restrict__ focus_map, float* __restrict__ guided,
              int width, int height, int blocks_per_frame, int norm, int dw, int dh) {
    pdl_wait();                             // norm_kernel's (and, through it, tables_kernel's) output
    const int f = blockIdx.x / blocks_per_frame;
    const int b = blockIdx.x - f * blocks_per_frame;
    const int wq = width >> 2;
    const int idx = b * kRenderThreads + threadIdx.x;
    const int rb = idx / wq;
    const int x = (idx - rb * wq) << 2;
    const int y0 = rb * kRowsPerThread;
    if (__all_sync(0xffffffffu, y0 >= height)) return;          // whole warp past the image
    const int y1 = max(y0, min(y0 + kRowsPerThread, height));    // == y0 for a lane past the image: no rows
    const FrameMeta fm = meta[f];
    float scale = fm.inv_z;
    if (norm == MF_NORM_MAX) {
        const float z = __uint_as_float(fm.zmax_bits);
        scale = z > 0.f ? 1.0f / z : 0.f;
    }
    const size_t img = static_cast<size_t>(f) * height * width + x;

    // Which points matter for this warp's columns and this thread's 32-row strip (norm_kernel's strip masks): a point
    // whose factor is below kCullBelow over the whole strip adds < 1e-13 of the map's peak (S8(c)-D3 allows 1e-12).
    // Where no point matters the pixels are exact zeros, written by a pure streaming loop.  All tests are warp-uniform
    // except the row strip, which differs only between lanes of a warp that straddles two strips.
    static_assert(kRowsPerThread == kTile, "render_kernel's row strips are norm_kernel's tiles");
    const int tc = (width + kTile - 1) / kTile, tr = (height + kTile - 1) / kTile;
    uint32_t pts_live = 0u;
    if (scale != 0.f && y1 > y0)
        pts_live = (__ldg(colmask + static_cast<size_t>(f) * tc + (x >> 5)) | __ldg(colmask + static_cast<size_t>(f) * tc + ((x + 3) >> 5))) &
                   __ldg(rowmask + static_cast<size_t>(f) * tr + rb);
    pts_live = __reduce_or_sync(0xffffffffu, pts_live);
    const int ya = pts_live ? y0 : y1, yb = y1;                  // rows computed by this thread: [ya, yb)
    stream_zero_rows<HAS_DEPTH, HAS_G, LOWRES>(depth, focus_map, guided, img, width, y0, ya);
    if (pts_live) {
        float4 e[NP];
        const float* exf = ex + static_cast<size_t>(f) * NP * width + x;
        unsigned live = 0u;                 // groups of 4 points
#pragma unroll
        for (int q = 0; q < NP / 4; ++q)
            if (pts_live & (0xFu << (4 * q))) live |= 1u << q;
#pragma unroll
        for (int j = 0; j < NP; ++j)
            e[j] = (live & (1u << (j / 4))) ? __ldg(reinterpret_cast<const float4*>(exf + static_cast<size_t>(j) * width))
                                            : make_float4(0.f, 0.f, 0.f, 0.f);
        const float4* eyrow = reinterpret_cast<const float4*>(eyt + static_cast<size_t>(f) * height * NP);
        // The row factors of the warp's rows (one 32-row strip, two when the warp straddles strips) are staged in
        // shared memory with one batch of coalesced loads, so the row loop below never waits on L2 for them.
        extern __shared__ float s_rows[];                       // [warps][kStageRows][NP]
        float* wbuf = s_rows + (threadIdx.x >> 5) * (kStageRows * NP);
        const int ylo = __reduce_min_sync(0xffffffffu, ya < yb ? ya : INT_MAX);
        const int yhi = __reduce_max_sync(0xffffffffu, ya < yb ? yb : 0);
        const bool staged = yhi - ylo <= kStageRows;            // false only for images narrower than 128 pixels
        if (staged) {
            const int n4 = (yhi - ylo) * (NP / 4);
            for (int i = threadIdx.x & 31; i < n4; i += 32)
                reinterpret_cast<float4*>(wbuf)[i] = __ldg(eyrow + static_cast<size_t>(ylo) * (NP / 4) + i);
            __syncwarp();
        }
        constexpr int U = MF_RENDER_U;
        // LOWRES: depth is [count, dh, dw] at the model's resolution and is interpolated here (reading F1); the four
        // columns' taps are fixed for the thread, the row taps change per row.  One low-res row is interpolated
        // horizontally to the thread's four columns once (hrow): successive output rows reuse the same two low-res rows
        // (top, bot) until the row taps move on, so a thread loads each low-res row once per strip.
        int tx0[4] = {0, 0, 0, 0}, tx1[4] = {0, 0, 0, 0};
        float tlx[4] = {0.f, 0.f, 0.f, 0.f};
        const float* dlo = depth;
        if (LOWRES) {
#pragma unroll
            for (int c = 0; c < 4; ++c)
                bilinear_taps(x + c, width, dw, 1.0f / static_cast<float>(2 * width), tx0[c], tx1[c], tlx[c]);
            dlo = depth + static_cast<size_t>(f) * dh * dw;
        }
        const float inv_2h = 1.0f / static_cast<float>(2 * height);
        auto hrow = [&](int row) {
            const float* p = dlo + static_cast<size_t>(row) * dw;
            float v[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const float a = __ldg(p + tx0[c]);
                v[c] = fmaf(tlx[c], __ldg(p + tx1[c]) - a, a);
            }
            return make_float4(v[0], v[1], v[2], v[3]);
        };
        int it = -1, ib = -1, in = -1;                           // low-res rows held in top, bot, nxt
        float4 top = make_float4(0.f, 0.f, 0.f, 0.f), bot = top, nxt = top;
        for (int y = ya; y < yb; y += U) {
            float4 d[U];
            if (HAS_DEPTH && !LOWRES) {
#pragma unroll
                for (int r = 0; r < U; ++r)
                    if (y + r < yb) d[r] = ld_stream(reinterpret_cast<const float4*>(depth + img + static_cast<size_t>(y + r) * width));
            }
#pragma unroll
            for (int r = 0; r < U; ++r) {
                if (y + r < yb) {
                    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                    for (int q = 0; q < NP / 4; ++q) {
                        if (!(live & (1u << q))) continue;
                        const float4 w = staged ? reinterpret_cast<const float4*>(wbuf)[(y + r - ylo) * (NP / 4) + q]
                                                : __ldg(eyrow + static_cast<size_t>(y + r) * (NP / 4) + q);
                        const float wy[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            acc.x = fmaf(e[4 * q + k].x, wy[k], acc.x);
                            acc.y = fmaf(e[4 * q + k].y, wy[k], acc.y);
                            acc.z = fmaf(e[4 * q + k].z, wy[k], acc.z);
                            acc.w = fmaf(e[4 * q + k].w, wy[k], acc.w);
                        }
                    }
                    if (LOWRES) {
                        int ty0, ty1;
                        float ly;
                        bilinear_taps(y + r, height, dh, inv_2h, ty0, ty1, ly);
                        if (ty0 != it || ty1 != ib) {
                            if (ty0 == ib && ty1 == in) {       // the usual step when upsampling: slide down one low-res row
                                top = bot;
                                bot = nxt;
                            } else {
                                top = hrow(ty0);
                                bot = hrow(ty1);
                            }
                            it = ty0;
                            ib = ty1;
                            in = min(ib + 1, dh - 1);
                            nxt = hrow(in);
                        }
                        d[r] = make_float4(fmaf(ly, bot.x - top.x, top.x), fmaf(ly, bot.y - top.y, top.y),
                                           fmaf(ly, bot.z - top.z, top.z), fmaf(ly, bot.w - top.w, top.w));
                    }
                    const float4 m = make_float4(acc.x * scale, acc.y * scale, acc.z * scale, acc.w * scale);
                    const size_t o = img + static_cast<size_t>(y + r) * width;
                    st_stream(reinterpret_cast<float4*>(focus_map + o), m);
                    if (HAS_G)
                        st_stream(reinterpret_cast<float4*>(guided + o),
                                  make_float4(m.x != 0.f ? m.x * d[r].x : 0.f, m.y != 0.f ? m.y * d[r].y : 0.f,
                                              m.z != 0.f ? m.z * d[r].z : 0.f, m.w != 0.f ? m.w * d[r].w : 0.f));     // reading G1
                }
            }
        }
    }
}

template <int NP>
static void launch_render(const Workspace& ws, const float* depth, float* focus_map, float* guided, int count,
                          int width, int height, int norm, int dw, int dh, cudaStream_t stream) {
    const int row_blocks = (height + kRowsPerThread - 1) / kRowsPerThread;
    const long long threads = static_cast<long long>(width / 4) * row_blocks;
    const int bpf = static_cast<int>((threads + kRenderThreads - 1) / kRenderThreads);
    const unsigned grid = static_cast<unsigned>(bpf) * static_cast<unsigned>(count);
    const size_t smem = sizeof(float) * (kRenderThreads / 32) * kStageRows * NP;
    if (smem > 48 * 1024) {
        cudaFuncSetAttribute(render_kernel<NP, true, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
        cudaFuncSetAttribute(render_kernel<NP, true, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
        cudaFuncSetAttribute(render_kernel<NP, false, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
    }
    if (guided && dw > 0)
        launch_pdl(render_kernel<NP, true, true, true>, dim3(grid), dim3(kRenderThreads), smem, stream, ws.ex, ws.eyt, ws.meta,
                   ws.colmask, ws.rowmask, depth, focus_map, guided, width, height, bpf, norm, dw, dh);
    else if (guided)
        launch_pdl(render_kernel<NP, true, true, false>, dim3(grid), dim3(kRenderThreads), smem, stream, ws.ex, ws.eyt, ws.meta,
                   ws.colmask, ws.rowmask, depth, focus_map, guided, width, height, bpf, norm, 0, 0);
    else
        launch_pdl(render_kernel<NP, false, false, false>, dim3(grid), dim3(kRenderThreads), smem, stream, ws.ex, ws.eyt,
                   ws.meta, ws.colmask, ws.rowmask, depth, focus_map, guided, width, height, bpf, norm, 0, 0);
}

}  // namespace mf

extern "C" size_t mf_motion_focus_workspace_size(int count, int width, int height, int n_points) {
    if (count < 1 || width < 1 || height < 1 || n_points < 1 || n_points > mf::kMaxPoints) return 0;
    return mf::carve(nullptr, count, width, height, n_points, nullptr);
}

// depth_width == 0: depth is [count, height, width]; otherwise [count, depth_height, depth_width], interpolated (reading F1)
static mf_status motion_focus_impl(const double* global_w2c, mf_intrinsics K, int num_frames, int render_begin, int render_end,
                                   int width, int height, const float* depth, int depth_width, int depth_height,
                                   const mf_focus_params* params, float* focus_map, float* guided_depth, float* focus_uv,
                                   int32_t* focus_index, void* workspace, size_t workspace_bytes, void* stream) {
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
    pp.width = width; pp.height = height;

    const int tc = (width + kTile - 1) / kTile, tr = (height + kTile - 1) / kTile;
    const size_t smem = sizeof(float) * (npad * static_cast<size_t>(tc + tr) + kMaxPoints + 8 * kTile * npad);
    // CTAs per frame in norm_kernel: kNormBlocks when the call is short, fewer when it holds so many frames that the call's CTAs
    // would need several waves of these latency-bound CTAs: two of them (256 threads, 118 registers) are resident per SM.
    // (Measured, 20 back-to-back calls: 1 / 2 / 3 / 4 / 8 / 16 CTAs per SM as the budget give 5451 / 5392 / 5384 / 5335 / 5180 /
    // 5008 GB/s for 240 frames of 960x544 and 8626 / 8709 / 8663 / 8687 / 8685 / 8689 for 64 frames of 4K.)
    const int norm_blocks = std::max(1, std::min(kNormBlocks, (2 * sm_count() + count - 1) / count));
    if (focus_map && smem > 200 * 1024) return fail(MF_ERR_UNSUPPORTED, "mf_motion_focus: image too large for the bound tables");
    if (validate_only()) return MF_OK;
    if (focus_map) {
        if (smem > 48 * 1024)
            MF_CUDA_OK(cudaFuncSetAttribute(norm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem)));
    }
    const size_t img = static_cast<size_t>(width) * height;

    // points + tables + normaliser of frames [f0, f0+n) (small, latency-bound launches)
    auto prepare = [&](int f0, int n, cudaStream_t q) -> cudaError_t {
        PointParams g = pp;
        g.render_begin = render_begin + f0;
        g.count = n;
        float* uv = focus_uv ? focus_uv + 2 * static_cast<size_t>(f0) : nullptr;
        int32_t* fi = focus_index ? focus_index + f0 : nullptr;
        if (!focus_map) {
            points_kernel<<<(n + 3) / 4, 128, 0, q>>>(global_w2c, g, ws.pts + static_cast<size_t>(f0) * kMaxPoints,
                                                     ws.meta + f0, uv, fi);
            return cudaGetLastError();
        }
        float* ex = ws.ex + static_cast<size_t>(f0) * npad * width;
        float* eyt = ws.eyt + static_cast<size_t>(f0) * height * npad;
        const int chunks = (npad * (width + height) + kTableItems * 256 - 1) / (kTableItems * 256);
        tables_kernel<<<dim3(chunks, n), 256, 0, q>>>(global_w2c, g, ws.pts + static_cast<size_t>(f0) * kMaxPoints, ws.meta + f0,
                                                      uv, fi, ex, eyt, npad, width, height);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        return launch_pdl(norm_kernel, dim3(norm_blocks, n), dim3(256), smem, q, ws.pts + static_cast<size_t>(f0) * kMaxPoints,
                          ws.meta + f0, ex, eyt, ws.colmask + static_cast<size_t>(f0) * tc, ws.rowmask + static_cast<size_t>(f0) * tr,
                          npad, width, height, static_cast<int>(params->norm));
    };
    // the HBM-bound pass over frames [f0, f0+n)
    auto render = [&](int f0, int n, cudaStream_t q) -> cudaError_t {
        Workspace w = ws;
        w.meta = ws.meta + f0;
        w.ex = ws.ex + static_cast<size_t>(f0) * npad * width;
        w.eyt = ws.eyt + static_cast<size_t>(f0) * height * npad;
        w.colmask = ws.colmask + static_cast<size_t>(f0) * tc;
        w.rowmask = ws.rowmask + static_cast<size_t>(f0) * tr;
        const float* d = depth ? depth + f0 * (depth_width > 0 ? static_cast<size_t>(depth_width) * depth_height : img) : nullptr;
        float* m = focus_map + f0 * img;
        float* gd = guided_depth ? guided_depth + f0 * img : nullptr;
        switch (npad) {
            case 8: launch_render<8>(w, d, m, gd, n, width, height, params->norm, depth_width, depth_height, q); break;
            case 16: launch_render<16>(w, d, m, gd, n, width, height, params->norm, depth_width, depth_height, q); break;
            case 24: launch_render<24>(w, d, m, gd, n, width, height, params->norm, depth_width, depth_height, q); break;
            default: launch_render<32>(w, d, m, gd, n, width, height, params->norm, depth_width, depth_height, q); break;
        }
        return cudaGetLastError();
    };

    MF_CUDA_OK(prepare(0, count, s));
    if (focus_map) MF_CUDA_OK(render(0, count, s));
    return MF_OK;
}

extern "C" mf_status mf_motion_focus(const double* global_w2c, mf_intrinsics K, int num_frames, int render_begin,
                                     int render_end, int width, int height, const float* depth,
                                     const mf_focus_params* params, float* focus_map, float* guided_depth,
                                     float* focus_uv, int32_t* focus_index, void* workspace, size_t workspace_bytes,
                                     void* stream) {
    return motion_focus_impl(global_w2c, K, num_frames, render_begin, render_end, width, height, depth, 0, 0, params, focus_map,
                             guided_depth, focus_uv, focus_index, workspace, workspace_bytes, stream);
}

extern "C" mf_status mf_motion_focus_upsampled(const double* global_w2c, mf_intrinsics K, int num_frames, int render_begin,
                                               int render_end, int width, int height, const float* depth_lowres,
                                               int depth_width, int depth_height, const mf_focus_params* params,
                                               float* focus_map, float* guided_depth, float* focus_uv, int32_t* focus_index,
                                               void* workspace, size_t workspace_bytes, void* stream) {
    if (!depth_lowres || !guided_depth || !focus_map)
        return mf::fail(MF_ERR_INVALID_ARG, "mf_motion_focus_upsampled: depth_lowres, focus_map and guided_depth are required");
    if (depth_width < 1 || depth_height < 1)
        return mf::fail(MF_ERR_INVALID_ARG, "mf_motion_focus_upsampled: bad depth size %dx%d", depth_width, depth_height);
    if (width > 32767 || height > 32767 || depth_width > 32767 || depth_height > 32767)     // bilinear_taps works in int32
        return mf::fail(MF_ERR_UNSUPPORTED, "mf_motion_focus_upsampled: sizes above 32767 are not supported");
    return motion_focus_impl(global_w2c, K, num_frames, render_begin, render_end, width, height, depth_lowres, depth_width,
                             depth_height, params, focus_map, guided_depth, focus_uv, focus_index, workspace, workspace_bytes, stream);
}
