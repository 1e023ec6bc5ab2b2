// rasterize_feat.cu -- xpr_rasterize_featn_fwd / _bwd and xpr_depth_bwd (xpr_rasterize_feat_fwd / _bwd are the FEAT
// instantiations of rasterize_fwd_kernel / rasterize_bwd_kernel in rasterize.cu): compositing with the
// rendered features of SURVEY 8(f) f3 ("rendered features such as depth", Table 2; DESIGN.md
// reading C31): next to the colour, the same walk blends the depth image D = sum_k z_k alpha_k T_k and the
// accumulated opacity A = sum_k alpha_k T_k (no background term), and the reverse pass takes dL/dD and dL/dA.
//
// Same layout as rasterize.cu: one CTA per 16x16 tile, the tile's list staged through shared memory in
// batches, decisions taken on `power` in the fixed fp32 order of rule R3.  The record carries z in the slot
// rasterize.cu leaves unused, so the feature costs no extra shared-memory read.
#include "common.cuh"

namespace xpr {
namespace {

constexpr int BLOCK = TILE * TILE;

struct FeatParams {
    int W, H, TW;
    float amax, tmin;
    float bg[3];
    const uint32_t* order;
};

#ifndef XPR_FEAT_PPT_MIN_TILES
#define XPR_FEAT_PPT_MIN_TILES 4096      // same switch as rasterize.cu: throughput shape for large images
#endif

__device__ __forceinline__ float opac_exp(float power, float l2o) {   // o exp(power) = ex2(power log2 e + log2 o)
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(fmaf(power, 1.4426950408889634f, l2o)));
    return y;
}

__device__ __forceinline__ float fast_rcp(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Transposed butterfly over 8 per-lane values (9 shuffles); lane L with (L & 3) == 0 ends with the total of value L >> 2.
__device__ __forceinline__ float warp_reduce8(const float (&v)[8], int lane) {
    float w[4], x[2];
    const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float send = b4 ? v[i] : v[i + 4], keep = b4 ? v[i + 4] : v[i];
        w[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const float send = b3 ? w[i] : w[i + 2], keep = b3 ? w[i + 2] : w[i];
        x[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    }
    const float send = b2 ? x[0] : x[1], keep = b2 ? x[1] : x[0];
    float y = keep + __shfl_xor_sync(0xffffffffu, send, 4);
    y += __shfl_xor_sync(0xffffffffu, y, 2);
    y += __shfl_xor_sync(0xffffffffu, y, 1);
    return y;
}

// ---- N-channel features (xpr_rasterize_featn_fwd / _bwd, reading C31) --------------------------------
// F[p, c] = sum_k feat[g_k, c] alpha_k T_k over the colour pass's contributing sequence: the walk is REPLAYED from the
// colour pass's n_contrib (an entry contributes iff pos < n_contrib and it passes the two gates on `power`, the same
// bit-identical decisions; the exit test is implied by n_contrib).  Channels are processed in chunks of CH = 8:
// grid = (tiles, chunks), one launch for any C.  Two pixels per thread, forward and backward.
constexpr int FEATN_CH = 8;

template <int CH, int PPT>
__global__ void __launch_bounds__(BLOCK / PPT)
rasterize_featn_fwd_kernel(FeatParams P, const float2* __restrict__ mean2d, const float4* __restrict__ conic_opac,
                           const float* __restrict__ lnv, const float* __restrict__ feat, int C,
                           const uint32_t* __restrict__ vals, const uint2* __restrict__ ranges,
                           const uint32_t* __restrict__ n_contrib, float* __restrict__ feat_img) {
    // PPT = 2: a thread owns the pixels (x, y) and (x + 8, y), as rasterize_fwd_kernel: the record, the channel values
    // and the row terms of `power` are read / formed once per two pixels
    constexpr int THREADS = BLOCK / PPT, ROW = TILE / PPT;
    __shared__ float4 s_rec[2 * THREADS];          // (mx, my, qa, qb | qc, thr, log2 o, -)
    __shared__ float s_f[CH * THREADS];            // CH channels per entry
    __shared__ uint32_t s_max[THREADS / 32];
    const int tile = P.order ? (int)P.order[blockIdx.x] : (int)blockIdx.x;
    const int tx = tile % P.TW, ty = tile / P.TW;
    const int c0 = blockIdx.y * CH;
    const int py = ty * TILE + (threadIdx.x / ROW);
    const float pyc = (float)py + 0.5f;
    const uint2 rg = ranges[tile];
    int64_t pid[PPT];
    bool in[PPT];
    uint32_t n[PPT], wmax = 0;
    float pxc[PPT], T[PPT], F[PPT][CH];
#pragma unroll
    for (int k = 0; k < PPT; ++k) {
        const int px = tx * TILE + (threadIdx.x % ROW) + 8 * k;
        in[k] = (px < P.W) && (py < P.H);
        pid[k] = (int64_t)py * P.W + px;
        pxc[k] = (float)px + 0.5f;
        n[k] = in[k] ? n_contrib[pid[k]] : 0u;
        wmax = max(wmax, n[k]);
        T[k] = 1.0f;
#pragma unroll
        for (int c = 0; c < CH; ++c) F[k][c] = 0.0f;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) wmax = max(wmax, __shfl_xor_sync(0xffffffffu, wmax, o));
    if ((threadIdx.x & 31) == 0) s_max[threadIdx.x >> 5] = wmax;
    __syncthreads();
    uint32_t max_n = 0;
#pragma unroll
    for (int w = 0; w < THREADS / 32; ++w) max_n = max(max_n, s_max[w]);

    for (uint32_t base = 0; base < max_n; base += THREADS) {
        const uint32_t cnt = min((uint32_t)THREADS, max_n - base);
        __syncthreads();
        if (threadIdx.x < cnt) {
            const uint32_t g = vals[rg.x + base + threadIdx.x];
            const float2 m = mean2d[g];
            const float4 co = conic_opac[g];
            s_rec[2 * threadIdx.x] = make_float4(m.x, m.y, -0.5f * co.x, -co.y);
            s_rec[2 * threadIdx.x + 1] = make_float4(-0.5f * co.z, -lnv[g], __log2f(co.w), 0.0f);
#pragma unroll
            for (int c = 0; c < CH; ++c) s_f[CH * threadIdx.x + c] = (c0 + c < C) ? feat[(size_t)g * C + c0 + c] : 0.0f;
        }
        __syncthreads();
        if (base >= wmax) continue;                 // warp-uniform
        const uint32_t lim = min(cnt, wmax - base);
        for (uint32_t j = 0; j < lim; ++j) {
            const float4 ge = s_rec[2 * j], ga = s_rec[2 * j + 1];
            const float dy = pyc - ge.y;
            const float t1 = __fmul_rn(ge.w, dy), t2 = __fmul_rn(__fmul_rn(ga.x, dy), dy);
            float w[PPT];
            bool any = false;
#pragma unroll
            for (int k = 0; k < PPT; ++k) {
                const float dx = pxc[k] - ge.x;
                const float power = __fmaf_rn(__fmaf_rn(ge.z, dx, t1), dx, t2);      // rule R3
                const bool c = (base + j < n[k]) && !(power > 0.0f) && !(power < ga.y);
                const float alpha = c ? fminf(P.amax, opac_exp(power, ga.z)) : 0.0f;
                w[k] = alpha * T[k];
                T[k] = T[k] * (1.0f - alpha);
                any |= c;
            }
            if (!any) continue;
            const float4* f4 = reinterpret_cast<const float4*>(s_f + CH * j);
#pragma unroll
            for (int q = 0; q < CH / 4; ++q) {
                const float4 f = f4[q];
#pragma unroll
                for (int k = 0; k < PPT; ++k) {
                    F[k][4 * q] = fmaf(f.x, w[k], F[k][4 * q]); F[k][4 * q + 1] = fmaf(f.y, w[k], F[k][4 * q + 1]);
                    F[k][4 * q + 2] = fmaf(f.z, w[k], F[k][4 * q + 2]); F[k][4 * q + 3] = fmaf(f.w, w[k], F[k][4 * q + 3]);
                }
            }
        }
    }
#pragma unroll
    for (int k = 0; k < PPT; ++k) {
        if (!in[k]) continue;
#pragma unroll
        for (int c = 0; c < CH; ++c)
            if (c0 + c < C) feat_img[pid[k] * C + c0 + c] = F[k][c];
    }
}

// Backward for gF = dL/dF alone (the colour / D / A parts come from their own kernels and add: every step is linear
// in the incoming gradient).  With gc_k = sum_c gF_c feat[g_k, c] (a scalar per pixel-pair):
//   dL/dfeat[g_k, c] += alpha_k T_k gF_c,     dL/dalpha_k = T_k gc_k - Q_k / (1 - alpha_k),
//   Q_k = sum_c gF_c SF_kc = sum_{j>k} gc_j alpha_j T_j    -- ONE running scalar instead of CH running sums,
// and from dL/dalpha on as rasterize_bwd_kernel.  6 + CH values per (warp, Gaussian) go through two transposed
// butterflies; the geometric gradients are ADDED to g_mean2d / g_conic / g_opac by every channel chunk.
template <int CH, int PPT>
__global__ void __launch_bounds__(BLOCK / PPT)
rasterize_featn_bwd_kernel(FeatParams P, const float2* __restrict__ mean2d, const float4* __restrict__ conic_opac,
                           const float* __restrict__ lnv, const float* __restrict__ feat, int C,
                           const uint32_t* __restrict__ vals, const uint2* __restrict__ ranges,
                           const float* __restrict__ final_T, const uint32_t* __restrict__ n_contrib,
                           const float* __restrict__ dL_dF, float* __restrict__ g_mean2d,
                           float* __restrict__ g_conic, float* __restrict__ g_opac, float* __restrict__ g_feat) {
    static_assert(CH == 8, "two butterflies of 8: 6 geometric + 2 channels, then 6 channels");
    constexpr int THREADS = BLOCK / PPT, BATCH = THREADS, TPR = TILE / PPT;
    __shared__ float4 s_geo[BATCH];    // mx, my, A, B
    __shared__ float4 s_gate[BATCH];   // C, thr, o, index (bits)
    __shared__ float s_l2o[BATCH];
    __shared__ float s_f[CH * BATCH];
    __shared__ uint32_t s_max[THREADS / 32];
    const int tile = P.order ? (int)P.order[blockIdx.x] : (int)blockIdx.x;
    const int tx = tile % P.TW, ty = tile / P.TW;
    const int c0 = blockIdx.y * CH;
    const int lane = threadIdx.x & 31;
    const int px0 = tx * TILE + (threadIdx.x % TPR) * PPT;
    const int py = ty * TILE + (threadIdx.x / TPR);
    const float pyc = (float)py + 0.5f;
    const uint2 rg = ranges[tile];

    uint32_t n[PPT];
    float T[PPT], Q[PPT], gF[PPT][CH], pxc[PPT];
    uint32_t wmax = 0;
#pragma unroll
    for (int k = 0; k < PPT; ++k) {
        const int px = px0 + k;
        pxc[k] = (float)px + 0.5f;
        n[k] = 0; T[k] = 0.0f; Q[k] = 0.0f;
#pragma unroll
        for (int c = 0; c < CH; ++c) gF[k][c] = 0.0f;
        if (px < P.W && py < P.H) {
            const int64_t pid = (int64_t)py * P.W + px;
            n[k] = n_contrib[pid];
            T[k] = final_T[pid];
#pragma unroll
            for (int c = 0; c < CH; ++c)
                if (c0 + c < C) gF[k][c] = dL_dF[pid * C + c0 + c];
        }
        wmax = max(wmax, n[k]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) wmax = max(wmax, __shfl_xor_sync(0xffffffffu, wmax, o));
    if (lane == 0) s_max[threadIdx.x >> 5] = wmax;
    __syncthreads();
    uint32_t max_n = 0;
#pragma unroll
    for (int w = 0; w < THREADS / 32; ++w) max_n = max(max_n, s_max[w]);

    // butterfly 1: mx my A B C o f0 f1; butterfly 2: f2 .. f7 (lanes 4 i own value i)
    const int vi = lane >> 2;
    const bool red_lane = (lane & 3) == 0;
    float* const base1 = (vi < 2) ? (g_mean2d + vi) : (vi < 5) ? (g_conic + (vi - 2)) : (vi == 5) ? g_opac
                                                                                      : (g_feat + c0 + (vi - 6));
    const uint32_t stride1 = (vi < 2) ? 2u : (vi < 5) ? 3u : (vi == 5) ? 1u : (uint32_t)C;
    const bool ok1 = red_lane && (vi < 6 || c0 + (vi - 6) < C);
    const bool ok2 = red_lane && vi < 6 && (c0 + 2 + vi < C);

    for (uint32_t hi = max_n; hi > 0;) {
        const uint32_t cnt = min((uint32_t)BATCH, hi);
        __syncthreads();
        if (threadIdx.x < cnt) {      // slot j holds list position hi-1-j (descending)
            const uint32_t g = vals[rg.x + hi - 1 - threadIdx.x];
            const float2 m = mean2d[g];
            const float4 co = conic_opac[g];
            s_geo[threadIdx.x] = make_float4(m.x, m.y, co.x, co.y);
            s_gate[threadIdx.x] = make_float4(co.z, -lnv[g], co.w, __uint_as_float(g));
            s_l2o[threadIdx.x] = __log2f(co.w);
#pragma unroll
            for (int c = 0; c < CH; ++c) s_f[CH * threadIdx.x + c] = (c0 + c < C) ? feat[(size_t)g * C + c0 + c] : 0.0f;
        }
        __syncthreads();
        for (uint32_t j = 0; j < cnt; ++j) {
            const uint32_t pos = hi - 1 - j;
            if (pos >= wmax) continue;     // warp-uniform
            const float4 ge = s_geo[j];
            const float4 ga = s_gate[j];
            const float Ac = ge.z, Bc = ge.w, Cc = ga.x;
            const float qa = -0.5f * Ac, qb = -Bc, qc = -0.5f * Cc;
            const float dy = pyc - ge.y;
            const float t1 = __fmul_rn(qb, dy), t2 = __fmul_rn(__fmul_rn(qc, dy), dy);
            float dx[PPT], power[PPT];
            bool contrib[PPT], any_c = false;
#pragma unroll
            for (int k = 0; k < PPT; ++k) {
                dx[k] = pxc[k] - ge.x;
                power[k] = __fmaf_rn(__fmaf_rn(qa, dx[k], t1), dx[k], t2);
                contrib[k] = (pos < n[k]) && !(power[k] > 0.0f) && !(power[k] < ga.y);
                any_c |= contrib[k];
            }
            if (!__any_sync(0xffffffffu, any_c)) continue;
            const float l2o = s_l2o[j];
            float f[CH];
            {
                const float4* f4 = reinterpret_cast<const float4*>(s_f + CH * j);
#pragma unroll
                for (int q = 0; q < CH / 4; ++q) {
                    const float4 t = f4[q];
                    f[4 * q] = t.x; f[4 * q + 1] = t.y; f[4 * q + 2] = t.z; f[4 * q + 3] = t.w;
                }
            }
            float gf[CH];
#pragma unroll
            for (int c = 0; c < CH; ++c) gf[c] = 0.0f;
            float sp = 0.f, spx = 0.f, spxx = 0.f;
#pragma unroll
            for (int k = 0; k < PPT; ++k) {            // branch-free: a pixel that does not contribute has alpha = 0
                const float og = contrib[k] ? opac_exp(power[k], l2o) : 0.0f;
                const float alpha = fminf(P.amax, og);
                const float inv = fast_rcp(1.0f - alpha);
                T[k] = T[k] * inv;
                const float w = alpha * T[k];
                float gc = 0.0f;
#pragma unroll
                for (int c = 0; c < CH; ++c) {
                    gf[c] = fmaf(w, gF[k][c], gf[c]);
                    gc = fmaf(gF[k][c], f[c], gc);
                }
                const float dalpha = fmaf(T[k], gc, -(inv * Q[k]));
                Q[k] = fmaf(gc, w, Q[k]);
                const float live = (og < P.amax) ? dalpha : 0.0f;   // C14
                const float dpow = og * live;
                const float dxp = dx[k] * dpow;
                sp += dpow; spx += dxp; spxx = fmaf(dx[k], dxp, spxx);
            }
            float v1[8], v2[8];
            {
                const float sy = dy * sp;
                v1[0] = fmaf(Ac, spx, Bc * sy); v1[1] = fmaf(Bc, spx, Cc * sy);
                v1[2] = -0.5f * spxx; v1[3] = -dy * spx; v1[4] = -0.5f * dy * sy;
                v1[5] = sp; v1[6] = gf[0]; v1[7] = gf[1];
#pragma unroll
                for (int c = 0; c < 6; ++c) v2[c] = gf[2 + c];
                v2[6] = v2[7] = 0.0f;
            }
            float tot1 = warp_reduce8(v1, lane);
            const float tot2 = warp_reduce8(v2, lane);
            const uint32_t g = __float_as_uint(ga.w);
            if (vi == 5) tot1 *= fast_rcp(ga.z);       // dL/do = (sum dpow) / o
            if (ok1) atomicAdd(base1 + (size_t)stride1 * g, tot1);
            if (ok2) atomicAdd(g_feat + (size_t)C * g + c0 + 2 + vi, tot2);
        }
        hi -= cnt;
    }
}

// z = (W mu + t)_z  =>  dL/dmu += W[2,:] dL/dz for a Gaussian that was not culled
__global__ void depth_bwd_kernel(int64_t N, float w0, float w1, float w2, const uint32_t* __restrict__ tile_count,
                                 const float* __restrict__ g_depth, float* __restrict__ g_means) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N || tile_count[i] == 0) return;
    const float gz = g_depth[i];
    g_means[3 * i] += w0 * gz; g_means[3 * i + 1] += w1 * gz; g_means[3 * i + 2] += w2 * gz;
}

void make_feat_params(const xpr_camera* cam, const xpr_config* cfg, FeatParams& P) {
    P.W = cam->width; P.H = cam->height; P.TW = tiles_x(cam);
    P.amax = cfg->alpha_max; P.tmin = cfg->t_min;
    for (int i = 0; i < 3; ++i) P.bg[i] = cfg->bg[i];
    P.order = cfg->tile_order;
}

}  // namespace
}  // namespace xpr

using namespace xpr;

extern "C" int32_t xpr_rasterize_featn_fwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* mean2d,
                                           const float* conic_opac, const float* lnv, const float* feat, int32_t C,
                                           const uint32_t* vals_sorted, const uint32_t* tile_ranges,
                                           const uint32_t* n_contrib, float* feat_img, void* stream) {
    if (int32_t s = check_cam_cfg(cam, cfg)) return s;
    if (N < 0 || C < 1 || C > 65535 * FEATN_CH) return XPR_ERR_INVALID_ARG;
    if (!aligned(tile_ranges, 8) || !aligned(n_contrib, 4) || !aligned(feat_img, 4)) return XPR_ERR_INVALID_ARG;
    if (N > 0 && (!aligned(mean2d, 8) || !aligned(conic_opac, 16) || !aligned(lnv, 4) || !aligned(feat, 4) ||
                  !aligned(vals_sorted, 4)))
        return XPR_ERR_INVALID_ARG;
    FeatParams P;
    make_feat_params(cam, cfg, P);
    const dim3 grid(tiles_x(cam) * tiles_y(cam), (C + FEATN_CH - 1) / FEATN_CH);
    rasterize_featn_fwd_kernel<FEATN_CH, 2><<<grid, BLOCK / 2, 0, (cudaStream_t)stream>>>(
        P, reinterpret_cast<const float2*>(mean2d), reinterpret_cast<const float4*>(conic_opac), lnv, feat, C,
        vals_sorted, reinterpret_cast<const uint2*>(tile_ranges), n_contrib, feat_img);
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}

extern "C" int32_t xpr_rasterize_featn_bwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* mean2d,
                                           const float* conic_opac, const float* lnv, const float* feat, int32_t C,
                                           const uint32_t* vals_sorted, const uint32_t* tile_ranges,
                                           const float* final_T, const uint32_t* n_contrib, const float* dL_dfeat,
                                           float* g_mean2d, float* g_conic, float* g_opac, float* g_feat,
                                           int32_t zero_init, void* stream) {
    if (int32_t s = check_cam_cfg(cam, cfg)) return s;
    if (N < 0 || C < 1 || C > 65535 * FEATN_CH) return XPR_ERR_INVALID_ARG;
    if (!aligned(tile_ranges, 8) || !aligned(final_T, 4) || !aligned(n_contrib, 4) || !aligned(dL_dfeat, 4))
        return XPR_ERR_INVALID_ARG;
    if (N == 0) return XPR_OK;
    if (!aligned(mean2d, 8) || !aligned(conic_opac, 16) || !aligned(lnv, 4) || !aligned(feat, 4) ||
        !aligned(vals_sorted, 4) || !aligned(g_mean2d, 4) || !aligned(g_conic, 4) || !aligned(g_opac, 4) ||
        !aligned(g_feat, 4))
        return XPR_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)N;
    if (zero_init & 1) {
        XPR_CUDA(cudaMemsetAsync(g_mean2d, 0, sizeof(float) * 2 * n, st));
        XPR_CUDA(cudaMemsetAsync(g_conic, 0, sizeof(float) * 3 * n, st));
        XPR_CUDA(cudaMemsetAsync(g_opac, 0, sizeof(float) * n, st));
    }
    if (zero_init & 2) XPR_CUDA(cudaMemsetAsync(g_feat, 0, sizeof(float) * n * (size_t)C, st));
    FeatParams P;
    make_feat_params(cam, cfg, P);
    const dim3 grid(tiles_x(cam) * tiles_y(cam), (C + FEATN_CH - 1) / FEATN_CH);
    rasterize_featn_bwd_kernel<FEATN_CH, 2><<<grid, BLOCK / 2, 0, st>>>(
        P, reinterpret_cast<const float2*>(mean2d), reinterpret_cast<const float4*>(conic_opac), lnv, feat, C,
        vals_sorted, reinterpret_cast<const uint2*>(tile_ranges), final_T, n_contrib, dL_dfeat, g_mean2d, g_conic,
        g_opac, g_feat);
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}

extern "C" int32_t xpr_depth_bwd(int64_t N, const xpr_camera* cam, const uint32_t* tile_count, const float* g_depth,
                                 float* g_means, void* stream) {
    if (!cam || N < 0) return XPR_ERR_INVALID_ARG;
    if (N == 0) return XPR_OK;
    if (!aligned(tile_count, 4) || !aligned(g_depth, 4) || !aligned(g_means, 4)) return XPR_ERR_INVALID_ARG;
    const int threads = 256;
    const int64_t blocks = (N + threads - 1) / threads;
    depth_bwd_kernel<<<(unsigned)blocks, threads, 0, (cudaStream_t)stream>>>(N, cam->w2c[8], cam->w2c[9], cam->w2c[10],
                                                                              tile_count, g_depth, g_means);
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}
