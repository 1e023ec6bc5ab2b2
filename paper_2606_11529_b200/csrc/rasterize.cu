// rasterize.cu -- xpr_rasterize_fwd / xpr_rasterize_bwd: per-tile front-to-back alpha compositing
// (Algorithm 1, Listing 1) and its reverse-mode pass.
//
// One CTA per 16x16 tile, one thread per pixel.  The tile's list vals_sorted[start..end) is
// staged through shared memory in batches; every thread walks the batch with warp-broadcast
// LDS.128 reads.  Decisions (the power > 0 guard and the alpha gate) are taken on `power`,
// computed in the fixed fp32 order of rule R3 with explicit _rn intrinsics, never on exp().
#include "common.cuh"

namespace xpr {
namespace {

constexpr int BLOCK = TILE * TILE;   // 256 threads = 256 pixels

struct RasterParams {
    int W, H, TW;
    float amax, tmin;
    float bg[3];
    const uint32_t* order;   // xpr_config.tile_order: CTA b works on tile order[b] (longest lists first), or NULL
};

// power = fma(fma(qa, dx, qb*dy), dx, (qc*dy)*dy) with qa = -A/2, qb = -B, qc = -C/2 (R3, C25)
__device__ __forceinline__ float eval_power(float qa, float qb, float qc, float dx, float dy) {
    return __fmaf_rn(__fmaf_rn(qa, dx, __fmul_rn(qb, dy)), dx, __fmul_rn(__fmul_rn(qc, dy), dy));
}

// o * exp(power) = ex2(power * log2 e + log2 o): one FFMA + one MUFU; l2o = log2 o is staged with the record
__device__ __forceinline__ float opac_exp(float power, float l2o) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(fmaf(power, 1.4426950408889634f, l2o)));
    return y;
}

__device__ __forceinline__ float fast_exp(float x) {   // ex2.approx(x * log2 e); x in [-lnv, 0]
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x * 1.4426950408889634f));
    return y;
}

// Forward compositing (a8).  One CTA per 16x16 tile, in two shapes:
//   PPT = 2: 128 threads, a thread owns the two pixels (x, y) and (x + 8, y) of one row, so the row terms
//            of `power` (dy, qb*dy, (qc*dy)*dy) and the shared-memory reads of a list entry are paid once
//            per two pixels -- fewer instructions per pixel-pair (throughput shape, large images);
//   PPT = 1: 256 threads, one pixel each -- twice the warps on a tile, i.e. half the critical path of a
//            heavy tile (latency shape, images with few tiles where the longest list bounds the kernel).
// The arithmetic per pixel is exactly eval_power's (rule R3) in both.
// STATS = true: the same walk, additionally counting pixel-pair events into stats[0..3] =
// {visited, passed both gates, blended, sum of n_contrib} (xpr_rasterize_stats; roofline accounting).
#ifndef XPR_FWD_PPT2_MIN_TILES
#define XPR_FWD_PPT2_MIN_TILES 4096
#endif
constexpr int FWD_PPT2_MIN_TILES = XPR_FWD_PPT2_MIN_TILES;

// FEAT = true (xpr_rasterize_feat_fwd, reading C31): the same walk also blends the depth image
// D = sum z alpha T and the accumulated opacity A = sum alpha T; z rides in the record's unused slot.
template <bool STATS, int PPT, bool BF, bool FEAT = false>
__global__ void __launch_bounds__(BLOCK / PPT)
rasterize_fwd_kernel(RasterParams P, const float2* __restrict__ mean2d, const float4* __restrict__ conic_opac,
                     const float* __restrict__ rgb, const float* __restrict__ lnv,
                     const uint32_t* __restrict__ vals, const uint2* __restrict__ ranges,
                     float* __restrict__ image, float* __restrict__ final_T, uint32_t* __restrict__ n_contrib,
                     unsigned long long* __restrict__ stats, const float* __restrict__ depth = nullptr,
                     float* __restrict__ depth_img = nullptr, float* __restrict__ alpha_img = nullptr) {
    // record of one list entry: 3 x float4 = (mx, my, qa, qb | qc, thr = -lnv, log2 o, z (FEAT) | r, g, b, -)
    constexpr int FWD_BATCH = BLOCK / PPT;          // one list entry staged per thread
    __shared__ float4 s_rec[3 * FWD_BATCH];
    const int tile = P.order ? (int)P.order[blockIdx.x] : (int)blockIdx.x;
    const int tx = tile % P.TW, ty = tile / P.TW;
    constexpr int FWD_THREADS = BLOCK / PPT, ROW = TILE / PPT;
    const int px0 = tx * TILE + (threadIdx.x % ROW), px1 = px0 + 8, py = ty * TILE + (threadIdx.x / ROW);
    const bool in0 = (px0 < P.W) && (py < P.H), in1 = (PPT == 2) && (px1 < P.W) && (py < P.H);
    const float pxc0 = (float)px0 + 0.5f, pxc1 = (float)px1 + 0.5f, pyc = (float)py + 0.5f;
    const uint2 rg = ranges[tile];
    const uint32_t len = rg.y - rg.x;

    float Ta = 1.0f, Ca0 = 0.0f, Ca1 = 0.0f, Ca2 = 0.0f;     // pixel (px0, py)
    float Tb = 1.0f, Cb0 = 0.0f, Cb1 = 0.0f, Cb2 = 0.0f;     // pixel (px1, py)
    float Da = 0.0f, Aa = 0.0f, Db = 0.0f, Ab = 0.0f;         // FEAT: depth image and accumulated opacity
    uint32_t last_a = 0, last_b = 0;
    bool act_a = in0, act_b = in1;                            // still compositing
    uint32_t n_visit = 0, n_pass = 0, n_blend = 0;

    // The list is walked in groups of 4 entries.  Phase 1 of a group computes the 4 (x PPT) values of
    // `power` -- independent of each other and of the transmittance, so their latencies overlap -- and
    // phase 2 runs the sequential part (gate, alpha, T' = T (1 - alpha), exit test, blend).
#define XPR_FWD_POWER(u, rp)                                                                          \
    {                                                                                                \
        const float4 ge = (rp)[0];                                                                   \
        const float4 ga = (rp)[1];                                                                   \
        const float dy = pyc - ge.y;                                                                 \
        const float t1 = __fmul_rn(ge.w, dy), t2 = __fmul_rn(__fmul_rn(ga.x, dy), dy);               \
        const float dxa = pxc0 - ge.x;                                                               \
        pw_a[u] = __fmaf_rn(__fmaf_rn(ge.z, dxa, t1), dxa, t2);                                      \
        if (PPT == 2) {                                                                              \
            const float dxb = pxc1 - ge.x;                                                           \
            pw_b[u] = __fmaf_rn(__fmaf_rn(ge.z, dxb, t1), dxb, t2);                                  \
        }                                                                                            \
        thr[u] = ga.y; op[u] = ga.z;                                                                 \
        if (FEAT) zz[u] = ga.w;                                                                      \
        if (BF) c_##u = (rp)[2];                                                                     \
    }
    // valid = power <= 0 (L289, C20); alpha >= alpha_thresh <=> power >= -lnv (L679, C12)
    // BF (lists produced with tile_cull: > 90 % of the visited pairs pass the gate): branch-free -- a pixel that
    // is done or gated enters with alpha = 0, so T' = T >= t_min and w = 0; otherwise the gated pairs are branched over
#define XPR_FWD_BLEND(act, power, u, rp, T, C0, C1, C2, last, pos, Dv, Av)                            \
    if (BF) {                                                                                        \
        if (STATS) {                                                                                 \
            if (act) { ++n_visit; if (!((power) > 0.0f) && !((power) < thr[u])) ++n_pass; }          \
        }                                                                                            \
        const bool pass = act && !((power) > 0.0f) && !((power) < thr[u]);                           \
        const float alpha = pass ? fminf(amax, opac_exp(power, op[u])) : 0.0f;      /* C11 */        \
        const float Tn = T * (1.0f - alpha);                                                         \
        const bool stop = Tn < tmin;                                        /* C12: stop, no blend */\
        const bool blend = pass && !stop;                                                            \
        act = act && !stop;                                                                          \
        const float w = blend ? alpha * T : 0.0f;                                                    \
        C0 = fmaf(c_##u.x, w, C0); C1 = fmaf(c_##u.y, w, C1); C2 = fmaf(c_##u.z, w, C2);             \
        if (FEAT) { Dv = fmaf(zz[u], w, Dv); Av += w; }                                              \
        T = blend ? Tn : T;                                                                          \
        last = blend ? (pos) : last;                                                                 \
        if (STATS && blend) ++n_blend;                                                               \
    } else if (act) {                                                                                \
        if (STATS) ++n_visit;                                                                        \
        if (!((power) > 0.0f) && !((power) < thr[u])) {                                              \
            if (STATS) ++n_pass;                                                                     \
            const float alpha = fminf(amax, opac_exp(power, op[u]));        /* C11 */                \
            const float Tn = T * (1.0f - alpha);                                                     \
            if (Tn < tmin) {                                                /* C12: stop, no blend */\
                act = false;                                                                         \
            } else {                                                                                 \
                const float4 c = (rp)[2];                                                            \
                const float w = alpha * T;                                                           \
                C0 = fmaf(c.x, w, C0); C1 = fmaf(c.y, w, C1); C2 = fmaf(c.z, w, C2);                 \
                if (FEAT) { Dv = fmaf(zz[u], w, Dv); Av += w; }                                      \
                T = Tn;                                                                              \
                last = (pos);                                                                        \
                if (STATS) ++n_blend;                                                                \
            }                                                                                        \
        }                                                                                            \
    }
#define XPR_FWD_STEP(u, rp, pos)                                                                      \
    XPR_FWD_BLEND(act_a, pw_a[u], u, rp, Ta, Ca0, Ca1, Ca2, last_a, pos, Da, Aa)                      \
    if (PPT == 2) XPR_FWD_BLEND(act_b, pw_b[u], u, rp, Tb, Cb0, Cb1, Cb2, last_b, pos, Db, Ab)

    const float amax = P.amax, tmin = P.tmin;
    float pw_a[4], pw_b[4], thr[4], op[4], zz[4];
    float4 c_0, c_1, c_2, c_3;                         // colours of the group's entries
    for (uint32_t base = 0; base < len; base += FWD_BATCH) {
        if (__syncthreads_or(act_a || act_b) == 0) break;
        const uint32_t cnt = min((uint32_t)FWD_BATCH, len - base);
        for (uint32_t e = threadIdx.x; e < cnt; e += FWD_THREADS) {
            const uint32_t g = vals[rg.x + base + e];
            const float2 m = mean2d[g];
            const float4 co = conic_opac[g];
            float4* rec = s_rec + 3 * e;
            rec[0] = make_float4(m.x, m.y, -0.5f * co.x, -co.y);
            rec[1] = make_float4(-0.5f * co.z, -lnv[g], __log2f(co.w), FEAT ? depth[g] : 0.0f);
            rec[2] = make_float4(rgb[3 * g], rgb[3 * g + 1], rgb[3 * g + 2], 0.0f);
        }
        __syncthreads();
        if (act_a || act_b) {
            const float4* rq = s_rec;
            uint32_t j = 0;
            for (; j + 4 <= cnt && (act_a || act_b); j += 4, rq += 12) {
                XPR_FWD_POWER(0, rq) XPR_FWD_POWER(1, rq + 3) XPR_FWD_POWER(2, rq + 6) XPR_FWD_POWER(3, rq + 9)
                XPR_FWD_STEP(0, rq, base + j + 1)
                XPR_FWD_STEP(1, rq + 3, base + j + 2)
                XPR_FWD_STEP(2, rq + 6, base + j + 3)
                XPR_FWD_STEP(3, rq + 9, base + j + 4)
            }
            for (; j < cnt && (act_a || act_b); ++j, rq += 3) {
                XPR_FWD_POWER(0, rq)
                XPR_FWD_STEP(0, rq, base + j + 1)
            }
        }
    }
#undef XPR_FWD_POWER
#undef XPR_FWD_BLEND
#undef XPR_FWD_STEP
    if (STATS) {
        atomicAdd(stats + 0, (unsigned long long)n_visit); atomicAdd(stats + 1, (unsigned long long)n_pass);
        atomicAdd(stats + 2, (unsigned long long)n_blend); atomicAdd(stats + 3, (unsigned long long)(last_a + last_b));
        return;
    }
    if (in0) {
        const int64_t pid = (int64_t)py * P.W + px0;
        image[3 * pid] = fmaf(Ta, P.bg[0], Ca0);
        image[3 * pid + 1] = fmaf(Ta, P.bg[1], Ca1);
        image[3 * pid + 2] = fmaf(Ta, P.bg[2], Ca2);
        final_T[pid] = Ta;
        n_contrib[pid] = last_a;
        if (FEAT) { depth_img[pid] = Da; alpha_img[pid] = Aa; }
    }
    if (in1) {
        const int64_t pid = (int64_t)py * P.W + px1;
        image[3 * pid] = fmaf(Tb, P.bg[0], Cb0);
        image[3 * pid + 1] = fmaf(Tb, P.bg[1], Cb1);
        image[3 * pid + 2] = fmaf(Tb, P.bg[2], Cb2);
        final_T[pid] = Tb;
        n_contrib[pid] = last_b;
        if (FEAT) { depth_img[pid] = Db; alpha_img[pid] = Ab; }
    }
}

__device__ __forceinline__ float fast_rcp(float x) {   // rcp.approx (1 ulp); x = 1 - alpha in [0.01, 1]
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Transposed butterfly: reduces 8 per-lane values across the warp with 9 shuffles (4+2+1+1+1)
// instead of 40.  On return lane L with (L & 3) == 0 holds the warp total of value (L >> 2).
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

// Backward compositing (a9).  One CTA per 16x16 tile; a thread owns BWD_PPT consecutive pixels of one row
// (4 -> 64 threads, the throughput shape; 2 -> 128 threads for images with few tiles), so that a Gaussian's
// record is read from shared memory once per BWD_PPT pixel-pairs, the row terms of `power` are shared, and
// the per-Gaussian reduction runs once per 32 * BWD_PPT pixel-pairs: each lane first sums its own pixels in
// registers, then one transposed butterfly (14 shuffles for the 9 gradients) leaves the totals spread over
// lanes, which issue two RED instructions (8 lanes + 1 lane).
#ifndef XPR_BWD_PPT_SMALL
#define XPR_BWD_PPT_SMALL 2
#endif

#ifndef XPR_BWD_MINB
#define XPR_BWD_MINB 14      // 64-thread CTAs per SM in the throughput shape (72 registers, no spills; 12: +2.5 % time)
#endif
template <int BWD_PPT>
__global__ void __launch_bounds__(BLOCK / BWD_PPT, XPR_BWD_MINB * BWD_PPT / 4)
rasterize_bwd_kernel(RasterParams P, const float2* __restrict__ mean2d, const float4* __restrict__ conic_opac,
                     const float* __restrict__ rgb, const float* __restrict__ lnv,
                     const uint32_t* __restrict__ vals, const uint2* __restrict__ ranges,
                     const float* __restrict__ final_T, const uint32_t* __restrict__ n_contrib,
                     const float* __restrict__ dL, float* __restrict__ g_mean2d, float* __restrict__ g_conic,
                     float* __restrict__ g_opac, float* __restrict__ g_rgb) {
    constexpr int BWD_THREADS = BLOCK / BWD_PPT, BWD_BATCH = BWD_THREADS;
    __shared__ float4 s_geo[BWD_BATCH];   // mx, my, A, B
    __shared__ float4 s_gate[BWD_BATCH];  // C, thr, o, index (bits)
    __shared__ float4 s_col[BWD_BATCH];   // r, g, b, unused
    __shared__ uint32_t s_max[BWD_THREADS / 32];
    const int tile = P.order ? (int)P.order[blockIdx.x] : (int)blockIdx.x;
    const int tx = tile % P.TW, ty = tile / P.TW;
    const int lane = threadIdx.x & 31;
    // a thread owns BWD_PPT consecutive pixels of one row: they share dy and the row terms of `power`
    constexpr int TPR = TILE / BWD_PPT;                 // threads per tile row
    const int px0 = tx * TILE + (threadIdx.x % TPR) * BWD_PPT;
    const int py = ty * TILE + (threadIdx.x / TPR);
    const float pyc = (float)py + 0.5f;
    const uint2 rg = ranges[tile];

    uint32_t n[BWD_PPT];
    float T[BWD_PPT], Q[BWD_PPT], g0[BWD_PPT], g1[BWD_PPT], g2[BWD_PPT], pxc[BWD_PPT];
    uint32_t wmax = 0;
#pragma unroll
    for (int k = 0; k < BWD_PPT; ++k) {
        const int px = px0 + k;
        pxc[k] = (float)px + 0.5f;
        n[k] = 0; T[k] = 0.0f; g0[k] = g1[k] = g2[k] = 0.0f;
        if (px < P.W && py < P.H) {
            const int64_t pid = (int64_t)py * P.W + px;
            n[k] = n_contrib[pid];
            T[k] = final_T[pid];
            g0[k] = dL[3 * pid]; g1[k] = dL[3 * pid + 1]; g2[k] = dL[3 * pid + 2];
        }
        // colour behind the current entry, S_k = sum_{j>k} c_j alpha_j T_j + T_final bg (C13), enters only through
        // g . S_k: one running scalar Q_k = g . S_k = sum_{j>k} (g . c_j) alpha_j T_j + T_final (g . bg)
        Q[k] = T[k] * fmaf(g2[k], P.bg[2], fmaf(g1[k], P.bg[1], g0[k] * P.bg[0]));
        wmax = max(wmax, n[k]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) wmax = max(wmax, __shfl_xor_sync(0xffffffffu, wmax, o));
    if (lane == 0) s_max[threadIdx.x >> 5] = wmax;
    __syncthreads();
    uint32_t max_n = 0;
#pragma unroll
    for (int w = 0; w < BWD_THREADS / 32; ++w) max_n = max(max_n, s_max[w]);

    // lane (4 i) owns gradient i of the 8-value butterfly: its base pointer and per-Gaussian stride
    const int vi = lane >> 2;
    float* const red_base = (vi < 2) ? (g_mean2d + vi) : (vi < 5) ? (g_conic + (vi - 2)) : (g_rgb + (vi - 5));
    const uint32_t red_stride = (vi < 2) ? 2u : 3u;
    const bool red_lane = (lane & 3) == 0;

    for (uint32_t hi = max_n; hi > 0;) {
        const uint32_t cnt = min((uint32_t)BWD_BATCH, hi);
        __syncthreads();
        if (threadIdx.x < cnt) {      // slot j holds list position hi-1-j (descending)
            const uint32_t g = vals[rg.x + hi - 1 - threadIdx.x];
            const float2 m = mean2d[g];
            const float4 co = conic_opac[g];
            s_geo[threadIdx.x] = make_float4(m.x, m.y, co.x, co.y);
            s_gate[threadIdx.x] = make_float4(co.z, -lnv[g], co.w, __uint_as_float(g));
            s_col[threadIdx.x] = make_float4(rgb[3 * g], rgb[3 * g + 1], rgb[3 * g + 2], __log2f(co.w));
        }
        __syncthreads();
        for (uint32_t j = 0; j < cnt; ++j) {
            const uint32_t pos = hi - 1 - j;
            if (pos >= wmax) continue;     // warp-uniform: nobody in this warp got this far
            const float4 ge = s_geo[j];
            const float4 ga = s_gate[j];
            const float A = ge.z, Bc = ge.w, Cc = ga.x;
            const float qa = -0.5f * A, qb = -Bc, qc = -0.5f * Cc;
            const float dy = pyc - ge.y;
            const float t1 = __fmul_rn(qb, dy), t2 = __fmul_rn(__fmul_rn(qc, dy), dy);   // row terms of eval_power
            float dx[BWD_PPT], power[BWD_PPT];
            bool contrib[BWD_PPT], any_c = false;
#pragma unroll
            for (int k = 0; k < BWD_PPT; ++k) {
                dx[k] = pxc[k] - ge.x;
                power[k] = __fmaf_rn(__fmaf_rn(qa, dx[k], t1), dx[k], t2);               // = eval_power(qa, qb, qc, dx, dy)
                contrib[k] = (pos < n[k]) && !(power[k] > 0.0f) && !(power[k] < ga.y);
                any_c |= contrib[k];
            }
            if (!__any_sync(0xffffffffu, any_c)) continue;
            const float4 c = s_col[j];
            float v[8];                                // mx my A B C r g b
            v[5] = v[6] = v[7] = 0.f;
            // the thread's pixels share dy: accumulate sum dpow, sum dpow dx, sum dpow dx^2 and form the five
            // geometric gradients once per entry (dpow = dL/dpower of a pixel).  Branch-free over the pixels:
            // one that does not contribute enters with o G = 0, hence alpha = 0, 1/(1-alpha) = 1, w = 0 -- its T
            // and Q are unchanged and all its terms vanish.
            float sp = 0.f, spx = 0.f, spxx = 0.f;
#pragma unroll
            for (int k = 0; k < BWD_PPT; ++k) {
                const float og = contrib[k] ? opac_exp(power[k], c.w) : 0.0f;          // o G
                const float alpha = fminf(P.amax, og);
                const float inv = fast_rcp(1.0f - alpha);
                T[k] = T[k] * inv;                     // transmittance in front of this entry
                const float w = alpha * T[k];
                v[5] = fmaf(w, g0[k], v[5]); v[6] = fmaf(w, g1[k], v[6]); v[7] = fmaf(w, g2[k], v[7]);
                // dL/dalpha = sum_ch g_ch (c_ch T - S_ch / (1 - alpha)) = T (g . c) - (g . S) / (1 - alpha)
                const float gc = fmaf(g2[k], c.z, fmaf(g1[k], c.y, g0[k] * c.x));
                const float dalpha = fmaf(T[k], gc, -(inv * Q[k]));
                Q[k] = fmaf(gc, w, Q[k]);
                const float live = (og < P.amax) ? dalpha : 0.0f;   // C14: the clamp has zero derivative
                const float dpow = og * live;          // dL/dpower; dL/do = G live = dpow / o: summed as sp below
                const float dxp = dx[k] * dpow;
                sp += dpow; spx += dxp; spxx = fmaf(dx[k], dxp, spxx);
            }
            {
                const float sy = dy * sp;              // sum dpow dy
                v[0] = fmaf(A, spx, Bc * sy); v[1] = fmaf(Bc, spx, Cc * sy);
                v[2] = -0.5f * spxx; v[3] = -dy * spx; v[4] = -0.5f * dy * sy;
            }
            const float tot = warp_reduce8(v, lane);
            const float sp_tot = warp_sum(sp);         // dL/do = (sum dpow) / o, divided by the one lane that adds it
            const uint32_t g = __float_as_uint(ga.w);
            if (red_lane) atomicAdd(red_base + (size_t)red_stride * g, tot);
            if (lane == 0) atomicAdd(g_opac + g, sp_tot * fast_rcp(ga.z));
        }
        hi -= cnt;
    }
}

int32_t make_raster_params(const xpr_camera* cam, const xpr_config* cfg, RasterParams& P) {
    P.W = cam->width; P.H = cam->height; P.TW = tiles_x(cam);
    P.amax = cfg->alpha_max; P.tmin = cfg->t_min;
    for (int i = 0; i < 3; ++i) P.bg[i] = cfg->bg[i];
    P.order = cfg->tile_order;
    return XPR_OK;
}

}  // namespace
}  // namespace xpr

using namespace xpr;

extern "C" int32_t xpr_rasterize_fwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* mean2d,
                                     const float* conic_opac, const float* rgb, const float* lnv,
                                     const uint32_t* vals_sorted, const uint32_t* tile_ranges, float* image,
                                     float* final_T, uint32_t* n_contrib, void* stream) {
    if (int32_t s = check_cam_cfg(cam, cfg)) return s;
    if (N < 0) return XPR_ERR_INVALID_ARG;
    if (!aligned(tile_ranges, 8) || !aligned(image, 4) || !aligned(final_T, 4) || !aligned(n_contrib, 4))
        return XPR_ERR_INVALID_ARG;
    if (N > 0 && (!aligned(mean2d, 8) || !aligned(conic_opac, 16) || !aligned(rgb, 4) || !aligned(lnv, 4) ||
                  !aligned(vals_sorted, 4)))
        return XPR_ERR_INVALID_ARG;
    RasterParams P;
    make_raster_params(cam, cfg, P);
    const int T = tiles_x(cam) * tiles_y(cam);
    // throughput shape once the image has enough tiles for several waves of every SM; branch-free blend when
    // the lists were culled
#define XPR_FWD(PPT_, BF_)                                                                                          \
    rasterize_fwd_kernel<false, PPT_, BF_><<<T, BLOCK / PPT_, 0, (cudaStream_t)stream>>>(                             \
        P, reinterpret_cast<const float2*>(mean2d), reinterpret_cast<const float4*>(conic_opac), rgb, lnv,           \
        vals_sorted, reinterpret_cast<const uint2*>(tile_ranges), image, final_T, n_contrib, nullptr)
    const bool bf = cfg->tile_cull != 0;
    if (T >= FWD_PPT2_MIN_TILES) { if (bf) XPR_FWD(2, true); else XPR_FWD(2, false); }
    else                         { XPR_FWD(1, false); }      // latency shape: the branchy blend is shorter
#undef XPR_FWD
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}

extern "C" int32_t xpr_rasterize_feat_fwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* mean2d,
                                          const float* conic_opac, const float* rgb, const float* lnv,
                                          const float* depth, const uint32_t* vals_sorted,
                                          const uint32_t* tile_ranges, float* image, float* final_T,
                                          uint32_t* n_contrib, float* depth_img, float* alpha_img, void* stream) {
    if (int32_t s = check_cam_cfg(cam, cfg)) return s;
    if (N < 0) return XPR_ERR_INVALID_ARG;
    if (!aligned(tile_ranges, 8) || !aligned(image, 4) || !aligned(final_T, 4) || !aligned(n_contrib, 4) ||
        !aligned(depth_img, 4) || !aligned(alpha_img, 4))
        return XPR_ERR_INVALID_ARG;
    if (N > 0 && (!aligned(mean2d, 8) || !aligned(conic_opac, 16) || !aligned(rgb, 4) || !aligned(lnv, 4) ||
                  !aligned(depth, 4) || !aligned(vals_sorted, 4)))
        return XPR_ERR_INVALID_ARG;
    RasterParams P;
    make_raster_params(cam, cfg, P);
    const int T = tiles_x(cam) * tiles_y(cam);
    // the launch shapes of xpr_rasterize_fwd
#define XPR_FWD(PPT_, BF_)                                                                                          \
    rasterize_fwd_kernel<false, PPT_, BF_, true><<<T, BLOCK / PPT_, 0, (cudaStream_t)stream>>>(                       \
        P, reinterpret_cast<const float2*>(mean2d), reinterpret_cast<const float4*>(conic_opac), rgb, lnv,           \
        vals_sorted, reinterpret_cast<const uint2*>(tile_ranges), image, final_T, n_contrib, nullptr, depth,         \
        depth_img, alpha_img)
    const bool bf = cfg->tile_cull != 0;
    if (T >= FWD_PPT2_MIN_TILES) { if (bf) XPR_FWD(2, true); else XPR_FWD(2, false); }
    else                         { XPR_FWD(1, false); }
#undef XPR_FWD
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}

extern "C" int32_t xpr_rasterize_stats(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* mean2d,
                                       const float* conic_opac, const float* rgb, const float* lnv,
                                       const uint32_t* vals_sorted, const uint32_t* tile_ranges, uint64_t* stats,
                                       void* stream) {
    if (int32_t s = check_cam_cfg(cam, cfg)) return s;
    if (N < 0 || !aligned(tile_ranges, 8) || !aligned(stats, 8)) return XPR_ERR_INVALID_ARG;
    if (N > 0 && (!aligned(mean2d, 8) || !aligned(conic_opac, 16) || !aligned(rgb, 4) || !aligned(lnv, 4) ||
                  !aligned(vals_sorted, 4)))
        return XPR_ERR_INVALID_ARG;
    RasterParams P;
    make_raster_params(cam, cfg, P);
    const int T = tiles_x(cam) * tiles_y(cam);
    XPR_CUDA(cudaMemsetAsync(stats, 0, 4 * sizeof(uint64_t), (cudaStream_t)stream));
    rasterize_fwd_kernel<true, 1, false><<<T, BLOCK, 0, (cudaStream_t)stream>>>(
        P, reinterpret_cast<const float2*>(mean2d), reinterpret_cast<const float4*>(conic_opac), rgb, lnv,
        vals_sorted, reinterpret_cast<const uint2*>(tile_ranges), nullptr, nullptr, nullptr,
        reinterpret_cast<unsigned long long*>(stats));
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}

extern "C" int32_t xpr_rasterize_bwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* mean2d,
                                     const float* conic_opac, const float* rgb, const float* lnv,
                                     const uint32_t* vals_sorted, const uint32_t* tile_ranges, const float* final_T,
                                     const uint32_t* n_contrib, const float* dL_dimage, float* g_mean2d,
                                     float* g_conic, float* g_opac, float* g_rgb, int32_t zero_init, void* stream) {
    if (int32_t s = check_cam_cfg(cam, cfg)) return s;
    if (N < 0) return XPR_ERR_INVALID_ARG;
    if (!aligned(tile_ranges, 8) || !aligned(final_T, 4) || !aligned(n_contrib, 4) || !aligned(dL_dimage, 4))
        return XPR_ERR_INVALID_ARG;
    if (N == 0) return XPR_OK;
    if (!aligned(mean2d, 8) || !aligned(conic_opac, 16) || !aligned(rgb, 4) || !aligned(lnv, 4) ||
        !aligned(vals_sorted, 4) || !aligned(g_mean2d, 4) || !aligned(g_conic, 4) || !aligned(g_opac, 4) ||
        !aligned(g_rgb, 4))
        return XPR_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    if (zero_init) {
        const size_t n = (size_t)N;
        if (g_conic == g_mean2d + 2 * n && g_opac == g_conic + 3 * n && g_rgb == g_opac + n) {
            XPR_CUDA(cudaMemsetAsync(g_mean2d, 0, sizeof(float) * 9 * n, st));      // one allocation: one fill
        } else {
            XPR_CUDA(cudaMemsetAsync(g_mean2d, 0, sizeof(float) * 2 * n, st));
            XPR_CUDA(cudaMemsetAsync(g_conic, 0, sizeof(float) * 3 * n, st));
            XPR_CUDA(cudaMemsetAsync(g_opac, 0, sizeof(float) * n, st));
            XPR_CUDA(cudaMemsetAsync(g_rgb, 0, sizeof(float) * 3 * n, st));
        }
    }
    RasterParams P;
    make_raster_params(cam, cfg, P);
    const int T = tiles_x(cam) * tiles_y(cam);
    // 4 pixels per thread (64 threads) is the throughput shape; images with few tiles are bounded by their
    // heaviest tile, where more warps per tile (2 pixels per thread) shorten the critical path
    if (T >= FWD_PPT2_MIN_TILES)
        rasterize_bwd_kernel<4><<<T, BLOCK / 4, 0, st>>>(
            P, reinterpret_cast<const float2*>(mean2d), reinterpret_cast<const float4*>(conic_opac), rgb, lnv,
            vals_sorted, reinterpret_cast<const uint2*>(tile_ranges), final_T, n_contrib, dL_dimage, g_mean2d, g_conic,
            g_opac, g_rgb);
    else
        rasterize_bwd_kernel<XPR_BWD_PPT_SMALL><<<T, BLOCK / XPR_BWD_PPT_SMALL, 0, st>>>(
            P, reinterpret_cast<const float2*>(mean2d), reinterpret_cast<const float4*>(conic_opac), rgb, lnv,
            vals_sorted, reinterpret_cast<const uint2*>(tile_ranges), final_T, n_contrib, dL_dimage, g_mean2d, g_conic,
            g_opac, g_rgb);
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}
