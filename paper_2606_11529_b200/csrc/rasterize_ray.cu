// rasterize_ray.cu -- xpr_rasterize_ray_fwd / _bwd: per-tile front-to-back compositing with the XPR-3DGUT
// evaluation (PAPER A.1.2 L437-444 Eq. 1, Listing 3) and its reverse-mode pass.
//
// Same tile / list / batch structure as rasterize.cu; the per-entry evaluation is the maximum response of the 3D
// Gaussian along the pixel's camera ray d (reading C27, camera frame):
//   d_c = M_c d,  c = o_c x d_c,  nhq = -1/2 |c|^2,  dd = |d_c|^2,  response = exp(nhq / dd).
// Decisions are taken on products in the fixed fp32 order of rule R3 (explicit _rn intrinsics), never on the
// quotient or on exp():  valid <=> nhq > ln(0.0113) dd (L500),  gate <=> nhq >= -lnv dd (C12).
#include <math.h>

#include "common.cuh"
#include "packed.cuh"

namespace xpr {
namespace {

constexpr int BLOCK = TILE * TILE;

struct RayRasterParams {
    int W, H, TW;
    float amax, tmin, lnr;     // lnr = (float) ln(0.0113)
    float bg[3];
    const uint32_t* order;     // xpr_config.tile_order: CTA b works on tile order[b] (longest lists first), or NULL
};

// evaluate (Listing 3) in the fixed fp32 order of DESIGN.md 3 (rule R3)
struct RayEval { float dc0, dc1, dc2, c0, c1, c2, nhq, dd; };
__device__ __forceinline__ RayEval eval_ray(const float4 r0, const float4 r1, const float4 r2, float d0, float d1,
                                            float d2) {
    RayEval e;
    e.dc0 = __fmaf_rn(r0.z, d2, __fmaf_rn(r0.y, d1, __fmul_rn(r0.x, d0)));
    e.dc1 = __fmaf_rn(r1.y, d2, __fmaf_rn(r1.x, d1, __fmul_rn(r0.w, d0)));
    e.dc2 = __fmaf_rn(r2.x, d2, __fmaf_rn(r1.w, d1, __fmul_rn(r1.z, d0)));
    const float o0 = r2.y, o1 = r2.z, o2 = r2.w;
    e.c0 = __fmaf_rn(o1, e.dc2, -__fmul_rn(o2, e.dc1));
    e.c1 = __fmaf_rn(o2, e.dc0, -__fmul_rn(o0, e.dc2));
    e.c2 = __fmaf_rn(o0, e.dc1, -__fmul_rn(o1, e.dc0));
    const float q = __fmaf_rn(e.c2, e.c2, __fmaf_rn(e.c1, e.c1, __fmul_rn(e.c0, e.c0)));
    e.dd = __fmaf_rn(e.dc2, e.dc2, __fmaf_rn(e.dc1, e.dc1, __fmul_rn(e.dc0, e.dc0)));
    e.nhq = __fmul_rn(-0.5f, q);
    return e;
}

// The same evaluation for a PAIR of pixels with the packed fp32 instructions of sm_100 (packed.cuh): the record operands are
// broadcast, the two rays sit in the two lanes; every lane is rounded exactly as the scalar code above (rule R3 holds).
struct RayEval2 { f32x2 dc0, dc1, dc2, c0, c1, c2, nhq, dd; };
__device__ __forceinline__ RayEval2 eval_ray2(const float4 r0, const float4 r1, const float4 r2, f32x2 d0, f32x2 d1, f32x2 d2) {
    RayEval2 e;
    e.dc0 = fma2(bcast2(r0.z), d2, fma2(bcast2(r0.y), d1, mul2(bcast2(r0.x), d0)));
    e.dc1 = fma2(bcast2(r1.y), d2, fma2(bcast2(r1.x), d1, mul2(bcast2(r0.w), d0)));
    e.dc2 = fma2(bcast2(r2.x), d2, fma2(bcast2(r1.w), d1, mul2(bcast2(r1.z), d0)));
    const f32x2 o0 = bcast2(r2.y), o1 = bcast2(r2.z), o2 = bcast2(r2.w);
    e.c0 = fma2(o1, e.dc2, neg2(mul2(o2, e.dc1)));
    e.c1 = fma2(o2, e.dc0, neg2(mul2(o0, e.dc2)));
    e.c2 = fma2(o0, e.dc1, neg2(mul2(o1, e.dc0)));
    const f32x2 q = fma2(e.c2, e.c2, fma2(e.c1, e.c1, mul2(e.c0, e.c0)));
    e.dd = fma2(e.dc2, e.dc2, fma2(e.dc1, e.dc1, mul2(e.dc0, e.dc0)));
    e.nhq = mul2(bcast2(-0.5f), q);
    return e;
}
// Forward (a8 with the f2 evaluation).  One CTA per tile in the two shapes of rasterize.cu: PPT = 2 (128 threads, a
// thread owns the pixels (x, y) and (x + 8, y): the shared-memory reads of a list entry are paid once per two
// pixels) for large images, PPT = 1 (256 threads) where the heaviest tile bounds the kernel.  Record of a list
// entry in shared memory: 5 x float4 = (M_c, o_c | thr = -lnv, log2 o, r, g | b).  STATS as in rasterize.cu.
struct RayPix {
    float d0, d1, d2, T, C0, C1, C2;
    float D, A;            // FEAT: rendered depth and accumulated opacity (reading C31)
    uint32_t last;
};

template <bool STATS, bool FEAT = false>
__device__ __forceinline__ void ray_blend(RayPix& p, int& act, float nhq, float dd, const float4* __restrict__ rec, uint32_t pos,
                                          float lnr, float amax, float tmin, uint32_t& n_visit, uint32_t& n_pass,
                                          uint32_t& n_blend) {
    if (!act) return;
    if (STATS) ++n_visit;
    const float4 at = rec[3];
    const float tv = __fmul_rn(lnr, dd), tg = __fmul_rn(at.x, dd);
    if ((nhq > tv) && !(nhq < tg)) {                      // valid (L500) and alpha >= alpha_thresh (C12)
        if (STATS) ++n_pass;
        const float power = nhq * rcp_approx(dd);
        const float alpha = fminf(amax, ex2_approx(fmaf(power, 1.4426950408889634f, at.y)));   // C11
        const float Tn = p.T * (1.0f - alpha);
        if (Tn < tmin) {                                  // C12: stop, no blend
            act = 0;
        } else {
            const float w = alpha * p.T;
            p.C0 = fmaf(at.z, w, p.C0); p.C1 = fmaf(at.w, w, p.C1); p.C2 = fmaf(rec[4].x, w, p.C2);
            if (FEAT) { p.D = fmaf(rec[4].y, w, p.D); p.A += w; }
            p.T = Tn;
            p.last = pos;
            if (STATS) ++n_blend;
        }
    }
}

#ifndef XPR_RAY_FWD_PPT2_MIN_TILES
#define XPR_RAY_FWD_PPT2_MIN_TILES 4096
#endif

template <bool STATS, int PPT, bool FEAT = false>
__global__ void __launch_bounds__(BLOCK / PPT)
rasterize_ray_fwd_kernel(RayRasterParams P, const float4* __restrict__ ray_rec, const float4* __restrict__ conic_opac,
                         const float* __restrict__ rgb, const float* __restrict__ lnv, const float* __restrict__ rays,
                         const uint32_t* __restrict__ vals, const uint2* __restrict__ ranges,
                         float* __restrict__ image, float* __restrict__ final_T, uint32_t* __restrict__ n_contrib,
                         unsigned long long* __restrict__ stats, const float* __restrict__ depth = nullptr,
                         float* __restrict__ depth_img = nullptr, float* __restrict__ alpha_img = nullptr) {
    constexpr int THREADS = BLOCK / PPT, BATCH = THREADS, ROW = TILE / PPT;
    __shared__ float4 s_rec[5 * BATCH];
    const int tile = P.order ? (int)P.order[blockIdx.x] : (int)blockIdx.x;
    const int tx = tile % P.TW, ty = tile / P.TW;
    const int py = ty * TILE + (threadIdx.x / ROW);
    int px[PPT];
    int inside[PPT];
    RayPix pix[PPT];
    int act[PPT];
    bool any_act = false;
#pragma unroll
    for (int k = 0; k < PPT; ++k) {
        px[k] = tx * TILE + (threadIdx.x % ROW) + 8 * k;
        inside[k] = ((px[k] < P.W) && (py < P.H)) ? 1 : 0;
        pix[k].d0 = 0.f; pix[k].d1 = 0.f; pix[k].d2 = 1.f;
        if (inside[k]) {
            const int64_t pid = (int64_t)py * P.W + px[k];
            pix[k].d0 = rays[3 * pid]; pix[k].d1 = rays[3 * pid + 1]; pix[k].d2 = rays[3 * pid + 2];
        }
        pix[k].T = 1.0f; pix[k].C0 = pix[k].C1 = pix[k].C2 = 0.0f; pix[k].D = pix[k].A = 0.0f; pix[k].last = 0; act[k] = inside[k] ? 1 : 0;
        any_act |= (inside[k] != 0);
    }
    const uint2 rg = ranges[tile];
    const uint32_t len = rg.y - rg.x;
    const float amax = P.amax, tmin = P.tmin, lnr = P.lnr;
    uint32_t n_visit = 0, n_pass = 0, n_blend = 0;
    // the pixel pair's ray components, lane 0 = pixel 0, lane 1 = pixel 1 (PPT == 2)
    const f32x2 D0 = pack2(pix[0].d0, pix[PPT - 1].d0), D1 = pack2(pix[0].d1, pix[PPT - 1].d1), D2 = pack2(pix[0].d2, pix[PPT - 1].d2);

    for (uint32_t base = 0; base < len; base += BATCH) {
        if (__syncthreads_or(any_act) == 0) break;
        const uint32_t cnt = min((uint32_t)BATCH, len - base);
        if (threadIdx.x < cnt) {
            const uint32_t g = vals[rg.x + base + threadIdx.x];
            float4* rec = s_rec + 5 * threadIdx.x;
            rec[0] = ray_rec[3 * (size_t)g]; rec[1] = ray_rec[3 * (size_t)g + 1]; rec[2] = ray_rec[3 * (size_t)g + 2];
            rec[3] = make_float4(-lnv[g], __log2f(conic_opac[g].w), rgb[3 * (size_t)g], rgb[3 * (size_t)g + 1]);
            rec[4] = make_float4(rgb[3 * (size_t)g + 2], FEAT ? depth[g] : 0.f, 0.f, 0.f);
        }
        __syncthreads();
        if (any_act) {
            // groups of 4: the evaluations are independent of the transmittance, so their latencies overlap; the
            // sequential part (gates, alpha, T' = T (1 - alpha), exit test, blend) follows
            const float4* rq = s_rec;
            uint32_t j = 0;
            for (; j + 4 <= cnt && any_act; j += 4, rq += 20) {
                float nhq[4][PPT], dd[4][PPT];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const float4 r0 = rq[5 * u], r1 = rq[5 * u + 1], r2 = rq[5 * u + 2];
                    if (PPT == 2) {
                        const RayEval2 e = eval_ray2(r0, r1, r2, D0, D1, D2);
                        unpack2(e.nhq, nhq[u][0], nhq[u][PPT - 1]); unpack2(e.dd, dd[u][0], dd[u][PPT - 1]);
                    } else {
                        const RayEval e = eval_ray(r0, r1, r2, pix[0].d0, pix[0].d1, pix[0].d2);
                        nhq[u][0] = e.nhq; dd[u][0] = e.dd;
                    }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u)
#pragma unroll
                    for (int k = 0; k < PPT; ++k)
                        ray_blend<STATS, FEAT>(pix[k], act[k], nhq[u][k], dd[u][k], rq + 5 * u, base + j + u + 1, lnr, amax, tmin,
                                         n_visit, n_pass, n_blend);
                any_act = (act[0] | act[PPT - 1]) != 0;
            }
            for (; j < cnt && any_act; ++j, rq += 5) {
                const float4 r0 = rq[0], r1 = rq[1], r2 = rq[2];
                if (PPT == 2) {
                    const RayEval2 e2 = eval_ray2(r0, r1, r2, D0, D1, D2);
                    float na, nb, da, db;
                    unpack2(e2.nhq, na, nb); unpack2(e2.dd, da, db);
                    ray_blend<STATS, FEAT>(pix[0], act[0], na, da, rq, base + j + 1, lnr, amax, tmin, n_visit, n_pass, n_blend);
                    ray_blend<STATS, FEAT>(pix[PPT - 1], act[PPT - 1], nb, db, rq, base + j + 1, lnr, amax, tmin, n_visit, n_pass, n_blend);
                } else {
                    const RayEval e = eval_ray(r0, r1, r2, pix[0].d0, pix[0].d1, pix[0].d2);
                    ray_blend<STATS, FEAT>(pix[0], act[0], e.nhq, e.dd, rq, base + j + 1, lnr, amax, tmin, n_visit, n_pass, n_blend);
                }
                any_act = (act[0] | act[PPT - 1]) != 0;
            }
        }
    }
    if (STATS) {
        uint32_t sum_last = 0;
#pragma unroll
        for (int k = 0; k < PPT; ++k) sum_last += pix[k].last;
        atomicAdd(stats + 0, (unsigned long long)n_visit); atomicAdd(stats + 1, (unsigned long long)n_pass);
        atomicAdd(stats + 2, (unsigned long long)n_blend); atomicAdd(stats + 3, (unsigned long long)sum_last);
        return;
    }
#pragma unroll
    for (int k = 0; k < PPT; ++k)
        if (inside[k]) {
            const int64_t pid = (int64_t)py * P.W + px[k];
            image[3 * pid] = fmaf(pix[k].T, P.bg[0], pix[k].C0);
            image[3 * pid + 1] = fmaf(pix[k].T, P.bg[1], pix[k].C1);
            image[3 * pid + 2] = fmaf(pix[k].T, P.bg[2], pix[k].C2);
            final_T[pid] = pix[k].T;
            n_contrib[pid] = pix[k].last;
            if (FEAT) { depth_img[pid] = pix[k].D; alpha_img[pid] = pix[k].A; }
        }
}

// Backward (a9 with the f2 evaluation).  A thread owns PPT consecutive pixels of a row and sums their 19 gradient
// terms per entry in registers; two transposed butterflies of 8 and one of 4 leave the warp totals spread over the
// lanes, which issue the RED instructions.  With g_p = dL/dpower, k = -g_p / dd:
//   dL/dc = k c,  dL/ddd = -g_p power/dd = k power,  dL/do_c = d_c x dL/dc.
// The record gradient is accumulated in a form that does not cancel: the plain sums (dL/dM_c = dL/dd_c d^T, dL/do_c)
// enter the chain rule only as dL/dM_c - dL/do_c p^T, whose two parts nearly cancel (a ray through the centre has
// c = 0) -- in fp32 that lost the small components of the scale and quaternion gradients.  With o_c = -M_c p,
// d_c = M_c d, c = o_c x d_c the difference is exactly  -(S_c - tr(S_c) I) M_c^-T + M_c D  with
//   S_c = sum k c c^T (6),   D = sum 2 dL/ddd d d^T (6),
// so the kernel sums g_ray_acc[N,16] = (S_c: xx xy xz yy yz zz | D: xx xy xz yy yz zz | sum dL/do_c (3) | unused) and
// xpr_ray_bwd applies M_c once per Gaussian in fp64.
// Transposed butterfly of 4 values (6 shuffles): lane L with (L & 7) == 0 holds the total of value L >> 3.
__device__ __forceinline__ float warp_reduce4(const float* v, int lane) {
    const bool b4 = lane & 16, b3 = lane & 8;
    float w[2];
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const float send = b4 ? v[i] : v[i + 2], keep = b4 ? v[i + 2] : v[i];
        w[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
    const float send = b3 ? w[0] : w[1], keep = b3 ? w[1] : w[0];
    float y = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    y += __shfl_xor_sync(0xffffffffu, y, 4);
    y += __shfl_xor_sync(0xffffffffu, y, 2);
    y += __shfl_xor_sync(0xffffffffu, y, 1);
    return y;
}

#ifndef XPR_RAY_BWD_PPT
#define XPR_RAY_BWD_PPT 4
#endif
#ifndef XPR_RAY_BWD_MINB
#define XPR_RAY_BWD_MINB 6
#endif
// FEAT (xpr_rasterize_ray_feat_bwd; reading C31, as rasterize.cu): with gD = dL/dD, gA = dL/dA of the pixel,
//   dL/dz_k = alpha_k T_k gD;  g . c_k becomes g . c_k + gD z_k;  the accumulated-opacity term is the constant -gA T_final in Q.
template <int PPT, bool FEAT = false>
__global__ void __launch_bounds__(BLOCK / PPT, XPR_RAY_BWD_MINB * PPT / 4)
rasterize_ray_bwd_kernel(RayRasterParams P, const float4* __restrict__ ray_rec, const float4* __restrict__ conic_opac,
                         const float* __restrict__ rgb, const float* __restrict__ lnv, const float* __restrict__ rays,
                         const uint32_t* __restrict__ vals, const uint2* __restrict__ ranges,
                         const float* __restrict__ final_T, const uint32_t* __restrict__ n_contrib,
                         const float* __restrict__ dL, float* __restrict__ g_acc, float* __restrict__ g_opac,
                         float* __restrict__ g_rgb, const float* __restrict__ depth = nullptr,
                         const float* __restrict__ dL_dD = nullptr, const float* __restrict__ dL_dA = nullptr,
                         float* __restrict__ g_depth = nullptr) {
    constexpr int THREADS = BLOCK / PPT, BATCH = THREADS;
    __shared__ float4 s_geo[3 * BATCH];
    __shared__ float4 s_gate[BATCH];   // thr, o, log2 o, index (bits)
    __shared__ float4 s_col[BATCH];    // r, g, b, -
    __shared__ uint32_t s_max[THREADS / 32];
    const int tile = P.order ? (int)P.order[blockIdx.x] : (int)blockIdx.x;
    const int tx = tile % P.TW, ty = tile / P.TW;
    const int lane = threadIdx.x & 31;
    constexpr int TPR = TILE / PPT;
    const int px0 = tx * TILE + (threadIdx.x % TPR) * PPT;
    const int py = ty * TILE + (threadIdx.x / TPR);
    const uint2 rg = ranges[tile];
    const float lnr = P.lnr;

    uint32_t n[PPT];
    float T[PPT], Q[PPT], g0[PPT], g1[PPT], g2[PPT], d0[PPT], d1[PPT], d2[PPT], gD[PPT];
    uint32_t wmax = 0;
#pragma unroll
    for (int k = 0; k < PPT; ++k) {
        const int px = px0 + k;
        n[k] = 0; T[k] = 0.0f; g0[k] = g1[k] = g2[k] = 0.0f; d0[k] = d1[k] = 0.0f; d2[k] = 1.0f; gD[k] = 0.0f;
        float gA = 0.0f;
        if (px < P.W && py < P.H) {
            const int64_t pid = (int64_t)py * P.W + px;
            n[k] = n_contrib[pid];
            T[k] = final_T[pid];
            g0[k] = dL[3 * pid]; g1[k] = dL[3 * pid + 1]; g2[k] = dL[3 * pid + 2];
            d0[k] = rays[3 * pid]; d1[k] = rays[3 * pid + 1]; d2[k] = rays[3 * pid + 2];
            if (FEAT) { gD[k] = dL_dD[pid]; gA = dL_dA[pid]; }
        }
        // Q_k = g . S_k, the colour behind the entry as one running scalar (rasterize.cu) (FEAT: - gA T_final)
        Q[k] = T[k] * (fmaf(g2[k], P.bg[2], fmaf(g1[k], P.bg[1], g0[k] * P.bg[0])) - gA);
        wmax = max(wmax, n[k]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) wmax = max(wmax, __shfl_xor_sync(0xffffffffu, wmax, o));
    if (lane == 0) s_max[threadIdx.x >> 5] = wmax;
    __syncthreads();
    uint32_t max_n = 0;
#pragma unroll
    for (int w = 0; w < THREADS / 32; ++w) max_n = max(max_n, s_max[w]);
    // the thread's pixels as PAIRS of neighbours (lane 0 = pixel 2p, lane 1 = pixel 2p + 1) for the packed fp32
    // instructions of sm_100 (packed.cuh): the evaluation, the blend weights and the accumulator terms run two pixels per
    // issue slot; the two lanes of an accumulator are added once per entry, before the warp reduction
    constexpr int NP = PPT / 2;
    f32x2 T2[NP], Q2[NP], g0_2[NP], g1_2[NP], g2_2[NP], gD_2[NP], d0_2[NP], d1_2[NP], d2_2[NP];
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        T2[p] = pack2(T[2 * p], T[2 * p + 1]); Q2[p] = pack2(Q[2 * p], Q[2 * p + 1]);
        g0_2[p] = pack2(g0[2 * p], g0[2 * p + 1]); g1_2[p] = pack2(g1[2 * p], g1[2 * p + 1]); g2_2[p] = pack2(g2[2 * p], g2[2 * p + 1]);
        gD_2[p] = pack2(gD[2 * p], gD[2 * p + 1]);
        d0_2[p] = pack2(d0[2 * p], d0[2 * p + 1]); d1_2[p] = pack2(d1[2 * p], d1[2 * p + 1]); d2_2[p] = pack2(d2[2 * p], d2[2 * p + 1]);
    }
    const float amax = P.amax;

    // lane 4 i owns value i of butterfly A (g_acc[0..8): S_c, D_xx, D_xy) and value i of butterfly B (g_acc[8..15):
    // D_xz .. D_zz, sum dL/do_c; value 7: dL/do); lane 8 i owns colour channel i of the 4-value butterfly
    const int vi = lane >> 2;
    const bool red_lane = (lane & 3) == 0;

    for (uint32_t hi = max_n; hi > 0;) {
        const uint32_t cnt = min((uint32_t)BATCH, hi);
        __syncthreads();
        if (threadIdx.x < cnt) {      // slot j holds list position hi-1-j (descending)
            const uint32_t g = vals[rg.x + hi - 1 - threadIdx.x];
            s_geo[3 * threadIdx.x] = ray_rec[3 * (size_t)g];
            s_geo[3 * threadIdx.x + 1] = ray_rec[3 * (size_t)g + 1];
            s_geo[3 * threadIdx.x + 2] = ray_rec[3 * (size_t)g + 2];
            const float o = conic_opac[g].w;
            s_gate[threadIdx.x] = make_float4(-lnv[g], o, __log2f(o), __uint_as_float(g));
            s_col[threadIdx.x] = make_float4(rgb[3 * (size_t)g], rgb[3 * (size_t)g + 1], rgb[3 * (size_t)g + 2],
                                             FEAT ? depth[g] : 0.0f);
        }
        __syncthreads();
        for (uint32_t j = 0; j < cnt; ++j) {
            const uint32_t pos = hi - 1 - j;
            if (pos >= wmax) continue;     // warp-uniform
            const float4 r0 = s_geo[3 * j], r1 = s_geo[3 * j + 1], r2 = s_geo[3 * j + 2];
            const float4 ga = s_gate[j];
            RayEval2 e2[NP];
            float nhq[PPT], dd[PPT];
            bool contrib[PPT], any_c = false;
#pragma unroll
            for (int p = 0; p < NP; ++p) {
                e2[p] = eval_ray2(r0, r1, r2, d0_2[p], d1_2[p], d2_2[p]);
                unpack2(e2[p].nhq, nhq[2 * p], nhq[2 * p + 1]); unpack2(e2[p].dd, dd[2 * p], dd[2 * p + 1]);
            }
#pragma unroll
            for (int k = 0; k < PPT; ++k) {
                const float tv = __fmul_rn(lnr, dd[k]), tg = __fmul_rn(ga.x, dd[k]);
                contrib[k] = (pos < n[k]) && (nhq[k] > tv) && !(nhq[k] < tg);
                any_c |= contrib[k];
            }
            if (!__any_sync(0xffffffffu, any_c)) continue;
            const float4 c = s_col[j];
            f32x2 va2[8], vb2[8], vc2[4];
#pragma unroll
            for (int i = 0; i < 8; ++i) va2[i] = vb2[i] = 0ull;
            vc2[0] = vc2[1] = vc2[2] = vc2[3] = 0ull;
#pragma unroll
            for (int p = 0; p < NP; ++p) {
                const int k = 2 * p;
                // a pixel that does not contribute enters with 1/dd = 0 and o G = 0: every term vanishes
                const f32x2 rdd2 = pack2(contrib[k] ? rcp_approx(dd[k]) : 0.0f, contrib[k + 1] ? rcp_approx(dd[k + 1]) : 0.0f);
                const f32x2 power2 = mul2(e2[p].nhq, rdd2);
                float ea, eb;
                unpack2(fma2(power2, bcast2(LOG2E), bcast2(ga.z)), ea, eb);
                const float og_a = contrib[k] ? ex2_approx(ea) : 0.0f, og_b = contrib[k + 1] ? ex2_approx(eb) : 0.0f;   // o G
                const f32x2 al2 = pack2(fminf(amax, og_a), fminf(amax, og_b));
                float oma_a, oma_b;
                unpack2(sub2(bcast2(1.0f), al2), oma_a, oma_b);
                const f32x2 inv2 = pack2(rcp_approx(oma_a), rcp_approx(oma_b));
                T2[p] = mul2(T2[p], inv2);             // transmittance in front of this entry
                const f32x2 w2 = mul2(al2, T2[p]);
                vc2[0] = fma2(w2, g0_2[p], vc2[0]); vc2[1] = fma2(w2, g1_2[p], vc2[1]); vc2[2] = fma2(w2, g2_2[p], vc2[2]);
                f32x2 gc2 = fma2(g2_2[p], bcast2(c.z), fma2(g1_2[p], bcast2(c.y), mul2(g0_2[p], bcast2(c.x))));
                if (FEAT) { vc2[3] = fma2(w2, gD_2[p], vc2[3]); gc2 = fma2(gD_2[p], bcast2(c.w), gc2); }   // dL/dz; g . c + gD z
                float da_a, da_b;
                unpack2(fma2(T2[p], gc2, neg2(mul2(inv2, Q2[p]))), da_a, da_b);
                Q2[p] = fma2(gc2, w2, Q2[p]);
                // C14: no gradient where the clamp is active; dL/dpower = o G dL/dalpha (dL/do = that / o, divided once per warp)
                const f32x2 gp2 = mul2(pack2(og_a, og_b), pack2((og_a < amax) ? da_a : 0.0f, (og_b < amax) ? da_b : 0.0f));
                vb2[7] = add2(vb2[7], gp2);
                const f32x2 k1 = mul2(neg2(gp2), rdd2);                  // dL/dc = k1 c
                const f32x2 gc0 = mul2(k1, e2[p].c0), gc1 = mul2(k1, e2[p].c1), gcz = mul2(k1, e2[p].c2);
                // S_c += k1 c c^T
                va2[0] = fma2(gc0, e2[p].c0, va2[0]); va2[1] = fma2(gc0, e2[p].c1, va2[1]); va2[2] = fma2(gc0, e2[p].c2, va2[2]);
                va2[3] = fma2(gc1, e2[p].c1, va2[3]); va2[4] = fma2(gc1, e2[p].c2, va2[4]); va2[5] = fma2(gcz, e2[p].c2, va2[5]);
                // D += 2 dL/ddd d d^T,  2 dL/ddd = 2 k1 power
                const f32x2 gdd2 = mul2(mul2(bcast2(2.0f), k1), power2);
                const f32x2 t0 = mul2(gdd2, d0_2[p]), t1 = mul2(gdd2, d1_2[p]), t2 = mul2(gdd2, d2_2[p]);
                va2[6] = fma2(t0, d0_2[p], va2[6]); va2[7] = fma2(t0, d1_2[p], va2[7]); vb2[0] = fma2(t0, d2_2[p], vb2[0]);
                vb2[1] = fma2(t1, d1_2[p], vb2[1]); vb2[2] = fma2(t1, d2_2[p], vb2[2]); vb2[3] = fma2(t2, d2_2[p], vb2[3]);
                // dL/do_c = d_c x dL/dc
                vb2[4] = add2(vb2[4], fma2(e2[p].dc1, gcz, neg2(mul2(e2[p].dc2, gc1))));
                vb2[5] = add2(vb2[5], fma2(e2[p].dc2, gc0, neg2(mul2(e2[p].dc0, gcz))));
                vb2[6] = add2(vb2[6], fma2(e2[p].dc0, gc1, neg2(mul2(e2[p].dc1, gc0))));
            }
            float va[8], vb[8], vc[4];
#pragma unroll
            for (int i = 0; i < 8; ++i) { va[i] = sum2(va2[i]); vb[i] = sum2(vb2[i]); }
#pragma unroll
            for (int i = 0; i < 4; ++i) vc[i] = sum2(vc2[i]);
            const float ta = warp_reduce8(va, lane);
            float tb = warp_reduce8(vb, lane);
            const float tc = warp_reduce4(vc, lane);
            const uint32_t g = __float_as_uint(ga.w);
            if (red_lane) {
                atomicAdd(g_acc + 16 * (size_t)g + vi, ta);
                if (vi == 7) atomicAdd(g_opac + g, tb * rcp_approx(ga.y));   // dL/do = (sum g_p) / o
                else atomicAdd(g_acc + 16 * (size_t)g + 8 + vi, tb);
            }
            if ((lane & 7) == 0 && lane < 24) atomicAdd(g_rgb + 3 * (size_t)g + (lane >> 3), tc);
            if (FEAT && lane == 24) atomicAdd(g_depth + g, tc);
        }
        hi -= cnt;
    }
}

int32_t make_params(const xpr_camera* cam, const xpr_config* cfg, RayRasterParams& P) {
    P.W = cam->width; P.H = cam->height; P.TW = tiles_x(cam);
    P.amax = cfg->alpha_max; P.tmin = cfg->t_min;
    P.lnr = (float)log(0.0113);
    for (int i = 0; i < 3; ++i) P.bg[i] = cfg->bg[i];
    P.order = cfg->tile_order;
    return XPR_OK;
}

int32_t check_ray_cam_cfg(const xpr_camera* cam, const xpr_config* cfg) {
    if (!cam || !cfg) return XPR_ERR_INVALID_ARG;
    if (cam->width <= 0 || cam->height <= 0) return XPR_ERR_INVALID_ARG;
    if (cfg->tile != TILE) return XPR_ERR_UNSUPPORTED;
    return XPR_OK;
}

}  // namespace
}  // namespace xpr

using namespace xpr;

static int32_t ray_fwd_impl(bool feat, const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* ray_rec,
                            const float* conic_opac, const float* rgb, const float* lnv, const float* depth,
                            const float* pixel_rays, const uint32_t* vals_sorted, const uint32_t* tile_ranges, float* image,
                            float* final_T, uint32_t* n_contrib, float* depth_img, float* alpha_img, void* stream) {
    if (int32_t s = check_ray_cam_cfg(cam, cfg)) return s;
    if (N < 0) return XPR_ERR_INVALID_ARG;
    if (!aligned(tile_ranges, 8) || !aligned(image, 4) || !aligned(final_T, 4) || !aligned(n_contrib, 4) ||
        !aligned(pixel_rays, 4))
        return XPR_ERR_INVALID_ARG;
    if (feat && (!aligned(depth_img, 4) || !aligned(alpha_img, 4))) return XPR_ERR_INVALID_ARG;
    if (N > 0 && (!aligned(ray_rec, 16) || !aligned(conic_opac, 16) || !aligned(rgb, 4) || !aligned(lnv, 4) ||
                  !aligned(vals_sorted, 4) || (feat && !aligned(depth, 4))))
        return XPR_ERR_INVALID_ARG;
    RayRasterParams P;
    make_params(cam, cfg, P);
    const int T = tiles_x(cam) * tiles_y(cam);
#define XPR_RAY_FWD(PPT_, FEAT_)                                                                                      \
    rasterize_ray_fwd_kernel<false, PPT_, FEAT_><<<T, BLOCK / PPT_, 0, (cudaStream_t)stream>>>(                       \
        P, reinterpret_cast<const float4*>(ray_rec), reinterpret_cast<const float4*>(conic_opac), rgb, lnv, pixel_rays, \
        vals_sorted, reinterpret_cast<const uint2*>(tile_ranges), image, final_T, n_contrib, nullptr, depth, depth_img, \
        alpha_img)
    // throughput shape once the image has enough tiles for several waves of every SM
    const bool big = T >= XPR_RAY_FWD_PPT2_MIN_TILES;
    if (feat) { if (big) XPR_RAY_FWD(2, true); else XPR_RAY_FWD(1, true); }
    else      { if (big) XPR_RAY_FWD(2, false); else XPR_RAY_FWD(1, false); }
#undef XPR_RAY_FWD
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}

extern "C" int32_t xpr_rasterize_ray_fwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* ray_rec,
                                         const float* conic_opac, const float* rgb, const float* lnv,
                                         const float* pixel_rays, const uint32_t* vals_sorted,
                                         const uint32_t* tile_ranges, float* image, float* final_T,
                                         uint32_t* n_contrib, void* stream) {
    return ray_fwd_impl(false, cam, cfg, N, ray_rec, conic_opac, rgb, lnv, nullptr, pixel_rays, vals_sorted, tile_ranges,
                        image, final_T, n_contrib, nullptr, nullptr, stream);
}

extern "C" int32_t xpr_rasterize_ray_feat_fwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* ray_rec,
                                              const float* conic_opac, const float* rgb, const float* lnv,
                                              const float* depth, const float* pixel_rays, const uint32_t* vals_sorted,
                                              const uint32_t* tile_ranges, float* image, float* final_T,
                                              uint32_t* n_contrib, float* depth_img, float* alpha_img, void* stream) {
    return ray_fwd_impl(true, cam, cfg, N, ray_rec, conic_opac, rgb, lnv, depth, pixel_rays, vals_sorted, tile_ranges,
                        image, final_T, n_contrib, depth_img, alpha_img, stream);
}

extern "C" int32_t xpr_rasterize_ray_stats(const xpr_camera* cam, const xpr_config* cfg, int64_t N,
                                           const float* ray_rec, const float* conic_opac, const float* rgb,
                                           const float* lnv, const float* pixel_rays, const uint32_t* vals_sorted,
                                           const uint32_t* tile_ranges, uint64_t* stats, void* stream) {
    if (int32_t s = check_ray_cam_cfg(cam, cfg)) return s;
    if (N < 0 || !aligned(tile_ranges, 8) || !aligned(stats, 8) || !aligned(pixel_rays, 4)) return XPR_ERR_INVALID_ARG;
    if (N > 0 && (!aligned(ray_rec, 16) || !aligned(conic_opac, 16) || !aligned(rgb, 4) || !aligned(lnv, 4) ||
                  !aligned(vals_sorted, 4)))
        return XPR_ERR_INVALID_ARG;
    RayRasterParams P;
    make_params(cam, cfg, P);
    const int T = tiles_x(cam) * tiles_y(cam);
    XPR_CUDA(cudaMemsetAsync(stats, 0, 4 * sizeof(uint64_t), (cudaStream_t)stream));
    rasterize_ray_fwd_kernel<true, 1><<<T, BLOCK, 0, (cudaStream_t)stream>>>(
        P, reinterpret_cast<const float4*>(ray_rec), reinterpret_cast<const float4*>(conic_opac), rgb, lnv, pixel_rays,
        vals_sorted, reinterpret_cast<const uint2*>(tile_ranges), nullptr, nullptr, nullptr,
        reinterpret_cast<unsigned long long*>(stats));
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}

static int32_t ray_bwd_impl(bool feat, const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* ray_rec,
                            const float* conic_opac, const float* rgb, const float* lnv, const float* depth,
                            const float* pixel_rays, const uint32_t* vals_sorted, const uint32_t* tile_ranges,
                            const float* final_T, const uint32_t* n_contrib, const float* dL_dimage, const float* dL_ddepth,
                            const float* dL_dalpha, float* g_ray_acc, float* g_opac, float* g_rgb, float* g_depth,
                            int32_t zero_init, void* stream) {
    if (int32_t s = check_ray_cam_cfg(cam, cfg)) return s;
    if (N < 0) return XPR_ERR_INVALID_ARG;
    if (!aligned(tile_ranges, 8) || !aligned(final_T, 4) || !aligned(n_contrib, 4) || !aligned(dL_dimage, 4) ||
        !aligned(pixel_rays, 4))
        return XPR_ERR_INVALID_ARG;
    if (feat && (!aligned(dL_ddepth, 4) || !aligned(dL_dalpha, 4))) return XPR_ERR_INVALID_ARG;
    if (N == 0) return XPR_OK;
    if (!aligned(ray_rec, 16) || !aligned(conic_opac, 16) || !aligned(rgb, 4) || !aligned(lnv, 4) ||
        !aligned(vals_sorted, 4) || !aligned(g_ray_acc, 16) || !aligned(g_opac, 4) || !aligned(g_rgb, 4))
        return XPR_ERR_INVALID_ARG;
    if (feat && (!aligned(depth, 4) || !aligned(g_depth, 4))) return XPR_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    if (zero_init) {
        const size_t n = (size_t)N;
        if (g_opac == g_ray_acc + 16 * n && g_rgb == g_opac + n) {
            const bool with_depth = feat && g_depth == g_rgb + 3 * n;
            XPR_CUDA(cudaMemsetAsync(g_ray_acc, 0, sizeof(float) * (with_depth ? 21 : 20) * n, st));   // one allocation: one fill
            if (feat && !with_depth) XPR_CUDA(cudaMemsetAsync(g_depth, 0, sizeof(float) * n, st));
        } else {
            XPR_CUDA(cudaMemsetAsync(g_ray_acc, 0, sizeof(float) * 16 * n, st));
            XPR_CUDA(cudaMemsetAsync(g_opac, 0, sizeof(float) * n, st));
            XPR_CUDA(cudaMemsetAsync(g_rgb, 0, sizeof(float) * 3 * n, st));
            if (feat) XPR_CUDA(cudaMemsetAsync(g_depth, 0, sizeof(float) * n, st));
        }
    }
    RayRasterParams P;
    make_params(cam, cfg, P);
    const int T = tiles_x(cam) * tiles_y(cam);
#define XPR_RAY_BWD(PPT_, FEAT_)                                                                                    \
    rasterize_ray_bwd_kernel<PPT_, FEAT_><<<T, BLOCK / PPT_, 0, st>>>(                                              \
        P, reinterpret_cast<const float4*>(ray_rec), reinterpret_cast<const float4*>(conic_opac), rgb, lnv, pixel_rays, \
        vals_sorted, reinterpret_cast<const uint2*>(tile_ranges), final_T, n_contrib, dL_dimage, g_ray_acc, g_opac,  \
        g_rgb, depth, dL_ddepth, dL_dalpha, g_depth)
    // more pixels per thread amortise the per-entry reduction (throughput shape); fewer give a heavy tile more warps
    const bool big = T >= XPR_RAY_FWD_PPT2_MIN_TILES;
    if (feat) { if (big) XPR_RAY_BWD(XPR_RAY_BWD_PPT, true); else XPR_RAY_BWD(2, true); }
    else      { if (big) XPR_RAY_BWD(XPR_RAY_BWD_PPT, false); else XPR_RAY_BWD(2, false); }
#undef XPR_RAY_BWD
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}

extern "C" int32_t xpr_rasterize_ray_bwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* ray_rec,
                                         const float* conic_opac, const float* rgb, const float* lnv,
                                         const float* pixel_rays, const uint32_t* vals_sorted,
                                         const uint32_t* tile_ranges, const float* final_T, const uint32_t* n_contrib,
                                         const float* dL_dimage, float* g_ray_acc, float* g_opac, float* g_rgb,
                                         int32_t zero_init, void* stream) {
    return ray_bwd_impl(false, cam, cfg, N, ray_rec, conic_opac, rgb, lnv, nullptr, pixel_rays, vals_sorted, tile_ranges,
                        final_T, n_contrib, dL_dimage, nullptr, nullptr, g_ray_acc, g_opac, g_rgb, nullptr, zero_init, stream);
}

extern "C" int32_t xpr_rasterize_ray_feat_bwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* ray_rec,
                                              const float* conic_opac, const float* rgb, const float* lnv,
                                              const float* depth, const float* pixel_rays, const uint32_t* vals_sorted,
                                              const uint32_t* tile_ranges, const float* final_T,
                                              const uint32_t* n_contrib, const float* dL_dimage, const float* dL_ddepth,
                                              const float* dL_dalpha, float* g_ray_acc, float* g_opac, float* g_rgb,
                                              float* g_depth, int32_t zero_init, void* stream) {
    return ray_bwd_impl(true, cam, cfg, N, ray_rec, conic_opac, rgb, lnv, depth, pixel_rays, vals_sorted, tile_ranges,
                        final_T, n_contrib, dL_dimage, dL_ddepth, dL_dalpha, g_ray_acc, g_opac, g_rgb, g_depth, zero_init,
                        stream);
}
