// rasterize_lin.cu -- xpr_lin_rasterize_fwd: front-to-back compositing of XPR-LinPrim (PAPER A.1.3
// L506-528, Listing 5): octahedra with homogeneous density.  Per (pixel, primitive) the ray's chord through
// the projected octahedron is the intersection of four slab pairs,
//   tau in [m_i - h_i, m_i + h_i],  m_i = -(kx_i dx + ky_i dy),  i = 0..3,
//   dtau = min_i (m_i + h_i) - max_i (m_i - h_i)   if positive,
//   alpha = min(alpha_max, 1 - exp(-sigma dtau))   (Beer-Lambert, L528; clamp, gate and exit as the Gaussian path, reading L5).
// The gate alpha >= alpha_thresh is decided on x = sigma dtau >= -log(1 - alpha_thresh), computed with individually
// rounded fp32 operations in the order of the oracle, never on exp() (rule R3).
// Same structure as rasterize.cu: one CTA per 16x16 tile, the 80-byte records of the tile's list gathered by cp.async
// through a three-stage ring, one barrier per batch, warp-broadcast LDS.128 reads.
#include "common.cuh"
#include "packed.cuh"

namespace xpr {
namespace {

constexpr int BLOCK = TILE * TILE;
constexpr int STAGES = 3;
constexpr int BATCH = 128;
constexpr int REC4 = 5;               // float4 per record: (mx, my, sigma, depth | kx0 ky0 h0 kx1 | ky1 h1 kx2 ky2 | h2 kx3 ky3 h3 | r g b -)

struct LinParams {
    int W, H, TW;
    float amax, tmin, req;
    float bg[3];
    const uint32_t* order;
};

__device__ __forceinline__ void stage_lin(float4* slot, const float4* __restrict__ rec, uint32_t g) {
    const float4* src = rec + REC4 * (size_t)g;
#pragma unroll
    for (int k = 0; k < REC4; ++k) cp_async16(slot + k, src + k);
}

// x = sigma dtau of one pixel for the record at rq (0 when the ray misses)
__device__ __forceinline__ float lin_chord(const float4* rq, float pxc, float pyc) {
    const float4 a = rq[0], b = rq[1], c = rq[2], d = rq[3];
    const float dx = __fsub_rn(pxc, a.x), dy = __fsub_rn(pyc, a.y);
    const float m0 = -__fmaf_rn(b.x, dx, __fmul_rn(b.y, dy)), m1 = -__fmaf_rn(b.w, dx, __fmul_rn(c.x, dy));
    const float m2 = -__fmaf_rn(c.z, dx, __fmul_rn(c.w, dy)), m3 = -__fmaf_rn(d.y, dx, __fmul_rn(d.z, dy));
    const float enter = fmaxf(fmaxf(__fsub_rn(m0, b.z), __fsub_rn(m1, c.y)), fmaxf(__fsub_rn(m2, d.x), __fsub_rn(m3, d.w)));
    const float exit = fminf(fminf(__fadd_rn(m0, b.z), __fadd_rn(m1, c.y)), fminf(__fadd_rn(m2, d.x), __fadd_rn(m3, d.w)));
    return (enter < exit) ? __fmul_rn(a.z, __fsub_rn(exit, enter)) : 0.0f;
}

// STATS: counts {visited, passed the gate, blended, sum of n_contrib} instead of writing an image
template <bool STATS>
__global__ void __launch_bounds__(BLOCK)
lin_rasterize_fwd_kernel(LinParams P, const float4* __restrict__ rec, const uint32_t* __restrict__ vals,
                         const uint2* __restrict__ ranges, float* __restrict__ image, float* __restrict__ final_T,
                         uint32_t* __restrict__ n_contrib, unsigned long long* __restrict__ stats) {
    constexpr int B = BATCH;                  // records per batch, staged by the first B threads (3 x 128 x 80 B = 30 KB)
    __shared__ float4 s_rec[STAGES][REC4 * B];
    const int tid = threadIdx.x;
    const int tile = P.order ? (int)P.order[blockIdx.x] : (int)blockIdx.x;
    const int tx = tile % P.TW, ty = tile / P.TW;
    const int px = tx * TILE + (tid % TILE), py = ty * TILE + (tid / TILE);
    const bool inside = (px < P.W) && (py < P.H);
    const float pxc = (float)px + 0.5f, pyc = (float)py + 0.5f;
    const uint2 rg = ranges[tile];
    const uint32_t len = rg.y - rg.x;
    const uint32_t* const list = vals + rg.x;
    float T = 1.0f, C0 = 0.0f, C1 = 0.0f, C2 = 0.0f;
    uint32_t last = 0, n_visit = 0, n_pass = 0, n_blend = 0;
    bool act = inside;
    const bool stager = tid < B;
    {
        uint32_t g0 = 0, g1 = 0;
        const bool s0 = stager && (uint32_t)tid < len, s1 = stager && (uint32_t)(B + tid) < len;
        if (s0) g0 = list[tid];
        if (s1) g1 = list[B + tid];
        if (s0) stage_lin(&s_rec[0][REC4 * tid], rec, g0);
        cp_async_commit();
        if (s1) stage_lin(&s_rec[1][REC4 * tid], rec, g1);
        cp_async_commit();
    }
    uint32_t g_next = (stager && (uint32_t)(2 * B + tid) < len) ? list[2 * B + tid] : 0u;
    uint32_t stage = 0;
    for (uint32_t base = 0; base < len; base += B) {
        cp_async_wait<1>();
        if (__syncthreads_or(act) == 0) break;
        {
            const uint32_t s2 = (stage + 2 >= STAGES) ? stage + 2 - STAGES : stage + 2;
            if (stager && base + 2 * B + tid < len) stage_lin(&s_rec[s2][REC4 * tid], rec, g_next);
            cp_async_commit();
            g_next = (stager && base + 3 * B + tid < len) ? list[base + 3 * B + tid] : 0u;
        }
        const uint32_t cnt = min((uint32_t)B, len - base);
        if (act) {
            const float4* rq = s_rec[stage];
            for (uint32_t j = 0; j < cnt && act; ++j, rq += REC4) {
                const float x = lin_chord(rq, pxc, pyc);
                if (STATS) ++n_visit;
                if (!(x >= P.req)) continue;                       // alpha < alpha_thresh, decided on sigma dtau
                if (STATS) ++n_pass;
                const float alpha = fminf(P.amax, 1.0f - ex2_approx(-x * LOG2E));
                const float Tn = T * (1.0f - alpha);
                if (Tn < P.tmin) { act = false; break; }            // C12: stop without blending
                const float4 col = rq[4];
                const float w = alpha * T;
                C0 = fmaf(col.x, w, C0); C1 = fmaf(col.y, w, C1); C2 = fmaf(col.z, w, C2);
                T = Tn;
                last = base + j + 1;
                if (STATS) ++n_blend;
            }
        }
        stage = (stage + 1 == STAGES) ? 0 : stage + 1;
    }
    cp_async_wait<0>();
    if (STATS) {
        atomicAdd(stats + 0, (unsigned long long)n_visit); atomicAdd(stats + 1, (unsigned long long)n_pass);
        atomicAdd(stats + 2, (unsigned long long)n_blend); atomicAdd(stats + 3, (unsigned long long)last);
        return;
    }
    if (inside) {
        const int64_t pid = (int64_t)py * P.W + px;
        image[3 * pid] = fmaf(T, P.bg[0], C0);
        image[3 * pid + 1] = fmaf(T, P.bg[1], C1);
        image[3 * pid + 2] = fmaf(T, P.bg[2], C2);
        final_T[pid] = T;
        n_contrib[pid] = last;
    }
}

// Backward compositing of LinPrim (f4; derivative of the loop above, the paper relies on AD, L106).  One CTA of 128
// threads per tile, a thread owns two consecutive pixels of a row; the list is walked back to front from the deepest
// n_contrib of the tile, T_k = T_{k+1} / (1 - alpha_k) restored on the way, with the one running scalar R = -g . S_k as in
// rasterize.cu.  Per (pixel, primitive), with G = dL/dx = exp(-x) dL/dalpha (0 when the clamp is active, C14) and the
// slab pairs en / ex the ray enters / leaves through (first index on ties, as the oracle):
//   dL/dsigma += dtau G;   gm = sigma G:   dL/dh_ex += gm, dL/dh_en += gm,
//   dL/dkx_ex -= dx gm, dL/dkx_en += dx gm (ky with dy),   dL/dmu2D += gm ((kx, ky)_ex - (kx, ky)_en).
// The 18 sums of a primitive are reduced over the warp by three transposed butterflies and added to g_lin_rec[N,20]
// (record layout, slots 3 and 19 unused) with one RED per value and warp.
__global__ void __launch_bounds__(BATCH)
lin_rasterize_bwd_kernel(LinParams P, const float4* __restrict__ rec, const uint32_t* __restrict__ vals,
                         const uint2* __restrict__ ranges, const float* __restrict__ final_T,
                         const uint32_t* __restrict__ n_contrib, const float* __restrict__ dL, float* __restrict__ g_rec) {
    constexpr int B = BATCH, THREADS = BATCH, PPT = 2;
    __shared__ float4 s_rec[STAGES][REC4 * B];
    __shared__ uint32_t s_idx[STAGES][B];
    __shared__ uint32_t s_max[THREADS / 32];
    const int tid = threadIdx.x, lane = tid & 31;
    const int tile = P.order ? (int)P.order[blockIdx.x] : (int)blockIdx.x;
    const int tx = tile % P.TW, ty = tile / P.TW;
    constexpr int TPR = TILE / PPT;
    const int px0 = tx * TILE + (tid % TPR) * PPT, py = ty * TILE + (tid / TPR);
    const float pyc = (float)py + 0.5f;
    const uint2 rg = ranges[tile];
    const uint32_t* const list = vals + rg.x;
    uint32_t n[PPT], wmax = 0;
    float T[PPT], R[PPT], g0[PPT], g1[PPT], g2[PPT], pxc[PPT];
#pragma unroll
    for (int h = 0; h < PPT; ++h) {
        const int px = px0 + h;
        n[h] = 0; T[h] = 0.0f; g0[h] = g1[h] = g2[h] = 0.0f;
        pxc[h] = (float)px + 0.5f;
        if (px < P.W && py < P.H) {
            const int64_t pid = (int64_t)py * P.W + px;
            n[h] = n_contrib[pid]; T[h] = final_T[pid];
            g0[h] = dL[3 * pid]; g1[h] = dL[3 * pid + 1]; g2[h] = dL[3 * pid + 2];
        }
        R[h] = -T[h] * fmaf(g2[h], P.bg[2], fmaf(g1[h], P.bg[1], g0[h] * P.bg[0]));
        wmax = max(wmax, n[h]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) wmax = max(wmax, __shfl_xor_sync(0xffffffffu, wmax, o));
    if (lane == 0) s_max[tid >> 5] = wmax;
    __syncthreads();
    uint32_t max_n = 0;
#pragma unroll
    for (int w = 0; w < THREADS / 32; ++w) max_n = max(max_n, s_max[w]);

    auto stage_entry = [&](uint32_t s, uint32_t g) {
        s_idx[s][tid] = g;
        stage_lin(&s_rec[s][REC4 * tid], rec, g);
    };
    {
        uint32_t e0 = 0, e1 = 0;
        if ((uint32_t)tid < max_n) e0 = list[max_n - 1u - (uint32_t)tid];
        if ((uint32_t)(B + tid) < max_n) e1 = list[max_n - 1u - (uint32_t)(B + tid)];
        if ((uint32_t)tid < max_n) stage_entry(0, e0);
        cp_async_commit();
        if ((uint32_t)(B + tid) < max_n) stage_entry(1, e1);
        cp_async_commit();
    }
    uint32_t g_next = ((uint32_t)(2 * B + tid) < max_n) ? list[max_n - 1u - (uint32_t)(2 * B + tid)] : 0u;
    // lane 4 i owns value i of a butterfly; record slots of the three groups
    const int vi = lane >> 2;
    const int slotA = (vi < 3) ? vi : (vi < 6) ? 13 + vi : vi - 2;      // mx my sigma | r g b | kx0 ky0
    const int slotB = 6 + vi;                                           // h0 kx1 ky1 h1 kx2 ky2 h2 kx3
    const int slotC = 14 + vi;                                          // ky3 h3 (vi < 2)
    const bool red_lane = (lane & 3) == 0;
    const float amax = P.amax, req = P.req;
    uint32_t stage = 0;
    for (uint32_t base = 0; base < max_n; base += B) {
        cp_async_wait<1>();
        __syncthreads();
        {
            const uint32_t s2 = (stage + 2 >= STAGES) ? stage + 2 - STAGES : stage + 2;
            if (base + 2 * B + tid < max_n) stage_entry(s2, g_next);
            cp_async_commit();
            g_next = (base + 3 * B + tid < max_n) ? list[max_n - 1u - (base + 3 * B + tid)] : 0u;
        }
        const uint32_t cnt = min((uint32_t)B, max_n - base);
        const float4* rq = s_rec[stage];
        for (uint32_t j = 0; j < cnt; ++j, rq += REC4) {
            const uint32_t pos = max_n - 1u - (base + j);
            if (pos >= wmax) continue;                 // warp-uniform
            const float4 a = rq[0], b = rq[1], c = rq[2], d = rq[3];
            const float kx[4] = {b.x, b.w, c.z, d.y}, ky[4] = {b.y, c.x, c.w, d.z}, hh[4] = {b.z, c.y, d.x, d.w};
            const float dy = __fsub_rn(pyc, a.y);
            float xs[PPT], dxs[PPT], dts[PPT];
            int ien[PPT], iex[PPT];
            bool con[PPT], any_c = false;
#pragma unroll
            for (int h = 0; h < PPT; ++h) {
                const float dx = __fsub_rn(pxc[h], a.x);
                float en = -INFINITY, ex = INFINITY;
                int ie = 0, ix = 0;
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const float m = -__fmaf_rn(kx[i], dx, __fmul_rn(ky[i], dy));
                    const float lo = __fsub_rn(m, hh[i]), hi = __fadd_rn(m, hh[i]);
                    if (lo > en) { en = lo; ie = i; }
                    if (hi < ex) { ex = hi; ix = i; }
                }
                const float dt = __fsub_rn(ex, en);
                const float x = (en < ex) ? __fmul_rn(a.z, dt) : 0.0f;
                xs[h] = x; dxs[h] = dx; dts[h] = dt; ien[h] = ie; iex[h] = ix;
                con[h] = (pos < n[h]) && (x >= req);
                any_c |= con[h];
            }
            if (!__any_sync(0xffffffffu, any_c)) continue;
            const float4 col = rq[4];
            float vA[8], vB[8], vC[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) vA[k] = vB[k] = vC[k] = 0.0f;
#pragma unroll
            for (int h = 0; h < PPT; ++h) {
                const float ea = con[h] ? ex2_approx(-xs[h] * LOG2E) : 1.0f;      // exp(-x) = 1 - a
                const float av = 1.0f - ea;
                const float al = fminf(amax, av);
                const float inv = rcp_approx(1.0f - al);
                T[h] *= inv;                                                      // transmittance in front of this entry
                const float w = al * T[h];
                vA[3] = fmaf(w, g0[h], vA[3]); vA[4] = fmaf(w, g1[h], vA[4]); vA[5] = fmaf(w, g2[h], vA[5]);
                const float gc = fmaf(g2[h], col.z, fmaf(g1[h], col.y, g0[h] * col.x));
                const float da = fmaf(inv, R[h], T[h] * gc);                      // dL/dalpha = T (g . c) - Q / (1 - alpha)
                R[h] = fmaf(-gc, w, R[h]);
                const float G = (con[h] && av < amax) ? ea * da : 0.0f;           // dL/dx (C14)
                const float gm = a.z * G;
                vA[2] = fmaf((G != 0.0f) ? dts[h] : 0.0f, G, vA[2]);          // (a miss has dtau = -inf)
                const float gx = dxs[h] * gm, gy = dy * gm;
                float skx[4], sky[4], sh_[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const float se = (float)((int)(ien[h] == i) - (int)(iex[h] == i));    // +1 entering, -1 leaving
                    const float sb = (float)((int)(ien[h] == i) + (int)(iex[h] == i));
                    skx[i] = se * gx; sky[i] = se * gy; sh_[i] = sb * gm;
                    vA[0] = fmaf(-se * kx[i], gm, vA[0]); vA[1] = fmaf(-se * ky[i], gm, vA[1]);
                }
                vA[6] += skx[0]; vA[7] += sky[0]; vB[0] += sh_[0];
                vB[1] += skx[1]; vB[2] += sky[1]; vB[3] += sh_[1];
                vB[4] += skx[2]; vB[5] += sky[2]; vB[6] += sh_[2];
                vB[7] += skx[3]; vC[0] += sky[3]; vC[1] += sh_[3];
            }
            const float tA = warp_reduce8(vA, lane), tB = warp_reduce8(vB, lane), tC = warp_reduce8(vC, lane);
            float* const gp = g_rec + 20 * (size_t)s_idx[stage][j];
            if (red_lane) {
                if (tA != 0.0f) atomicAdd(gp + slotA, tA);
                if (tB != 0.0f) atomicAdd(gp + slotB, tB);
                if (vi < 2 && tC != 0.0f) atomicAdd(gp + slotC, tC);
            }
        }
        stage = (stage + 1 == STAGES) ? 0 : stage + 1;
    }
    cp_async_wait<0>();
}

int32_t make_lin_params(const xpr_camera* cam, const xpr_config* cfg, LinParams& P) {
    if (!cam || !cfg) return XPR_ERR_INVALID_ARG;
    if (cam->width <= 0 || cam->height <= 0) return XPR_ERR_INVALID_ARG;
    if (cfg->tile != TILE) return XPR_ERR_UNSUPPORTED;
    if (cfg->views > 1 || cam->model != 0) return XPR_ERR_UNSUPPORTED;
    P.W = cam->width; P.H = cam->height; P.TW = tiles_x(cam);
    P.amax = cfg->alpha_max; P.tmin = cfg->t_min;
    P.req = (float)(-log(1.0 - (double)cfg->alpha_thresh));      // R2
    for (int i = 0; i < 3; ++i) P.bg[i] = cfg->bg[i];
    P.order = cfg->tile_order;
    return XPR_OK;
}

}  // namespace
}  // namespace xpr

using namespace xpr;

extern "C" int32_t xpr_lin_rasterize_fwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* lin_rec,
                                         const uint32_t* vals_sorted, const uint32_t* tile_ranges, float* image,
                                         float* final_T, uint32_t* n_contrib, void* stream) {
    LinParams P;
    if (int32_t s = make_lin_params(cam, cfg, P)) return s;
    if (N < 0) return XPR_ERR_INVALID_ARG;
    if (!aligned(tile_ranges, 8) || !aligned(image, 4) || !aligned(final_T, 4) || !aligned(n_contrib, 4))
        return XPR_ERR_INVALID_ARG;
    if (N > 0 && (!aligned(lin_rec, 16) || !aligned(vals_sorted, 4))) return XPR_ERR_INVALID_ARG;
    const int T = tiles_x(cam) * tiles_y(cam);
    lin_rasterize_fwd_kernel<false><<<T, BLOCK, 0, (cudaStream_t)stream>>>(
        P, reinterpret_cast<const float4*>(lin_rec), vals_sorted, reinterpret_cast<const uint2*>(tile_ranges), image, final_T,
        n_contrib, nullptr);
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}

extern "C" int32_t xpr_lin_rasterize_stats(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* lin_rec,
                                           const uint32_t* vals_sorted, const uint32_t* tile_ranges, uint64_t* stats,
                                           void* stream) {
    LinParams P;
    if (int32_t s = make_lin_params(cam, cfg, P)) return s;
    if (N < 0 || !aligned(tile_ranges, 8) || !aligned(stats, 8)) return XPR_ERR_INVALID_ARG;
    if (N > 0 && (!aligned(lin_rec, 16) || !aligned(vals_sorted, 4))) return XPR_ERR_INVALID_ARG;
    const int T = tiles_x(cam) * tiles_y(cam);
    XPR_CUDA(cudaMemsetAsync(stats, 0, 4 * sizeof(uint64_t), (cudaStream_t)stream));
    lin_rasterize_fwd_kernel<true><<<T, BLOCK, 0, (cudaStream_t)stream>>>(
        P, reinterpret_cast<const float4*>(lin_rec), vals_sorted, reinterpret_cast<const uint2*>(tile_ranges), nullptr, nullptr,
        nullptr, reinterpret_cast<unsigned long long*>(stats));
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}

extern "C" int32_t xpr_lin_rasterize_bwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* lin_rec,
                                         const uint32_t* vals_sorted, const uint32_t* tile_ranges, const float* final_T,
                                         const uint32_t* n_contrib, const float* dL_dimage, float* g_lin_rec, void* stream) {
    LinParams P;
    if (int32_t s = make_lin_params(cam, cfg, P)) return s;
    if (N < 0) return XPR_ERR_INVALID_ARG;
    if (!aligned(tile_ranges, 8) || !aligned(final_T, 4) || !aligned(n_contrib, 4) || !aligned(dL_dimage, 4))
        return XPR_ERR_INVALID_ARG;
    if (N == 0) return XPR_OK;
    if (!aligned(lin_rec, 16) || !aligned(vals_sorted, 4) || !aligned(g_lin_rec, 16)) return XPR_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    XPR_CUDA(cudaMemsetAsync(g_lin_rec, 0, (size_t)N * 20 * sizeof(float), st));
    const int T = tiles_x(cam) * tiles_y(cam);
    lin_rasterize_bwd_kernel<<<T, BATCH, 0, st>>>(P, reinterpret_cast<const float4*>(lin_rec), vals_sorted,
                                                  reinterpret_cast<const uint2*>(tile_ranges), final_T, n_contrib, dL_dimage,
                                                  g_lin_rec);
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}
