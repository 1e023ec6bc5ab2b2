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
