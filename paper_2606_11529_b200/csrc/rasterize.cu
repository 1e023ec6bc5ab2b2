// rasterize.cu -- xpr_rasterize_fwd / xpr_rasterize_bwd (+ the depth / accumulated-opacity variants
// xpr_rasterize_feat_fwd / _bwd): per-tile front-to-back alpha compositing (Algorithm 1,
// Listing 1) and its reverse-mode pass.
//
// One CTA per 16x16 tile.  The tile's list vals_sorted[start..end) is a list of Gaussian indices; the shader
// data p_sd of a Gaussian is one 48-byte record shade_rec[g] = 3 x float4
//     (mx, my, qa, qb | qc, lnv, log2 o, z | r, g, b, o),   qa = -A/2, qb = -B, qc = -C/2   (C25),
// written by xpr_project.  Batches of records are gathered into shared memory with cp.async (16-byte LDGSTS, no
// register staging) through a three-stage ring: while batch b is walked, the copies of batches b+1 and b+2 are
// in flight and the list indices of batch b+3 are being loaded, so a CTA waits for memory only at its start and
// there is one barrier per batch.  Every thread walks the batch with warp-broadcast LDS.128 reads.
// Decisions (the power > 0 guard and the alpha gate) are taken on `power`, computed in the fixed fp32 order of
// rule R3 (carried negated: `gate`), never on exp().  A thread owns 2 (forward) or 8 (backward) pixels of one tile row and works on them
// as PAIRS with the packed fp32 instructions of sm_100 (fma.rn.f32x2 -> FFMA2 ...: two individually rounded
// results per issue slot -- the kernels are issue-bound), packed.cuh.
#include "common.cuh"
#include "packed.cuh"

namespace xpr {
namespace {

constexpr int BLOCK = TILE * TILE;   // 256 pixels
constexpr int STAGES = 3;            // cp.async ring depth

struct RasterParams {
    int W, H, TW;
    int T;                   // tiles per view: tile index b of a batch of views is view b / T, tile b % T of that view
    float amax, tmin;
    float bg[3];
    const uint32_t* order;   // xpr_config.tile_order: CTA b works on tile order[b] (longest lists first), or NULL
    int vec;                 // backward: W % 4 == 0 and the per-pixel arrays are 16-byte aligned (128-bit prologue loads)
};

// Both gates of a list entry on m = -power: valid (power <= 0, L289) and alpha >= alpha_thresh (power >= -lnv, L679)
// <=> 0 <= m <= lnv <=> bits(m) <= bits(lnv) as unsigned integers, for lnv > 0 (xpr_project culls a Gaussian with
// lnv <= 0: its extent is empty).  m < 0 has the sign bit set and compares above every positive float.
__device__ __forceinline__ bool gate(float m, uint32_t lnv_bits) { return __float_as_uint(m) <= lnv_bits; }

// gather one record (3 x 16 bytes) into a ring slot
__device__ __forceinline__ void stage_record(float4* slot, const float4* __restrict__ rec, uint32_t g) {
    const float4* src = rec + 3 * (size_t)g;
    cp_async16(slot, src);
    cp_async16(slot + 1, src + 1);
    cp_async16(slot + 2, src + 2);
}

// Forward compositing (a8).  One CTA per 16x16 tile, in two shapes:
//   PPT = 2: 128 threads, a thread owns the two pixels (x, y) and (x + 8, y) of one row, so the row terms
//            of `power` (dy, qb*dy, (qc*dy)*dy) and the shared-memory reads of a list entry are paid once
//            per two pixels, and the pixel pair shares packed instructions (throughput shape, large images);
//   PPT = 1: 256 threads, one pixel each -- twice the warps on a tile, i.e. half the critical path of a
//            heavy tile (latency shape, images with few tiles where the longest list bounds the kernel).
// The arithmetic per pixel is exactly power = fma(fma(qa, dx, qb*dy), dx, (qc*dy)*dy) (rule R3) in both.
// BF (lists produced with tile_cull: > 90 % of the visited pairs pass the gate): branch-free blend -- a pixel
//   that is done or gated enters with alpha = 0, so T' = T >= t_min and w = 0; otherwise gated pairs are branched over.
// STATS = true: the same walk, additionally counting pixel-pair events into stats[0..3] =
//   {visited, passed both gates, blended, sum of n_contrib} (xpr_rasterize_stats; roofline accounting).
// FEAT = true (xpr_rasterize_feat_fwd, reading C31): the same walk also blends the depth image
//   D = sum z alpha T and the accumulated opacity A = sum alpha T; z rides in the record.
#ifndef XPR_FWD_PPT2_MIN_TILES
#define XPR_FWD_PPT2_MIN_TILES 4096
#endif
constexpr int FWD_PPT2_MIN_TILES = XPR_FWD_PPT2_MIN_TILES;

#ifndef XPR_FWD_MINB
#define XPR_FWD_MINB 1
#endif
template <bool STATS, int PPT, bool BF, bool FEAT>
__global__ void __launch_bounds__(BLOCK / PPT, (PPT == 2 && BF) ? XPR_FWD_MINB : 0)
rasterize_fwd_kernel(RasterParams P, const float4* __restrict__ rec, const uint32_t* __restrict__ vals,
                     const uint2* __restrict__ ranges, float* __restrict__ image, float* __restrict__ final_T,
                     uint32_t* __restrict__ n_contrib, unsigned long long* __restrict__ stats,
                     float* __restrict__ depth_img, float* __restrict__ alpha_img) {
    constexpr int THREADS = BLOCK / PPT, B = THREADS, ROW = TILE / PPT;
    constexpr bool PACKED = BF && (PPT == 2);
    __shared__ float4 s_rec[STAGES][3 * B];
    const int tid = threadIdx.x;
    const int tile = P.order ? (int)P.order[blockIdx.x] : (int)blockIdx.x;
    const int view = tile / P.T, vt = tile - view * P.T;       // batch of views: the images are stacked, [V, H, W, .]
    const int64_t vbase = (int64_t)view * P.H * P.W;
    const int tx = vt % P.TW, ty = vt / P.TW;
    const int px0 = tx * TILE + (tid % ROW), px1 = px0 + 8, py = ty * TILE + (tid / ROW);
    const bool in0 = (px0 < P.W) && (py < P.H), in1 = (PPT == 2) && (px1 < P.W) && (py < P.H);
    const float pxc0 = (float)px0 + 0.5f, pxc1 = (float)px1 + 0.5f, pyc = (float)py + 0.5f;
    const f32x2 px2 = pack2(pxc0, pxc1);
    const uint2 rg = ranges[tile];
    const uint32_t len = rg.y - rg.x;
    const uint32_t* const list = vals + rg.x;

    // pixel state: scalar (branchy shapes) or packed pairs (lane 0 = pixel a, lane 1 = pixel b)
    float Ta = 1.0f, Ca0 = 0.0f, Ca1 = 0.0f, Ca2 = 0.0f, Tb = 1.0f, Cb0 = 0.0f, Cb1 = 0.0f, Cb2 = 0.0f;
    float Da = 0.0f, Aa = 0.0f, Db = 0.0f, Ab = 0.0f;
    f32x2 T2 = pack2(1.0f, 1.0f), C0_2 = 0ull, C1_2 = 0ull, C2_2 = 0ull, D2 = 0ull, A2 = 0ull;
    uint32_t last_a = 0, last_b = 0;
    bool act_a = in0, act_b = in1;                            // still compositing
    uint32_t n_visit = 0, n_pass = 0, n_blend = 0;
    float amax = P.amax, tmin = P.tmin;
    asm volatile("" : "+f"(amax), "+f"(tmin));     // keep both in registers (else re-read from the constant bank per entry)

    // ---- staging ring: batches 0 and 1 on their way, indices of batch 2 loading -------------------------------
    {
        uint32_t g0 = 0, g1 = 0;
        if ((uint32_t)tid < len) g0 = list[tid];
        if ((uint32_t)(B + tid) < len) g1 = list[B + tid];
        if ((uint32_t)tid < len) stage_record(&s_rec[0][3 * tid], rec, g0);
        cp_async_commit();
        if ((uint32_t)(B + tid) < len) stage_record(&s_rec[1][3 * tid], rec, g1);
        cp_async_commit();
    }
    uint32_t g_next = ((uint32_t)(2 * B + tid) < len) ? list[2 * B + tid] : 0u;   // index of this thread's entry of batch b + 2

    float pw_a[4], pw_b[4], l2o[4], zz[4];          // pw: MINUS power (see `power` below)
    uint32_t lim[4];                                // bits of lnv: the gate's upper limit
    f32x2 pw2[4];
    float4 col[4];                                             // colours of the group's entries (BF)
    uint32_t stage = 0;
    for (uint32_t base = 0; base < len; base += B) {
        cp_async_wait<1>();                                    // this thread's copies of batch b have landed
        if (__syncthreads_or(act_a || act_b) == 0) break;      // ... everyone's; and everyone is done with batch b - 1
        {   // batch b + 2 goes into the slot batch b - 1 just left; then the indices of batch b + 3 start loading
            const uint32_t s2 = (stage + 2 >= STAGES) ? stage + 2 - STAGES : stage + 2;
            if (base + 2 * B + tid < len) stage_record(&s_rec[s2][3 * tid], rec, g_next);
            cp_async_commit();
            g_next = (base + 3 * B + tid < len) ? list[base + 3 * B + tid] : 0u;
        }
        const uint32_t cnt = min((uint32_t)B, len - base);
        // The list is walked in groups of 4 entries.  Phase 1 of a group computes the 4 (x PPT) values of
        // `power` -- independent of each other and of the transmittance, so their latencies overlap -- and
        // phase 2 runs the sequential part (gate, alpha, T' = T (1 - alpha), exit test, blend).
        auto power = [&](int u, const float4* rq) {
            const float4 ge = rq[0];
            const float4 ga = rq[1];
            const float dy = pyc - ge.y;
            // the kernel carries -power: every operand negated, every rounding symmetric, so the bits are those of
            // rule R3's power with the sign flipped -- and both gates become ONE unsigned compare (below)
            const float t1 = __fmul_rn(-ge.w, dy), t2 = __fmul_rn(__fmul_rn(-ga.x, dy), dy);
            if (PPT == 2) {
                const f32x2 dx2 = sub2(px2, bcast2(ge.x));
                pw2[u] = fma2(fma2(bcast2(-ge.z), dx2, bcast2(t1)), dx2, bcast2(t2));
                if (!PACKED) unpack2(pw2[u], pw_a[u], pw_b[u]);
            } else {
                const float dxa = pxc0 - ge.x;
                pw_a[u] = __fmaf_rn(__fmaf_rn(-ge.z, dxa, t1), dxa, t2);
            }
            lim[u] = __float_as_uint(ga.y); l2o[u] = ga.z;
            if (FEAT) zz[u] = ga.w;
            if (BF) col[u] = rq[2];
        };
        // valid = power <= 0 (L289, C20); alpha >= alpha_thresh <=> power >= -lnv (L679, C12): with m = -power both
        // read 0 <= m <= lnv, and for lnv > 0 (every visible Gaussian) that is bits(m) <= bits(lnv) as unsigned integers
        // (a negative m has the sign bit set and compares above any positive float; m = +0 when power = -0)
        auto blend_packed = [&](int u, uint32_t pos) {
            float pa, pb;
            unpack2(pw2[u], pa, pb);
            const bool pass_a = act_a && gate(pa, lim[u]);
            const bool pass_b = act_b && gate(pb, lim[u]);
            float ea, eb;                                       // o exp(power) = ex2(power log2 e + log2 o)
            unpack2(fma2(pw2[u], bcast2(-LOG2E), bcast2(l2o[u])), ea, eb);
            // a gated or finished pixel gets alpha = 0 (SASS: a predicated MUFU.EX2 over a zeroed register pair; selecting
            // the exponent, ex2(-inf) = 0, measured 1.2 % slower)
            const float al_a = fminf(amax, pass_a ? ex2_approx(ea) : 0.0f);           // C11
            const float al_b = fminf(amax, pass_b ? ex2_approx(eb) : 0.0f);
            const f32x2 al2 = pack2(al_a, al_b);
            float tn_a, tn_b, w_a, w_b, t_a, t_b;
            unpack2(mul2(T2, sub2(bcast2(1.0f), al2)), tn_a, tn_b);             // T' = T (1 - alpha)
            unpack2(mul2(al2, T2), w_a, w_b);
            unpack2(T2, t_a, t_b);
            act_a = act_a && !(tn_a < tmin);                    // C12: stop without blending
            act_b = act_b && !(tn_b < tmin);
            // a pixel that was done or gated has alpha = 0: w = 0 and T' = T already; only the stopping entry needs the select
            // (measured: zeroing alpha instead and recomputing w, T' with two more packed products is 3 % slower)
            const f32x2 w2 = pack2(act_a ? w_a : 0.0f, act_b ? w_b : 0.0f);
            T2 = pack2(act_a ? tn_a : t_a, act_b ? tn_b : t_b);
            C0_2 = fma2(bcast2(col[u].x), w2, C0_2);
            C1_2 = fma2(bcast2(col[u].y), w2, C1_2);
            C2_2 = fma2(bcast2(col[u].z), w2, C2_2);
            if (FEAT) { D2 = fma2(bcast2(zz[u]), w2, D2); A2 = add2(A2, w2); }
            last_a = (pass_a && act_a) ? pos : last_a;
            last_b = (pass_b && act_b) ? pos : last_b;
        };
        auto blend_scalar = [&](bool& act, float pw, int u, const float4* rq, float& T, float& C0, float& C1, float& C2,
                                uint32_t& last, uint32_t pos, float& Dv, float& Av) {
            if (BF) {
                const bool pass = act && gate(pw, lim[u]);
                const float alpha = pass ? fminf(amax, ex2_approx(fmaf(pw, -LOG2E, l2o[u]))) : 0.0f;
                const float Tn = T * (1.0f - alpha);
                const bool stop = Tn < tmin;
                const bool bl = pass && !stop;
                act = act && !stop;
                const float w = bl ? alpha * T : 0.0f;
                C0 = fmaf(col[u].x, w, C0); C1 = fmaf(col[u].y, w, C1); C2 = fmaf(col[u].z, w, C2);
                if (FEAT) { Dv = fmaf(zz[u], w, Dv); Av += w; }
                T = bl ? Tn : T;
                last = bl ? pos : last;
            } else if (act) {
                if (STATS) ++n_visit;
                if (gate(pw, lim[u])) {
                    if (STATS) ++n_pass;
                    const float alpha = fminf(amax, ex2_approx(fmaf(pw, -LOG2E, l2o[u])));
                    const float Tn = T * (1.0f - alpha);
                    if (Tn < tmin) {
                        act = false;
                    } else {
                        const float4 c = rq[2];
                        const float w = alpha * T;
                        C0 = fmaf(c.x, w, C0); C1 = fmaf(c.y, w, C1); C2 = fmaf(c.z, w, C2);
                        if (FEAT) { Dv = fmaf(zz[u], w, Dv); Av += w; }
                        T = Tn;
                        last = pos;
                        if (STATS) ++n_blend;
                    }
                }
            }
        };
        auto step = [&](int u, const float4* rq, uint32_t pos) {
            if (PACKED) {
                blend_packed(u, pos);
            } else {
                blend_scalar(act_a, pw_a[u], u, rq, Ta, Ca0, Ca1, Ca2, last_a, pos, Da, Aa);
                if (PPT == 2) blend_scalar(act_b, pw_b[u], u, rq, Tb, Cb0, Cb1, Cb2, last_b, pos, Db, Ab);
            }
        };
        if (act_a || act_b) {
            const float4* rq = s_rec[stage];
            uint32_t j = 0;
            for (; j + 4 <= cnt && (act_a || act_b); j += 4, rq += 12) {
                power(0, rq); power(1, rq + 3); power(2, rq + 6); power(3, rq + 9);
                step(0, rq, base + j + 1);
                step(1, rq + 3, base + j + 2);
                step(2, rq + 6, base + j + 3);
                step(3, rq + 9, base + j + 4);
            }
            for (; j < cnt && (act_a || act_b); ++j, rq += 3) {
                power(0, rq);
                step(0, rq, base + j + 1);
            }
        }
        stage = (stage + 1 == STAGES) ? 0 : stage + 1;
    }
    cp_async_wait<0>();
    if (PACKED) {
        unpack2(T2, Ta, Tb);
        unpack2(C0_2, Ca0, Cb0); unpack2(C1_2, Ca1, Cb1); unpack2(C2_2, Ca2, Cb2);
        if (FEAT) { unpack2(D2, Da, Db); unpack2(A2, Aa, Ab); }
    }
    if (STATS) {
        atomicAdd(stats + 0, (unsigned long long)n_visit); atomicAdd(stats + 1, (unsigned long long)n_pass);
        atomicAdd(stats + 2, (unsigned long long)n_blend); atomicAdd(stats + 3, (unsigned long long)(last_a + last_b));
        return;
    }
    if (in0) {
        const int64_t pid = vbase + (int64_t)py * P.W + px0;
        image[3 * pid] = fmaf(Ta, P.bg[0], Ca0);
        image[3 * pid + 1] = fmaf(Ta, P.bg[1], Ca1);
        image[3 * pid + 2] = fmaf(Ta, P.bg[2], Ca2);
        final_T[pid] = Ta;
        n_contrib[pid] = last_a;
        if (FEAT) { depth_img[pid] = Da; alpha_img[pid] = Aa; }
    }
    if (in1) {
        const int64_t pid = vbase + (int64_t)py * P.W + px1;
        image[3 * pid] = fmaf(Tb, P.bg[0], Cb0);
        image[3 * pid + 1] = fmaf(Tb, P.bg[1], Cb1);
        image[3 * pid + 2] = fmaf(Tb, P.bg[2], Cb2);
        final_T[pid] = Tb;
        n_contrib[pid] = last_b;
        if (FEAT) { depth_img[pid] = Db; alpha_img[pid] = Ab; }
    }
}

// Backward compositing (a9).  One CTA per 16x16 tile; a thread owns PPT consecutive pixels of one row
// (8 -> 32 threads, ONE WARP PER TILE, the throughput shape; 2 -> 128 threads for images with few tiles), handled as PPT/2
// packed pairs, so that a Gaussian's record is read from shared memory once per PPT pixel-pairs, the row terms of
// `power` are shared, and the per-Gaussian reduction runs once per 32 * PPT pixel-pairs: each lane first sums
// its own pixels in registers, then one transposed butterfly (14 shuffles for the 9 gradients) leaves the totals
// spread over lanes, which issue two RED instructions (8 lanes + 1 lane).
//
// Per pixel, branch-free (a gated pixel enters with o G = 0, hence alpha = 0, 1/(1-alpha) = 1, w = 0): restore
// T_k = T_{k+1} / (1 - alpha_k); dL/dc_k = w g; dL/dalpha_k = T_k (g . c_k) - Q_k / (1 - alpha_k) with the ONE running
// scalar Q_k = g . S_k (S_k = colour behind k, C13), kept negated (R = -Q) so that both uses are FMAs.
// FEAT (xpr_rasterize_feat_bwd; reading C31): with gD = dL/dD, gA = dL/dA of the pixel,
//   dL/dz_k = alpha_k T_k gD,  dL/dalpha_k = T_k (g . c_k + gD z_k + gA) - (g . S + gD SD + gA SA) / (1 - alpha_k);
// SA telescopes (alpha_j T_j = T_j - T_{j+1}): gA (T_k - SA_k / (1 - alpha_k)) = gA T_final / (1 - alpha_k), so the
// accumulated-opacity term is the per-pixel constant -gA T_final inside Q: Q_k = sum_{j>k} (g . c_j + gD z_j) alpha_j T_j
// + T_final (g . bg - gA).
#ifndef XPR_BWD_PPT_SMALL
#define XPR_BWD_PPT_SMALL 2
#endif
#ifndef XPR_BWD_PPT_LARGE
#define XPR_BWD_PPT_LARGE 8  // pixels per thread in the throughput shape (8: one warp per tile; 4: two)
#endif
#ifndef XPR_BWD_MINB
#define XPR_BWD_MINB 14      // 64-thread CTAs per SM in the throughput shape (72 registers; 12: +1.5 % time, 10: +3 %)
#endif
#ifndef XPR_BWD_MINB8
#define XPR_BWD_MINB8 16     // 32-thread CTAs per SM at 8 pixels per thread (124 registers; 20 spills, 12: +8 % time)
#endif
template <int PPT, bool FEAT>
__global__ void __launch_bounds__(BLOCK / PPT, PPT == 8 ? XPR_BWD_MINB8 : XPR_BWD_MINB * PPT / 4)
rasterize_bwd_kernel(RasterParams P, const float4* __restrict__ rec, const uint32_t* __restrict__ vals,
                     const uint2* __restrict__ ranges, const float* __restrict__ final_T,
                     const uint32_t* __restrict__ n_contrib, const float* __restrict__ dL,
                     const float* __restrict__ dL_dD, const float* __restrict__ dL_dA, float* __restrict__ g_mean2d,
                     float* __restrict__ g_conic, float* __restrict__ g_opac, float* __restrict__ g_rgb,
                     float* __restrict__ g_depth, int loss_kind, const float* __restrict__ image,
                     const float* __restrict__ target) {
    // loss_kind < 0: dL is the incoming gradient.  loss_kind 0 / 1 (xpr_rasterize_bwd_loss): the gradient of the loss
    // sum |I - target| / sum (I - target)^2 is formed here from the rendered image and the target, the values
    // xpr_loss_grad would have written (one pass over the image and one launch less per step).
    constexpr int THREADS = BLOCK / PPT, B = THREADS, NP = PPT / 2;
    __shared__ float4 s_rec[STAGES][3 * B];
    __shared__ uint32_t s_idx[STAGES][B];
    __shared__ uint32_t s_max[THREADS / 32];
    const int tid = threadIdx.x, lane = tid & 31;
    const int tile = P.order ? (int)P.order[blockIdx.x] : (int)blockIdx.x;
    const int view = tile / P.T, vt = tile - view * P.T;
    const int64_t vbase = (int64_t)view * P.H * P.W;
    const int tx = vt % P.TW, ty = vt / P.TW;
    // a thread owns PPT consecutive pixels of one row: they share dy and the row terms of `power`
    constexpr int TPR = TILE / PPT;                 // threads per tile row
    const int px0 = tx * TILE + (tid % TPR) * PPT;
    const int py = ty * TILE + (tid / TPR);
    const float pyc = (float)py + 0.5f;
    const uint2 rg = ranges[tile];
    const uint32_t* const list = vals + rg.x;

    uint32_t n[PPT];
    f32x2 px2[NP], T2[NP], R2[NP], g0_2[NP], g1_2[NP], g2_2[NP], gD_2[NP];
    uint32_t wmax = 0;
    {
        // per-pixel inputs: n_contrib, T_final and dL/dpixel (or image and target).  A thread's PPT pixels are consecutive,
        // so when the row is whole and the arrays are 16-byte aligned (P.vec: W % 4 == 0) they are read as 128-bit words
        float tt[PPT], a0[PPT], a1[PPT], a2[PPT], aD[PPT], gA[PPT];
        auto sgn = [](float d) { return d > 0.0f ? 1.0f : (d < 0.0f ? -1.0f : d); };
#pragma unroll
        for (int k = 0; k < PPT; ++k) { n[k] = 0; tt[k] = a0[k] = a1[k] = a2[k] = aD[k] = gA[k] = 0.0f; }
        if ((PPT % 4 == 0) && P.vec && (px0 + PPT <= P.W) && (py < P.H)) {
            const int64_t pid0 = vbase + (int64_t)py * P.W + px0;
            constexpr int Q = (PPT % 4 == 0) ? PPT / 4 : 1;
            float c[12 * Q];
#pragma unroll
            for (int v = 0; v < Q; ++v) {
                const uint4 nv = __ldg(reinterpret_cast<const uint4*>(n_contrib + pid0) + v);
                const float4 tv = __ldg(reinterpret_cast<const float4*>(final_T + pid0) + v);
                n[4 * v] = nv.x; n[4 * v + 1] = nv.y; n[4 * v + 2] = nv.z; n[4 * v + 3] = nv.w;
                tt[4 * v] = tv.x; tt[4 * v + 1] = tv.y; tt[4 * v + 2] = tv.z; tt[4 * v + 3] = tv.w;
                if (FEAT) {
                    const float4 dv = __ldg(reinterpret_cast<const float4*>(dL_dD + pid0) + v);
                    const float4 av = __ldg(reinterpret_cast<const float4*>(dL_dA + pid0) + v);
                    aD[4 * v] = dv.x; aD[4 * v + 1] = dv.y; aD[4 * v + 2] = dv.z; aD[4 * v + 3] = dv.w;
                    gA[4 * v] = av.x; gA[4 * v + 1] = av.y; gA[4 * v + 2] = av.z; gA[4 * v + 3] = av.w;
                }
            }
#pragma unroll
            for (int v = 0; v < 3 * Q; ++v) {
                float4 x;
                if (loss_kind < 0) x = __ldg(reinterpret_cast<const float4*>(dL + 3 * pid0) + v);
                else {
                    const float4 im = __ldg(reinterpret_cast<const float4*>(image + 3 * pid0) + v);
                    const float4 tg = __ldg(reinterpret_cast<const float4*>(target + 3 * pid0) + v);
                    const float d0 = im.x - tg.x, d1 = im.y - tg.y, d2 = im.z - tg.z, d3 = im.w - tg.w;
                    x = loss_kind == 0 ? make_float4(sgn(d0), sgn(d1), sgn(d2), sgn(d3)) : make_float4(2.0f * d0, 2.0f * d1, 2.0f * d2, 2.0f * d3);
                }
                c[4 * v] = x.x; c[4 * v + 1] = x.y; c[4 * v + 2] = x.z; c[4 * v + 3] = x.w;
            }
#pragma unroll
            for (int k = 0; k < 4 * Q; ++k) { a0[k] = c[3 * k]; a1[k] = c[3 * k + 1]; a2[k] = c[3 * k + 2]; }
        } else {
#pragma unroll
            for (int k = 0; k < PPT; ++k) {
                const int px = px0 + k;
                if (px < P.W && py < P.H) {
                    const int64_t pid = vbase + (int64_t)py * P.W + px;
                    n[k] = n_contrib[pid];
                    tt[k] = final_T[pid];
                    if (loss_kind < 0) {
                        a0[k] = dL[3 * pid]; a1[k] = dL[3 * pid + 1]; a2[k] = dL[3 * pid + 2];
                    } else {
                        const float d0 = image[3 * pid] - target[3 * pid], d1 = image[3 * pid + 1] - target[3 * pid + 1],
                                    d2 = image[3 * pid + 2] - target[3 * pid + 2];
                        a0[k] = loss_kind == 0 ? sgn(d0) : 2.0f * d0;
                        a1[k] = loss_kind == 0 ? sgn(d1) : 2.0f * d1;
                        a2[k] = loss_kind == 0 ? sgn(d2) : 2.0f * d2;
                    }
                    if (FEAT) { aD[k] = dL_dD[pid]; gA[k] = dL_dA[pid]; }
                }
            }
        }
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            float q[2];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int k = 2 * p + h;
                // Q = g . S behind the last entry = T_final (g . bg) (C13) (FEAT: - gA T_final)
                q[h] = tt[k] * (fmaf(a2[k], P.bg[2], fmaf(a1[k], P.bg[1], a0[k] * P.bg[0])) - gA[k]);
                wmax = max(wmax, n[k]);
            }
            px2[p] = pack2((float)(px0 + 2 * p) + 0.5f, (float)(px0 + 2 * p + 1) + 0.5f);
            T2[p] = pack2(tt[2 * p], tt[2 * p + 1]); R2[p] = pack2(-q[0], -q[1]);
            g0_2[p] = pack2(a0[2 * p], a0[2 * p + 1]); g1_2[p] = pack2(a1[2 * p], a1[2 * p + 1]);
            g2_2[p] = pack2(a2[2 * p], a2[2 * p + 1]);
            gD_2[p] = pack2(aD[2 * p], aD[2 * p + 1]);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) wmax = max(wmax, __shfl_xor_sync(0xffffffffu, wmax, o));
    if (lane == 0) s_max[tid >> 5] = wmax;
    __syncthreads();
    uint32_t max_n = 0;
#pragma unroll
    for (int w = 0; w < THREADS / 32; ++w) max_n = max(max_n, s_max[w]);

    // lane (4 i) owns gradient i of the 8-value butterfly: its base pointer and per-Gaussian stride
    const int vi = lane >> 2;
    float* const red_base = (vi < 2) ? (g_mean2d + vi) : (vi < 5) ? (g_conic + (vi - 2)) : (g_rgb + (vi - 5));
    const uint32_t red_stride = (vi < 2) ? 2u : 3u;
    const bool red_lane = (lane & 3) == 0;

    // staging ring over the list positions max_n-1 ... 0 (descending): entry e = b B + j is position max_n-1-e
    auto stage_entry = [&](uint32_t s, uint32_t g) {
        s_idx[s][tid] = g;
        stage_record(&s_rec[s][3 * tid], rec, g);
    };
    {
        uint32_t g0 = 0, g1 = 0;
        if ((uint32_t)tid < max_n) g0 = list[max_n - 1u - (uint32_t)tid];
        if ((uint32_t)(B + tid) < max_n) g1 = list[max_n - 1u - (uint32_t)(B + tid)];
        if ((uint32_t)tid < max_n) stage_entry(0, g0);
        cp_async_commit();
        if ((uint32_t)(B + tid) < max_n) stage_entry(1, g1);
        cp_async_commit();
    }
    // index of this thread's entry of batch b + 2, loaded one batch ahead of the copy that needs it
    uint32_t g_next = ((uint32_t)(2 * B + tid) < max_n) ? list[max_n - 1u - (uint32_t)(2 * B + tid)] : 0u;

    const float amax = P.amax;
    uint32_t stage = 0;
    for (uint32_t base = 0; base < max_n; base += B) {
        cp_async_wait<1>();
        __syncthreads();               // batch b visible to all; everyone is done with batch b - 1
        {
            const uint32_t s2 = (stage + 2 >= STAGES) ? stage + 2 - STAGES : stage + 2;
            if (base + 2 * B + tid < max_n) stage_entry(s2, g_next);
            cp_async_commit();
            g_next = (base + 3 * B + tid < max_n) ? list[max_n - 1u - (base + 3 * B + tid)] : 0u;
        }
        const uint32_t cnt = min((uint32_t)B, max_n - base);
        const float4* rq = s_rec[stage];
        for (uint32_t j = 0; j < cnt; ++j, rq += 3) {
            const uint32_t pos = max_n - 1u - (base + j);
            if (pos >= wmax) continue;     // warp-uniform: nobody in this warp got this far
            const float4 ge = rq[0];       // mx my qa qb
            const float4 ga = rq[1];       // qc thr log2o z
            const float dy = pyc - ge.y;
            const float t1 = __fmul_rn(-ge.w, dy), t2 = __fmul_rn(__fmul_rn(-ga.x, dy), dy);   // row terms of -power
            const uint32_t lim = __float_as_uint(ga.y);                                          // bits of lnv
            f32x2 dx2[NP], pw2[NP];                                                              // pw2 = -power (forward kernel)
            bool contrib[PPT], any_c = false;
#pragma unroll
            for (int p = 0; p < NP; ++p) {
                dx2[p] = sub2(px2[p], bcast2(ge.x));
                pw2[p] = fma2(fma2(bcast2(-ge.z), dx2[p], bcast2(t1)), dx2[p], bcast2(t2));  // rule R3, per lane, negated
                float pa, pb;
                unpack2(pw2[p], pa, pb);
                contrib[2 * p] = (pos < n[2 * p]) && gate(pa, lim);
                contrib[2 * p + 1] = (pos < n[2 * p + 1]) && gate(pb, lim);
                any_c |= contrib[2 * p] || contrib[2 * p + 1];
            }
            if (!__any_sync(0xffffffffu, any_c)) continue;
            const float4 c = rq[2];        // r g b o
            // the thread's pixels share dy: accumulate sum dpow, sum dpow dx, sum dpow dx^2 and form the five
            // geometric gradients once per entry (dpow = dL/dpower of a pixel)
            f32x2 sp2, spx2, spxx2, vr2, vg2, vb2, sz2;
#pragma unroll
            for (int p = 0; p < NP; ++p) {
                float ea, eb;
                unpack2(fma2(pw2[p], bcast2(-LOG2E), bcast2(ga.z)), ea, eb);
                const float og_a = contrib[2 * p] ? ex2_approx(ea) : 0.0f;          // o G
                const float og_b = contrib[2 * p + 1] ? ex2_approx(eb) : 0.0f;
                const f32x2 al2 = pack2(fminf(amax, og_a), fminf(amax, og_b));       // C11
                float oma_a, oma_b;
                unpack2(sub2(bcast2(1.0f), al2), oma_a, oma_b);
                const f32x2 inv2 = pack2(rcp_approx(oma_a), rcp_approx(oma_b));
                T2[p] = mul2(T2[p], inv2);                                           // transmittance in front of this entry
                const f32x2 w2 = mul2(al2, T2[p]);
                if (p == 0) { vr2 = mul2(w2, g0_2[p]); vg2 = mul2(w2, g1_2[p]); vb2 = mul2(w2, g2_2[p]); }
                else { vr2 = fma2(w2, g0_2[p], vr2); vg2 = fma2(w2, g1_2[p], vg2); vb2 = fma2(w2, g2_2[p], vb2); }
                // g . c (FEAT: + gD z)
                f32x2 gc2 = fma2(g2_2[p], bcast2(c.z), fma2(g1_2[p], bcast2(c.y), mul2(g0_2[p], bcast2(c.x))));
                if (FEAT) {
                    gc2 = fma2(gD_2[p], bcast2(ga.w), gc2);
                    sz2 = (p == 0) ? mul2(w2, gD_2[p]) : fma2(w2, gD_2[p], sz2);     // dL/dz
                }
                // dL/dalpha = T (g . c) - Q / (1 - alpha) = T gc + inv R;   R <- R - gc w
                const f32x2 da2 = fma2(inv2, R2[p], mul2(T2[p], gc2));
                R2[p] = fma2(neg2(gc2), w2, R2[p]);
                // C14: the clamp has zero derivative; dL/dpower = o G dL/dalpha (dL/do = G dL/dalpha = dpow / o: summed as sp).
                // The mask as a 1 / 0 factor (one FSET per pixel and one packed product instead of compare + select per pixel)
                const f32x2 m2 = pack2((og_a < amax) ? 1.0f : 0.0f, (og_b < amax) ? 1.0f : 0.0f);
                const f32x2 dpow2 = mul2(mul2(pack2(og_a, og_b), da2), m2);
                const f32x2 dxp2 = mul2(dx2[p], dpow2);
                if (p == 0) { sp2 = dpow2; spx2 = dxp2; spxx2 = mul2(dx2[p], dxp2); }
                else { sp2 = add2(sp2, dpow2); spx2 = add2(spx2, dxp2); spxx2 = fma2(dx2[p], dxp2, spxx2); }
            }
            float v[8];                                // mx my A B C r g b
            const float sp = sum2(sp2), spx = sum2(spx2), spxx = sum2(spxx2);
            v[5] = sum2(vr2); v[6] = sum2(vg2); v[7] = sum2(vb2);
            {
                // dpower/dm = (A dx + B dy, B dx + C dy) = -(2 qa dx + qb dy, qb dx + 2 qc dy); dpower/d(A, B, C) = (-dx^2/2, -dx dy, -dy^2/2)
                const float sy = dy * sp;              // sum dpow dy
                v[0] = -fmaf(2.0f * ge.z, spx, ge.w * sy); v[1] = -fmaf(ge.w, spx, 2.0f * ga.x * sy);
                v[2] = -0.5f * spxx; v[3] = -dy * spx; v[4] = -0.5f * dy * sy;
            }
            const float tot = warp_reduce8(v, lane);
            const uint32_t g = s_idx[stage][j];
            if (FEAT) {
                // lanes 0-15 end with the warp total of sp, lanes 16-31 with that of sz
                const float sz = sum2(sz2);
                float r2 = ((lane & 16) ? sz : sp) + __shfl_xor_sync(0xffffffffu, (lane & 16) ? sp : sz, 16);
#pragma unroll
                for (int o = 8; o > 0; o >>= 1) r2 += __shfl_xor_sync(0xffffffffu, r2, o);
                if (red_lane) atomicAdd(red_base + red_stride * g, tot);
                if (lane == 0) atomicAdd(g_opac + g, r2 * rcp_approx(c.w));
                if (lane == 16) atomicAdd(g_depth + g, r2);
            } else {
                const float sp_tot = warp_sum(sp);     // dL/do = (sum dpow) / o, divided by the one lane that adds it
                if (red_lane) atomicAdd(red_base + red_stride * g, tot);
                if (lane == 0) atomicAdd(g_opac + g, sp_tot * rcp_approx(c.w));
            }
        }
        stage = (stage + 1 == STAGES) ? 0 : stage + 1;
    }
    cp_async_wait<0>();
}

// xpr_shade_record: the 48-byte shader record from the separate projection outputs (for callers that did not
// get it from xpr_project).  One thread per Gaussian; culled Gaussians are skipped (their record is never read).
__global__ void __launch_bounds__(256)
shade_record_kernel(int64_t N, const float2* __restrict__ mean2d, const float4* __restrict__ conic_opac,
                    const float* __restrict__ rgb, const float* __restrict__ lnv, const float* __restrict__ depth,
                    const uint32_t* __restrict__ tcount, float4* __restrict__ rec) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N || tcount[i] == 0u) return;
    const float2 m = mean2d[i];
    const float4 co = conic_opac[i];
    rec[3 * i] = make_float4(m.x, m.y, -0.5f * co.x, -co.y);
    rec[3 * i + 1] = make_float4(-0.5f * co.z, lnv[i], __log2f(co.w), depth ? depth[i] : 0.0f);
    rec[3 * i + 2] = make_float4(rgb[3 * i], rgb[3 * i + 1], rgb[3 * i + 2], co.w);
}

void make_raster_params(const xpr_camera* cam, const xpr_config* cfg, RasterParams& P) {
    P.W = cam->width; P.H = cam->height; P.TW = tiles_x(cam); P.T = tiles_x(cam) * tiles_y(cam);
    P.amax = cfg->alpha_max; P.tmin = cfg->t_min;
    for (int i = 0; i < 3; ++i) P.bg[i] = cfg->bg[i];
    P.order = cfg->tile_order;
    P.vec = 0;
}

template <bool FEAT>
int32_t launch_fwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* shade_rec,
                   const uint32_t* vals_sorted, const uint32_t* tile_ranges, float* image, float* final_T,
                   uint32_t* n_contrib, float* depth_img, float* alpha_img, void* stream) {
    if (int32_t s = check_cam_cfg(cam, cfg)) return s;
    if (N < 0) return XPR_ERR_INVALID_ARG;
    if (!aligned(tile_ranges, 8) || !aligned(image, 4) || !aligned(final_T, 4) || !aligned(n_contrib, 4))
        return XPR_ERR_INVALID_ARG;
    if (FEAT && (!aligned(depth_img, 4) || !aligned(alpha_img, 4))) return XPR_ERR_INVALID_ARG;
    if (N > 0 && (!aligned(shade_rec, 16) || !aligned(vals_sorted, 4))) return XPR_ERR_INVALID_ARG;
    RasterParams P;
    make_raster_params(cam, cfg, P);
    const int T = tiles_x(cam) * tiles_y(cam) * num_views(cfg);
    // throughput shape once the image has enough tiles for several waves of every SM; branch-free blend when
    // the lists were culled
#define XPR_FWD(PPT_, BF_)                                                                                          \
    rasterize_fwd_kernel<false, PPT_, BF_, FEAT><<<T, BLOCK / PPT_, 0, (cudaStream_t)stream>>>(                       \
        P, reinterpret_cast<const float4*>(shade_rec), vals_sorted, reinterpret_cast<const uint2*>(tile_ranges),     \
        image, final_T, n_contrib, nullptr, depth_img, alpha_img)
    const bool bf = cfg->tile_cull != 0;
    if (T >= FWD_PPT2_MIN_TILES) { if (bf) XPR_FWD(2, true); else XPR_FWD(2, false); }
    else                         { XPR_FWD(1, false); }      // latency shape: the branchy blend is shorter
#undef XPR_FWD
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}

template <bool FEAT>
int32_t launch_bwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* shade_rec,
                   const uint32_t* vals_sorted, const uint32_t* tile_ranges, const float* final_T,
                   const uint32_t* n_contrib, const float* dL_dimage, const float* dL_ddepth, const float* dL_dalpha,
                   float* g_mean2d, float* g_conic, float* g_opac, float* g_rgb, float* g_depth, int32_t zero_init,
                   void* stream, int loss_kind = -1, const float* image = nullptr, const float* target = nullptr) {
    if (int32_t s = check_cam_cfg(cam, cfg)) return s;
    if (N < 0) return XPR_ERR_INVALID_ARG;
    if (N >= (1ll << 30)) return XPR_ERR_UNSUPPORTED;      // xpr_bin_sort's limit; the kernel indexes the gradients with 32 bits
    if (!aligned(tile_ranges, 8) || !aligned(final_T, 4) || !aligned(n_contrib, 4)) return XPR_ERR_INVALID_ARG;
    if (loss_kind < 0 ? !aligned(dL_dimage, 4) : (loss_kind > 1 || !aligned(image, 4) || !aligned(target, 4)))
        return XPR_ERR_INVALID_ARG;
    if (FEAT && (!aligned(dL_ddepth, 4) || !aligned(dL_dalpha, 4))) return XPR_ERR_INVALID_ARG;
    if (N == 0) return XPR_OK;
    if (!aligned(shade_rec, 16) || !aligned(vals_sorted, 4) || !aligned(g_mean2d, 4) || !aligned(g_conic, 4) ||
        !aligned(g_opac, 4) || !aligned(g_rgb, 4) || (FEAT && !aligned(g_depth, 4)))
        return XPR_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    if (zero_init) {
        const size_t n = (size_t)N;
        const bool adjacent = g_conic == g_mean2d + 2 * n && g_opac == g_conic + 3 * n && g_rgb == g_opac + n;
        if (adjacent && (!FEAT || g_depth == g_rgb + 3 * n)) {
            XPR_CUDA(cudaMemsetAsync(g_mean2d, 0, sizeof(float) * (FEAT ? 10 : 9) * n, st));   // one allocation: one fill
        } else {
            XPR_CUDA(cudaMemsetAsync(g_mean2d, 0, sizeof(float) * 2 * n, st));
            XPR_CUDA(cudaMemsetAsync(g_conic, 0, sizeof(float) * 3 * n, st));
            XPR_CUDA(cudaMemsetAsync(g_opac, 0, sizeof(float) * n, st));
            XPR_CUDA(cudaMemsetAsync(g_rgb, 0, sizeof(float) * 3 * n, st));
            if (FEAT) XPR_CUDA(cudaMemsetAsync(g_depth, 0, sizeof(float) * n, st));
        }
    }
    RasterParams P;
    make_raster_params(cam, cfg, P);
    P.vec = (cam->width % 4 == 0) && aligned(final_T, 16) && aligned(n_contrib, 16) &&
            (loss_kind < 0 ? aligned(dL_dimage, 16) : (aligned(image, 16) && aligned(target, 16))) &&
            (!FEAT || (aligned(dL_ddepth, 16) && aligned(dL_dalpha, 16)));
    const int T = tiles_x(cam) * tiles_y(cam) * num_views(cfg);
    // 8 pixels per thread (one warp per tile) is the throughput shape; images with few tiles are bounded by their
    // heaviest tile, where more warps per tile (2 pixels per thread) shorten the critical path
#define XPR_BWD(PPT_)                                                                                               \
    rasterize_bwd_kernel<PPT_, FEAT><<<T, BLOCK / PPT_, 0, st>>>(                                                     \
        P, reinterpret_cast<const float4*>(shade_rec), vals_sorted, reinterpret_cast<const uint2*>(tile_ranges),     \
        final_T, n_contrib, dL_dimage, dL_ddepth, dL_dalpha, g_mean2d, g_conic, g_opac, g_rgb, g_depth, loss_kind,   \
        image, target)
    if (T >= FWD_PPT2_MIN_TILES) XPR_BWD(XPR_BWD_PPT_LARGE);
    else                         XPR_BWD(XPR_BWD_PPT_SMALL);
#undef XPR_BWD
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}

}  // namespace
}  // namespace xpr

using namespace xpr;

extern "C" int32_t xpr_shade_record(int64_t N, const float* mean2d, const float* conic_opac, const float* rgb,
                                    const float* lnv, const float* depth, const uint32_t* tile_count,
                                    float* shade_rec, void* stream) {
    if (N < 0) return XPR_ERR_INVALID_ARG;
    if (N == 0) return XPR_OK;
    if (!aligned(mean2d, 8) || !aligned(conic_opac, 16) || !aligned(rgb, 4) || !aligned(lnv, 4) ||
        (depth && !aligned(depth, 4)) || !aligned(tile_count, 4) || !aligned(shade_rec, 16))
        return XPR_ERR_INVALID_ARG;
    shade_record_kernel<<<(unsigned)((N + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
        N, reinterpret_cast<const float2*>(mean2d), reinterpret_cast<const float4*>(conic_opac), rgb, lnv, depth,
        tile_count, reinterpret_cast<float4*>(shade_rec));
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}

extern "C" int32_t xpr_rasterize_fwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* shade_rec,
                                     const uint32_t* vals_sorted, const uint32_t* tile_ranges, float* image,
                                     float* final_T, uint32_t* n_contrib, void* stream) {
    return launch_fwd<false>(cam, cfg, N, shade_rec, vals_sorted, tile_ranges, image, final_T, n_contrib, nullptr,
                             nullptr, stream);
}

extern "C" int32_t xpr_rasterize_feat_fwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N,
                                          const float* shade_rec, const uint32_t* vals_sorted,
                                          const uint32_t* tile_ranges, float* image, float* final_T,
                                          uint32_t* n_contrib, float* depth_img, float* alpha_img, void* stream) {
    return launch_fwd<true>(cam, cfg, N, shade_rec, vals_sorted, tile_ranges, image, final_T, n_contrib, depth_img,
                            alpha_img, stream);
}

extern "C" int32_t xpr_rasterize_stats(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* shade_rec,
                                       const uint32_t* vals_sorted, const uint32_t* tile_ranges, uint64_t* stats,
                                       void* stream) {
    if (int32_t s = check_cam_cfg(cam, cfg)) return s;
    if (N < 0 || !aligned(tile_ranges, 8) || !aligned(stats, 8)) return XPR_ERR_INVALID_ARG;
    if (N > 0 && (!aligned(shade_rec, 16) || !aligned(vals_sorted, 4))) return XPR_ERR_INVALID_ARG;
    RasterParams P;
    make_raster_params(cam, cfg, P);
    const int T = tiles_x(cam) * tiles_y(cam) * num_views(cfg);
    XPR_CUDA(cudaMemsetAsync(stats, 0, 4 * sizeof(uint64_t), (cudaStream_t)stream));
    rasterize_fwd_kernel<true, 1, false, false><<<T, BLOCK, 0, (cudaStream_t)stream>>>(
        P, reinterpret_cast<const float4*>(shade_rec), vals_sorted, reinterpret_cast<const uint2*>(tile_ranges), nullptr,
        nullptr, nullptr, reinterpret_cast<unsigned long long*>(stats), nullptr, nullptr);
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}

extern "C" int32_t xpr_rasterize_bwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* shade_rec,
                                     const uint32_t* vals_sorted, const uint32_t* tile_ranges, const float* final_T,
                                     const uint32_t* n_contrib, const float* dL_dimage, float* g_mean2d,
                                     float* g_conic, float* g_opac, float* g_rgb, int32_t zero_init, void* stream) {
    return launch_bwd<false>(cam, cfg, N, shade_rec, vals_sorted, tile_ranges, final_T, n_contrib, dL_dimage, nullptr,
                             nullptr, g_mean2d, g_conic, g_opac, g_rgb, nullptr, zero_init, stream);
}

extern "C" int32_t xpr_rasterize_bwd_loss(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* shade_rec,
                                          const uint32_t* vals_sorted, const uint32_t* tile_ranges, const float* image,
                                          const float* final_T, const uint32_t* n_contrib, int32_t loss_kind,
                                          const float* target, float* g_mean2d, float* g_conic, float* g_opac,
                                          float* g_rgb, int32_t zero_init, void* stream) {
    if (loss_kind != 0 && loss_kind != 1) return XPR_ERR_INVALID_ARG;
    return launch_bwd<false>(cam, cfg, N, shade_rec, vals_sorted, tile_ranges, final_T, n_contrib, nullptr, nullptr, nullptr,
                             g_mean2d, g_conic, g_opac, g_rgb, nullptr, zero_init, stream, loss_kind, image, target);
}

extern "C" int32_t xpr_rasterize_feat_bwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N,
                                          const float* shade_rec, const uint32_t* vals_sorted,
                                          const uint32_t* tile_ranges, const float* final_T,
                                          const uint32_t* n_contrib, const float* dL_dimage, const float* dL_ddepth,
                                          const float* dL_dalpha, float* g_mean2d, float* g_conic, float* g_opac,
                                          float* g_rgb, float* g_depth, int32_t zero_init, void* stream) {
    return launch_bwd<true>(cam, cfg, N, shade_rec, vals_sorted, tile_ranges, final_T, n_contrib, dL_dimage, dL_ddepth,
                            dL_dalpha, g_mean2d, g_conic, g_opac, g_rgb, g_depth, zero_init, stream);
}
