// project.cu -- xpr_project / xpr_project_bwd: per-Gaussian projection (EWA and unscented transform),
// SH -> RGB, tile rectangle / tile count, and the reverse-mode pass through all of it.
//
// One thread per Gaussian ("map_fn over primitives").  This translation unit is
// compiled with -fmad=false (rule R1): every fp32 operation that feeds depth
// bits, mean2d, the 2D covariance, the extents and floor/ceil is individually rounded, in the
// order DESIGN.md section 3 "Arithmetic order" fixes, so that tile rectangles, tile counts and
// sort keys are bit-reproducible.  Transcendentals that feed integers go through fp64 (rule R2).
//
// PAPER citations: Listing 1 L239-262 (3DGS project), L435 (conic, alpha_thresh), L437 and
// Listing 3 L447-486 (3DGUT project), L78 (Sigma = R S S^T R^T), L147 (half-open tile AABB).
#include <math.h>

#include "common.cuh"
#include "packed.cuh"

namespace xpr {
namespace {

struct ProjParams {
    float W[9], t[3];
    float fx, fy, cx, cy;
    double k[4];
    int model, projection, K, antialias;
    float alpha_thresh, z_near, lowpass;
    float lox, hix, loy, hiy;      // C6 Jacobian clamp bounds on x/z, y/z
    float gamma, wm0, wc0, wk;     // unscented-transform spread and weights
    float cpos[3];                 // camera position -W^T t
    int TW, TH;
};
struct ProjBatch { ProjParams p[XPR_MAX_VIEWS]; };   // one entry per view of a batch (xpr_config.views), kernel parameter

// Real SH basis, degree <= 3, index k = l^2 + l + m, Condon-Shortley sign (reading C5).
#define XPR_SH_C0 ((float)0.28209479177387814)   // 1/(2 sqrt(pi))
#define XPR_SH_C1 ((float)0.4886025119029199)    // sqrt(3/(4 pi))
#define XPR_SH_A2 ((float)1.0925484305920792)    // sqrt(15/pi)/2
#define XPR_SH_B2 ((float)0.31539156525252005)   // sqrt(5/pi)/4
#define XPR_SH_C2 ((float)0.5462742152960396)    // sqrt(15/pi)/4
#define XPR_SH_A3 ((float)0.5900435899266435)    // sqrt(35/(2 pi))/4
#define XPR_SH_B3 ((float)2.890611442640554)     // sqrt(105/pi)/2
#define XPR_SH_C3 ((float)0.4570457994644658)    // sqrt(21/(2 pi))/4
#define XPR_SH_D3 ((float)0.3731763325901154)    // sqrt(7/pi)/4
#define XPR_SH_E3 ((float)1.445305721320277)     // sqrt(105/pi)/4

__device__ __forceinline__ void sh_basis(float x, float y, float z, float* Y) {
    const float xx = x * x, yy = y * y, zz = z * z, xy = x * y, yz = y * z, xz = x * z;
    Y[0] = XPR_SH_C0;
    Y[1] = (-XPR_SH_C1) * y;
    Y[2] = XPR_SH_C1 * z;
    Y[3] = (-XPR_SH_C1) * x;
    Y[4] = XPR_SH_A2 * xy;
    Y[5] = (-XPR_SH_A2) * yz;
    Y[6] = XPR_SH_B2 * ((2.0f * zz - xx) - yy);
    Y[7] = (-XPR_SH_A2) * xz;
    Y[8] = XPR_SH_C2 * (xx - yy);
    Y[9] = ((-XPR_SH_A3) * y) * (3.0f * xx - yy);
    Y[10] = (XPR_SH_B3 * xy) * z;
    Y[11] = ((-XPR_SH_C3) * y) * ((4.0f * zz - xx) - yy);
    Y[12] = (XPR_SH_D3 * z) * ((2.0f * zz - 3.0f * xx) - 3.0f * yy);
    Y[13] = ((-XPR_SH_C3) * x) * ((4.0f * zz - xx) - yy);
    Y[14] = (XPR_SH_E3 * z) * (xx - yy);
    Y[15] = ((-XPR_SH_A3) * x) * (xx - 3.0f * yy);
}

// Camera model pi: camera-space point -> continuous pixel (C1, C2, C18); R2: atan2 and the radial
// polynomial in fp64.
__device__ __forceinline__ void camera_project(const ProjParams& P, const float p[3], float pix[2]) {
    if (P.model == 0) {
        pix[0] = P.fx * (p[0] / p[2]) + P.cx;
        pix[1] = P.fy * (p[1] / p[2]) + P.cy;
        return;
    }
    const float r = sqrtf(p[0] * p[0] + p[1] * p[1]);
    float s;
    if (r > 0.0f) {
        const double th = atan2((double)r, (double)p[2]);
        const double t2 = th * th;
        const double poly = 1.0 + t2 * (P.k[0] + t2 * (P.k[1] + t2 * (P.k[2] + t2 * P.k[3])));
        s = (float)((th * poly) / (double)r);
    } else {
        s = (float)(1.0 / (double)p[2]);
    }
    pix[0] = P.fx * (s * p[0]) + P.cx;
    pix[1] = P.fy * (s * p[1]) + P.cy;
}

// Forward intermediates of one Gaussian, kept in registers (backward recomputes them).
struct Fwd {
    float p[3];
    float u0, v0, u, v;
    bool clamp_u, clamp_v;
    float R[9], M[9], Sig[9];
    float T[6];
    float m[2];
    float a, b, c, ap, cp, det, det_raw, rho, o_eff;
    float A, B, C, lnv;
    int rect[4];
    uint32_t tc;
    // UT
    float pc[7][3], y[7][2];
};

// Returns true when the Gaussian passes every visibility test of PAPER L262 (C9, C26: all tests
// are written in the positive sense so that a NaN culls).  `full` = also keep what backward needs.
__device__ __forceinline__ bool project_geometry(const ProjParams& P, const float mu[3], const float sc[3],
                                                 const float q[4], float o, Fwd& F) {
    const float* W = P.W;
    for (int i = 0; i < 3; ++i) F.p[i] = ((W[3 * i] * mu[0] + W[3 * i + 1] * mu[1]) + W[3 * i + 2] * mu[2]) + P.t[i];
    if (!(F.p[2] > P.z_near)) return false;
    {   // R(q), (w,x,y,z), not renormalised (C3)
        const float w = q[0], x = q[1], y = q[2], z = q[3];
        const float xx = x * x, yy = y * y, zz = z * z, xy = x * y, xz = x * z, yz = y * z;
        const float wx = w * x, wy = w * y, wz = w * z;
        F.R[0] = 1.0f - 2.0f * (yy + zz); F.R[1] = 2.0f * (xy - wz); F.R[2] = 2.0f * (xz + wy);
        F.R[3] = 2.0f * (xy + wz); F.R[4] = 1.0f - 2.0f * (xx + zz); F.R[5] = 2.0f * (yz - wx);
        F.R[6] = 2.0f * (xz - wy); F.R[7] = 2.0f * (yz + wx); F.R[8] = 1.0f - 2.0f * (xx + yy);
    }
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) F.M[3 * i + j] = F.R[3 * i + j] * sc[j];

    if (P.projection == 0) {
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j)
                F.Sig[3 * i + j] = (F.M[3 * i] * F.M[3 * j] + F.M[3 * i + 1] * F.M[3 * j + 1]) + F.M[3 * i + 2] * F.M[3 * j + 2];
        F.u0 = F.p[0] / F.p[2]; F.v0 = F.p[1] / F.p[2];
        F.m[0] = P.fx * F.u0 + P.cx; F.m[1] = P.fy * F.v0 + P.cy;
        F.clamp_u = !(F.u0 >= P.lox && F.u0 <= P.hix);
        F.clamp_v = !(F.v0 >= P.loy && F.v0 <= P.hiy);
        {   // min(max(u0, lo), hi) with the comparison order of std::min/std::max
            float t0 = (F.u0 < P.lox) ? P.lox : F.u0; F.u = (P.hix < t0) ? P.hix : t0;
            float t1 = (F.v0 < P.loy) ? P.loy : F.v0; F.v = (P.hiy < t1) ? P.hiy : t1;
        }
        const float J00 = P.fx / F.p[2], J11 = P.fy / F.p[2];
        const float J02 = -(J00 * F.u), J12 = -(J11 * F.v);
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            F.T[j] = J00 * W[j] + J02 * W[6 + j];
            F.T[3 + j] = J11 * W[3 + j] + J12 * W[6 + j];
        }
        float V[6];
#pragma unroll
        for (int r = 0; r < 2; ++r)
#pragma unroll
            for (int j = 0; j < 3; ++j)
                V[3 * r + j] = (F.T[3 * r] * F.Sig[j] + F.T[3 * r + 1] * F.Sig[3 + j]) + F.T[3 * r + 2] * F.Sig[6 + j];
        F.a = (V[0] * F.T[0] + V[1] * F.T[1]) + V[2] * F.T[2];
        F.b = (V[0] * F.T[3] + V[1] * F.T[4]) + V[2] * F.T[5];
        F.c = (V[3] * F.T[3] + V[4] * F.T[4]) + V[5] * F.T[5];
    } else {
        F.clamp_u = F.clamp_v = false;
        // 2*3+1 sigma points: mu, mu +- gamma s_j R[:,j]
#pragma unroll
        for (int k = 0; k < 7; ++k) {
            float sg[3];
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                if (k == 0) sg[d] = mu[d];
                else {
                    const int j = (k - 1) >> 1;
                    const float off = P.gamma * F.M[3 * d + j];
                    sg[d] = (k & 1) ? (mu[d] + off) : (mu[d] - off);
                }
            }
#pragma unroll
            for (int i = 0; i < 3; ++i)
                F.pc[k][i] = ((W[3 * i] * sg[0] + W[3 * i + 1] * sg[1]) + W[3 * i + 2] * sg[2]) + P.t[i];
            if (!(F.pc[k][2] > 0.0f)) return false;   // C18: a sigma point behind the camera
            camera_project(P, F.pc[k], F.y[k]);
        }
        float mx = P.wm0 * F.y[0][0], my = P.wm0 * F.y[0][1];
#pragma unroll
        for (int k = 1; k < 7; ++k) { mx = mx + P.wk * F.y[k][0]; my = my + P.wk * F.y[k][1]; }
        F.m[0] = mx; F.m[1] = my;
        float a = 0.0f, b = 0.0f, c = 0.0f;
#pragma unroll
        for (int k = 0; k < 7; ++k) {
            const float wc = (k == 0) ? P.wc0 : P.wk;
            const float dx = F.y[k][0] - mx, dy = F.y[k][1] - my;
            a = a + wc * (dx * dx); b = b + wc * (dx * dy); c = c + wc * (dy * dy);
        }
        F.a = a; F.b = b; F.c = c;
    }
    // low-pass (C4), determinant, conic
    F.ap = F.a + P.lowpass; F.cp = F.c + P.lowpass;
    F.det = F.ap * F.cp - F.b * F.b;
    if (!(F.det > 0.0f)) return false;
    F.det_raw = F.a * F.c - F.b * F.b;
    if (P.antialias) {   // C19
        const float ratio = F.det_raw / F.det;
        F.rho = sqrtf((0.0f < ratio) ? ratio : 0.0f);
        F.o_eff = o * F.rho;
    } else { F.rho = 1.0f; F.o_eff = o; }
    if (P.projection == 0) { if (!(F.o_eff >= P.alpha_thresh)) return false; }   // C9: >= for EWA (L262)
    else                   { if (!(F.o_eff >  P.alpha_thresh)) return false; }   //     >  for UT  (L482)
    F.A = F.cp / F.det; F.B = (-F.b) / F.det; F.C = F.ap / F.det;
    F.lnv = (float)log((double)F.o_eff / (double)P.alpha_thresh);               // R2
    const float ex = sqrtf((2.0f * F.lnv) * F.ap), ey = sqrtf((2.0f * F.lnv) * F.cp);   // C7
    if (!(((ex < ey) ? ey : ex) > 0.0f)) return false;
    const float ts = (float)TILE;
    F.rect[0] = (int)fmin(fmax(floorf((F.m[0] - ex) / ts), 0.0f), (float)P.TW);
    F.rect[1] = (int)fmin(fmax(floorf((F.m[1] - ey) / ts), 0.0f), (float)P.TH);
    F.rect[2] = (int)fmin(fmax(ceilf((F.m[0] + ex) / ts), 0.0f), (float)P.TW);
    F.rect[3] = (int)fmin(fmax(ceilf((F.m[1] + ey) / ts), 0.0f), (float)P.TH);
    const long long tc = (long long)(F.rect[2] - F.rect[0]) * (long long)(F.rect[3] - F.rect[1]);
    if (!(tc > 0)) return false;
    F.tc = (uint32_t)tc;
    return true;
}

// View direction and SH basis (C5).
__device__ __forceinline__ void view_dir(const ProjParams& P, const float mu[3], float dir[3], float& dnorm) {
    float dv[3];
#pragma unroll
    for (int j = 0; j < 3; ++j) dv[j] = mu[j] - P.cpos[j];
    dnorm = sqrtf((dv[0] * dv[0] + dv[1] * dv[1]) + dv[2] * dv[2]);
#pragma unroll
    for (int j = 0; j < 3; ++j) dir[j] = dv[j] / dnorm;
}

template <int K>
__device__ __forceinline__ void load_sh(const float* __restrict__ sh, int64_t i, float* c) {
    const float* p = sh + (int64_t)3 * K * i;
    if constexpr ((3 * K) % 4 == 0) {
        const float4* p4 = reinterpret_cast<const float4*>(p);
#pragma unroll
        for (int j = 0; j < (3 * K) / 4; ++j) {
            const float4 v = __ldg(p4 + j);
            c[4 * j] = v.x; c[4 * j + 1] = v.y; c[4 * j + 2] = v.z; c[4 * j + 3] = v.w;
        }
    } else {
#pragma unroll
        for (int j = 0; j < 3 * K; ++j) c[j] = __ldg(p + j);
    }
}

// Forward kernel.  Most Gaussians are culled (90 % in config 3: half of them lie behind the camera, most of the rest
// project outside the image), and the survivors are scattered, so one thread per Gaussian from start to end runs the
// long geometry and the 48-coefficient colour evaluation with a dozen active lanes per warp (measured: 12 of 32, the
// kernel was issue-bound on divergent code).  A CTA therefore owns PROJ_THREADS * PROJ_IPT consecutive Gaussians and
// works in three phases, each over a dense list in shared memory:
//   A  every Gaussian: camera-space depth of the mean, the z_near test (the first test of project_geometry);
//      survivors are compacted, the others get tile_count = flags = 0;
//   B  every survivor of A: the full geometry (EWA or UT), rectangle, visibility; visible ones are compacted and their
//      geometric outputs written, the others get tile_count = flags = 0;
//   C  every visible Gaussian: view direction, SH basis, colour (the only reader of the 192-byte SH row), flags and
//      the packed shader record.
// Every Gaussian runs exactly the arithmetic of the one-thread version (same functions, same inputs): the outputs
// are bit-identical.
// measured on config 3 (us), before the inputs were staged through shared memory: 128 threads x 2: 49.2; 128 x 4: 50.2; 256 x 8: 51.3; 256 x 2: 52.1; 256 x 4 (72 registers):
// 57.5; one thread per Gaussian without compaction: 48.5 -- the kernel is bound by the latency of its gathers, not by issue
#ifndef XPR_PROJ_THREADS
#define XPR_PROJ_THREADS 128
#endif
#ifndef XPR_PROJ_IPT
#define XPR_PROJ_IPT 2
#endif
#ifndef XPR_PROJ_MINB
#define XPR_PROJ_MINB 6
#endif
constexpr int PROJ_THREADS = XPR_PROJ_THREADS, PROJ_IPT = XPR_PROJ_IPT, PROJ_CHUNK = PROJ_THREADS * PROJ_IPT;

template <int K>
__global__ void __launch_bounds__(PROJ_THREADS, XPR_PROJ_MINB)
project_kernel(int64_t N, const __grid_constant__ ProjBatch PB, const float* __restrict__ means, const float* __restrict__ scales,
               const float* __restrict__ quats, const float* __restrict__ opac, const float* __restrict__ sh,
               float* __restrict__ mean2d, float* __restrict__ conic_opac, float* __restrict__ rgb,
               float* __restrict__ depth, float* __restrict__ lnv, int32_t* __restrict__ rect,
               uint32_t* __restrict__ tcount, uint8_t* __restrict__ flags, float4* __restrict__ shade_rec) {
    __shared__ uint16_t s_a[PROJ_CHUNK], s_b[PROJ_CHUNK];     // survivors of phase A / of phase B (offsets in the chunk)
    __shared__ uint8_t s_clamp[PROJ_CHUNK];                   // clamp bits of the visible ones (by position in s_b)
    __shared__ uint32_t s_na, s_nb;
    // batch of views (xpr_config.views): blockIdx.y is the view; its outputs live at index v N + i, its tile rows at v TH
    const ProjParams& P = PB.p[blockIdx.y];
    const int64_t vo = (int64_t)blockIdx.y * N;
    const int yoff = (int)blockIdx.y * P.TH;
    const int tid = threadIdx.x, lane = tid & 31;
    const int64_t base = (int64_t)blockIdx.x * PROJ_CHUNK;
    const int n_here = (int)min((int64_t)PROJ_CHUNK, N - base);
    if (tid == 0) { s_na = 0u; s_nb = 0u; }
    // ---- staging: the CTA's 44 input bytes per Gaussian (means, scales, quats, opacities: four contiguous runs) go to
    // shared memory with 16-byte cp.async, all in flight at once and without registers -- the per-thread loads of the
    // phases kept ~18 KB in flight per SM where latency x bandwidth asks for ~35 KB (the kernel was bound by the
    // latency of its loads at 1/3 of the DRAM peak).  Phases A and B then read shared memory only.
    __shared__ __align__(16) float s_mu[3 * PROJ_CHUNK], s_sc[3 * PROJ_CHUNK], s_q[4 * PROJ_CHUNK], s_o[PROJ_CHUNK];
    {
        const float* gm = means + 3 * base; const float* gs = scales + 3 * base;
        const float* gq = quats + 4 * base; const float* go = opac + base;
        const bool bulk = n_here == PROJ_CHUNK && ((reinterpret_cast<uintptr_t>(gm) | reinterpret_cast<uintptr_t>(gs) |
                                                    reinterpret_cast<uintptr_t>(gq) | reinterpret_cast<uintptr_t>(go)) & 15u) == 0;
        if (bulk) {
            for (int v = tid; v < 3 * PROJ_CHUNK / 4; v += PROJ_THREADS) { cp_async16(s_mu + 4 * v, gm + 4 * v); cp_async16(s_sc + 4 * v, gs + 4 * v); }
            for (int v = tid; v < PROJ_CHUNK; v += PROJ_THREADS) cp_async16(s_q + 4 * v, gq + 4 * v);
            for (int v = tid; v < PROJ_CHUNK / 4; v += PROJ_THREADS) cp_async16(s_o + 4 * v, go + 4 * v);
            cp_async_commit();
            cp_async_wait<0>();
        } else {        // last chunk or unaligned arrays: element by element
            for (int v = tid; v < 3 * n_here; v += PROJ_THREADS) { s_mu[v] = __ldg(gm + v); s_sc[v] = __ldg(gs + v); }
            for (int v = tid; v < 4 * n_here; v += PROJ_THREADS) s_q[v] = __ldg(gq + v);
            for (int v = tid; v < n_here; v += PROJ_THREADS) s_o[v] = __ldg(go + v);
        }
    }
    __syncthreads();
    const uint32_t lt = (1u << lane) - 1u;
    // ---- phase A ---------------------------------------------------------------------------------------------
#pragma unroll
    for (int k = 0; k < PROJ_IPT; ++k) {
        const int j = k * PROJ_THREADS + tid;
        bool keep = false;
        if (j < n_here) {
            const int64_t i = base + j;
            const float m0 = s_mu[3 * j], m1 = s_mu[3 * j + 1], m2 = s_mu[3 * j + 2];
            const float pz = ((P.W[6] * m0 + P.W[7] * m1) + P.W[8] * m2) + P.t[2];     // = F.p[2] of project_geometry
            keep = pz > P.z_near;
            if (!keep) { tcount[vo + i] = 0u; flags[vo + i] = 0; }
        }
        const uint32_t m = __ballot_sync(0xffffffffu, keep);
        uint32_t pos = 0;
        if (lane == 0 && m) pos = atomicAdd(&s_na, (uint32_t)__popc(m));
        pos = __shfl_sync(0xffffffffu, pos, 0);
        if (keep) s_a[pos + __popc(m & lt)] = (uint16_t)j;
    }
    __syncthreads();
    // ---- phase B ---------------------------------------------------------------------------------------------
    const int na = (int)s_na;
    for (int idx0 = 0; idx0 < na; idx0 += PROJ_THREADS) {
        const int idx = idx0 + tid;
        bool vis = false;
        Fwd F;
        int64_t i = 0;
        if (idx < na) {
            const int j = s_a[idx];
            i = base + j;
            const float mu[3] = {s_mu[3 * j], s_mu[3 * j + 1], s_mu[3 * j + 2]};
            const float sc[3] = {s_sc[3 * j], s_sc[3 * j + 1], s_sc[3 * j + 2]};
            const float4 q4 = reinterpret_cast<const float4*>(s_q)[j];
            const float q[4] = {q4.x, q4.y, q4.z, q4.w};
            vis = project_geometry(P, mu, sc, q, s_o[j], F);
            if (!vis) { tcount[vo + i] = 0u; flags[vo + i] = 0; }
        }
        const uint32_t m = __ballot_sync(0xffffffffu, vis);
        uint32_t pos = 0;
        if (lane == 0 && m) pos = atomicAdd(&s_nb, (uint32_t)__popc(m));
        pos = __shfl_sync(0xffffffffu, pos, 0);
        if (vis) {
            const uint32_t slot = pos + (uint32_t)__popc(m & lt);
            s_b[slot] = (uint16_t)(i - base);
            s_clamp[slot] = (uint8_t)((F.clamp_u ? XPR_FLAG_CLAMP_U : 0) | (F.clamp_v ? XPR_FLAG_CLAMP_V : 0));
            const int64_t o = vo + i;
            reinterpret_cast<float2*>(mean2d)[o] = make_float2(F.m[0], F.m[1]);
            reinterpret_cast<float4*>(conic_opac)[o] = make_float4(F.A, F.B, F.C, F.o_eff);
            depth[o] = F.p[2];
            lnv[o] = F.lnv;
            reinterpret_cast<int4*>(rect)[o] = make_int4(F.rect[0], F.rect[1] + yoff, F.rect[2], F.rect[3] + yoff);
            tcount[o] = F.tc;
        }
    }
    __syncthreads();           // also makes this CTA's geometric outputs visible to phase C
    // ---- phase C ---------------------------------------------------------------------------------------------
    const int nb = (int)s_nb;
    for (int idx = tid; idx < nb; idx += PROJ_THREADS) {
        const int jb = s_b[idx];
        const int64_t i = base + jb;
        const float mu[3] = {s_mu[3 * jb], s_mu[3 * jb + 1], s_mu[3 * jb + 2]};
        float dir[3], dnorm, Y[16];
        view_dir(P, mu, dir, dnorm);
        sh_basis(dir[0], dir[1], dir[2], Y);
        float c[3 * K];
        load_sh<K>(sh, i, c);      // (gathering the rows by the whole CTA through shared memory measured no faster: 47.1 vs 45.1 us)
        uint8_t fl = (uint8_t)(XPR_FLAG_VISIBLE | s_clamp[idx]);
        float col[3];
#pragma unroll
        for (int ch = 0; ch < 3; ++ch) {
            float acc = Y[0] * c[ch];
#pragma unroll
            for (int k = 1; k < K; ++k) acc = acc + Y[k] * c[3 * k + ch];
            const float raw = acc + 0.5f;
            col[ch] = (0.0f < raw) ? raw : 0.0f;
            if (raw > 0.0f) fl |= (uint8_t)(XPR_FLAG_RGB_POS_R << ch);
        }
        const int64_t o = vo + i;
        rgb[3 * o] = col[0]; rgb[3 * o + 1] = col[1]; rgb[3 * o + 2] = col[2];
        flags[o] = fl;
        if (shade_rec) {   // shader data p_sd as the compositing kernels read it: pre-scaled conic (C25, exact)
            const float2 m = reinterpret_cast<const float2*>(mean2d)[o];        // written in phase B by this CTA
            const float4 co = reinterpret_cast<const float4*>(conic_opac)[o];
            shade_rec[3 * o] = make_float4(m.x, m.y, -0.5f * co.x, -co.y);
            shade_rec[3 * o + 1] = make_float4(-0.5f * co.z, lnv[o], __log2f(co.w), depth[o]);
            shade_rec[3 * o + 2] = make_float4(col[0], col[1], col[2], co.w);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// XPR-LinPrim projection (PAPER A.1.3 L506-560, readings L1-L4 of DESIGN.md): octahedron
// {x : |S^-1 R^T (x - mu)|_1 <= 1} with homogeneous density sigma = -log(1 - 0.99 o) / (2 min s).  The linear map from
// the local frame to (pixel x, pixel y, Euclidean depth) is A = J W R diag(s), J = [d pixel / d p ; p^T / |p|]; the rows
// c0, c1, c2 of A^-1 give the four slab pairs n_i = c0 +- c1 +- c2 of the projected octahedron.  The record holds, per
// slab, kx = n_x / n_z, ky = n_y / n_z, h = 1 / |n_z|: tau in [m - h, m + h], m = -(kx dx + ky dy).  One thread per
// primitive; fp32, every operation individually rounded (this file is compiled with -fmad=false), order as the oracle's.
// lin_rec[N,20] = (mu2D 2, sigma, depth | (kx, ky, h) x 4 | r, g, b, 0).
// ---------------------------------------------------------------------------------------------
struct LinGeom {
    float p[3], dist, R[9], Bm[9], J[9], Ai[9], sigma, smin;
    int jmin;
};

// Geometry of one primitive, shared by the forward and the backward kernel (which recomputes it so that every culling
// decision is the forward's).  Returns visibility; rec[0..15], rc, tc are set when visible.
__device__ __forceinline__ bool lin_geometry(const ProjParams& P, const float mu[3], const float* __restrict__ scales,
                                             const float* __restrict__ quats, const float* __restrict__ opac, int64_t i,
                                             LinGeom& G, float rec[20], int4& rc, uint32_t& tc) {
    const float* W = P.W;
    float* p = G.p;
    for (int a = 0; a < 3; ++a) p[a] = ((W[3 * a] * mu[0] + W[3 * a + 1] * mu[1]) + W[3 * a + 2] * mu[2]) + P.t[a];
    bool vis = p[2] > P.z_near;
    rc = make_int4(0, 0, 0, 0);
    tc = 0;
    G.dist = 0.0f;
    if (!vis) return false;
    const float sc[3] = {__ldg(scales + 3 * i), __ldg(scales + 3 * i + 1), __ldg(scales + 3 * i + 2)};
    const float4 q4 = __ldg(reinterpret_cast<const float4*>(quats) + i);
    const float o = __ldg(opac + i);
    const float x = p[0], y = p[1], z = p[2];
    const float dist = sqrtf((x * x + y * y) + z * z);
    G.dist = dist;
    const float u = x / z, v = y / z;
    const float m0 = P.fx * u + P.cx, m1 = P.fy * v + P.cy;
    float* R = G.R;
    {
        const float w = q4.x, qx = q4.y, qy = q4.z, qz = q4.w;
        const float xx = qx * qx, yy = qy * qy, zz = qz * qz, xy = qx * qy, xz = qx * qz, yz = qy * qz;
        const float wx = w * qx, wy = w * qy, wz = w * qz;
        R[0] = 1.0f - 2.0f * (yy + zz); R[1] = 2.0f * (xy - wz); R[2] = 2.0f * (xz + wy);
        R[3] = 2.0f * (xy + wz); R[4] = 1.0f - 2.0f * (xx + zz); R[5] = 2.0f * (yz - wx);
        R[6] = 2.0f * (xz - wy); R[7] = 2.0f * (yz + wx); R[8] = 1.0f - 2.0f * (xx + yy);
    }
    float* Bm = G.Bm;
    float A[9];
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) {
            const float r0 = R[b] * sc[b], r1 = R[3 + b] * sc[b], r2 = R[6 + b] * sc[b];
            Bm[3 * a + b] = (W[3 * a] * r0 + W[3 * a + 1] * r1) + W[3 * a + 2] * r2;
        }
    const float j00 = P.fx / z, j11 = P.fy / z;
    float* J = G.J;
    J[0] = j00; J[1] = 0.0f; J[2] = -(j00 * u); J[3] = 0.0f; J[4] = j11; J[5] = -(j11 * v);
    J[6] = x / dist; J[7] = y / dist; J[8] = z / dist;
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b)
            A[3 * a + b] = (J[3 * a] * Bm[b] + J[3 * a + 1] * Bm[3 + b]) + J[3 * a + 2] * Bm[6 + b];
    float cof[9];
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) {
            const int a1 = (a + 1) % 3, a2 = (a + 2) % 3, b1 = (b + 1) % 3, b2 = (b + 2) % 3;
            cof[3 * a + b] = A[3 * a1 + b1] * A[3 * a2 + b2] - A[3 * a1 + b2] * A[3 * a2 + b1];
        }
    const float det = (A[0] * cof[0] + A[1] * cof[1]) + A[2] * cof[2];
    vis = (fabsf(det) > 0.0f) && isfinite(det);
    float* Ai = G.Ai;
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) Ai[3 * a + b] = cof[3 * b + a] / det;
    const float smin = fminf(sc[0], fminf(sc[1], sc[2]));
    G.smin = smin;
    G.jmin = (sc[0] == smin) ? 0 : (sc[1] == smin) ? 1 : 2;
    const float sigma = (float)(-log(1.0 - 0.99 * (double)o) / (2.0 * (double)smin));     // R2
    G.sigma = sigma;
    vis = vis && (sigma > 0.0f) && isfinite(sigma);
    const float ex = fmaxf(fabsf(A[0]), fmaxf(fabsf(A[1]), fabsf(A[2])));
    const float ey = fmaxf(fabsf(A[3]), fmaxf(fabsf(A[4]), fabsf(A[5])));
    vis = vis && (fmaxf(ex, ey) > 0.0f);
    if (vis) {
        const float ts = (float)TILE;
        rc.x = (int)fminf(fmaxf(floorf((m0 - ex) / ts), 0.0f), (float)P.TW);
        rc.y = (int)fminf(fmaxf(floorf((m1 - ey) / ts), 0.0f), (float)P.TH);
        rc.z = (int)fminf(fmaxf(ceilf((m0 + ex) / ts), 0.0f), (float)P.TW);
        rc.w = (int)fminf(fmaxf(ceilf((m1 + ey) / ts), 0.0f), (float)P.TH);
        const long long t2 = (long long)(rc.z - rc.x) * (long long)(rc.w - rc.y);
        vis = t2 > 0;
        tc = (uint32_t)t2;
    }
    if (vis) {
        rec[0] = m0; rec[1] = m1; rec[2] = sigma; rec[3] = dist;
#pragma unroll
        for (int s = 0; s < 4; ++s) {
            const bool p1 = s < 2, p2 = (s & 1) == 0;
            float n[3];
#pragma unroll
            for (int k = 0; k < 3; ++k) n[k] = (Ai[k] + (p1 ? Ai[3 + k] : -Ai[3 + k])) + (p2 ? Ai[6 + k] : -Ai[6 + k]);
            float kx = 0.0f, ky = 0.0f, h = INFINITY;                                  // L4
            if (fabs((double)n[2]) >= 1e-12) { const float inv = 1.0f / n[2]; kx = n[0] * inv; ky = n[1] * inv; h = fabsf(inv); }
            rec[4 + 3 * s] = kx; rec[5 + 3 * s] = ky; rec[6 + 3 * s] = h;
        }
#pragma unroll
        for (int k = 0; k < 16; ++k)
            if (!isfinite(rec[k]) && !(k >= 4 && (k - 4) % 3 == 2)) vis = false;
    }
    return vis;
}

template <int K>
__global__ void __launch_bounds__(128)
lin_project_kernel(int64_t N, ProjParams P, const float* __restrict__ means, const float* __restrict__ scales,
                   const float* __restrict__ quats, const float* __restrict__ opac, const float* __restrict__ sh,
                   float4* __restrict__ lin_rec, float* __restrict__ depth, int32_t* __restrict__ rect,
                   uint32_t* __restrict__ tcount) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const float mu[3] = {__ldg(means + 3 * i), __ldg(means + 3 * i + 1), __ldg(means + 3 * i + 2)};
    float rec[20];
    int4 rc;
    uint32_t tc;
    LinGeom G;
    const bool vis = lin_geometry(P, mu, scales, quats, opac, i, G, rec, rc, tc);
    const float dist = G.dist;
    if (!vis) {          // culled: an all-zero record (xpr.h)
#pragma unroll
        for (int k = 0; k < 5; ++k) lin_rec[5 * i + k] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        depth[i] = 0.0f;
        reinterpret_cast<int4*>(rect)[i] = make_int4(0, 0, 0, 0);
        tcount[i] = 0u;
        return;
    }
    float dir[3], dnorm, Y[16];
    view_dir(P, mu, dir, dnorm);
    sh_basis(dir[0], dir[1], dir[2], Y);
    float c[3 * K];
    load_sh<K>(sh, i, c);
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) {
        float acc = Y[0] * c[ch];
#pragma unroll
        for (int k = 1; k < K; ++k) acc = acc + Y[k] * c[3 * k + ch];
        const float raw = acc + 0.5f;
        rec[16 + ch] = (0.0f < raw) ? raw : 0.0f;
    }
    rec[19] = 0.0f;
#pragma unroll
    for (int k = 0; k < 5; ++k) lin_rec[5 * i + k] = make_float4(rec[4 * k], rec[4 * k + 1], rec[4 * k + 2], rec[4 * k + 3]);
    depth[i] = dist;
    reinterpret_cast<int4*>(rect)[i] = rc;
    tcount[i] = tc;
}

// ---------------------------------------------------------------------------------------------
// Backward.  The forward intermediates are recomputed in fp32 exactly as above (so the clamp and
// culling decisions are the forward's); the chain rule itself runs in fp64 (the kernel is HBM- and
// latency-bound, not bound by the FP64 pipe, which runs at half the fp32 rate on B200), which keeps the ill-conditioned conic -> covariance
// step (G2 = -K G_K K) inside the 1e-3 relative gradient tolerance.
// ---------------------------------------------------------------------------------------------
typedef double B;

__device__ __forceinline__ void sh_basis_grad(B x, B y, B z, B dY[16][3]) {
    const B c1 = 0.4886025119029199, a2 = 1.0925484305920792, b2 = 0.31539156525252005, c2 = 0.5462742152960396;
    const B a3 = 0.5900435899266435, b3 = 2.890611442640554, c3 = 0.4570457994644658, d3 = 0.3731763325901154,
            e3 = 1.445305721320277;
    const B xx = x * x, yy = y * y, zz = z * z, xy = x * y, yz = y * z, xz = x * z;
#pragma unroll
    for (int k = 0; k < 16; ++k) dY[k][0] = dY[k][1] = dY[k][2] = 0;
    dY[1][1] = -c1; dY[2][2] = c1; dY[3][0] = -c1;
    dY[4][0] = a2 * y; dY[4][1] = a2 * x;
    dY[5][1] = -a2 * z; dY[5][2] = -a2 * y;
    dY[6][0] = -2 * b2 * x; dY[6][1] = -2 * b2 * y; dY[6][2] = 4 * b2 * z;
    dY[7][0] = -a2 * z; dY[7][2] = -a2 * x;
    dY[8][0] = 2 * c2 * x; dY[8][1] = -2 * c2 * y;
    dY[9][0] = -6 * a3 * xy; dY[9][1] = -3 * a3 * (xx - yy);
    dY[10][0] = b3 * yz; dY[10][1] = b3 * xz; dY[10][2] = b3 * xy;
    dY[11][0] = 2 * c3 * xy; dY[11][1] = -c3 * (4 * zz - xx - 3 * yy); dY[11][2] = -8 * c3 * yz;
    dY[12][0] = -6 * d3 * xz; dY[12][1] = -6 * d3 * yz; dY[12][2] = 3 * d3 * (2 * zz - xx - yy);
    dY[13][0] = -c3 * (4 * zz - 3 * xx - yy); dY[13][1] = 2 * c3 * xy; dY[13][2] = -8 * c3 * xz;
    dY[14][0] = 2 * e3 * xz; dY[14][1] = -2 * e3 * yz; dY[14][2] = e3 * (xx - yy);
    dY[15][0] = -3 * a3 * (xx - yy); dY[15][1] = 6 * a3 * xy;
}

// d pix / d p of the camera model (2x3).
__device__ __forceinline__ void camera_jac(const ProjParams& P, const B p[3], B Jp[2][3]) {
    const B x = p[0], y = p[1], z = p[2], fx = P.fx, fy = P.fy;
    if (P.model == 0) {
        Jp[0][0] = fx / z; Jp[0][1] = 0; Jp[0][2] = -fx * x / (z * z);
        Jp[1][0] = 0; Jp[1][1] = fy / z; Jp[1][2] = -fy * y / (z * z);
        return;
    }
    const B r2 = x * x + y * y, r = sqrt(r2);
    if (!(r > 0)) {
        Jp[0][0] = fx / z; Jp[0][1] = 0; Jp[0][2] = 0;
        Jp[1][0] = 0; Jp[1][1] = fy / z; Jp[1][2] = 0;
        return;
    }
    const B th = atan2(r, z), t2 = th * th;
    const B k1 = P.k[0], k2 = P.k[1], k3 = P.k[2], k4 = P.k[3];
    const B thd = th * (1.0 + t2 * (k1 + t2 * (k2 + t2 * (k3 + t2 * k4))));
    const B dthd = 1.0 + t2 * (3 * k1 + t2 * (5 * k2 + t2 * (7 * k3 + t2 * 9 * k4)));
    const B inv = 1.0 / (r2 + z * z);
    const B dth_dr = z * inv, dth_dz = -r * inv;
    const B s = thd / r;
    const B ds_dr = (dthd * dth_dr * r - thd) / r2;
    const B ds_dz = dthd * dth_dz / r;
    const B ds_dx = ds_dr * x / r, ds_dy = ds_dr * y / r;
    Jp[0][0] = fx * (s + x * ds_dx); Jp[0][1] = fx * x * ds_dy; Jp[0][2] = fx * x * ds_dz;
    Jp[1][0] = fy * y * ds_dx; Jp[1][1] = fy * (s + y * ds_dy); Jp[1][2] = fy * y * ds_dz;
}

template <int K>
__device__ __forceinline__ void store_sh_grad(float* __restrict__ g_sh, int64_t i, const float* g, bool accum = false) {
    float* p = g_sh + (int64_t)3 * K * i;
    if (accum) {       // batch of views: the views' contributions are summed (fp32 atomics; at most XPR_MAX_VIEWS terms)
#pragma unroll
        for (int j = 0; j < 3 * K; ++j)
            if (g[j] != 0.0f) atomicAdd(p + j, g[j]);
        return;
    }
    if constexpr ((3 * K) % 4 == 0) {
        float4* p4 = reinterpret_cast<float4*>(p);
#pragma unroll
        for (int j = 0; j < (3 * K) / 4; ++j) p4[j] = make_float4(g[4 * j], g[4 * j + 1], g[4 * j + 2], g[4 * j + 3]);
    } else {
#pragma unroll
        for (int j = 0; j < 3 * K; ++j) p[j] = g[j];
    }
}

// One visible Gaussian: recompute the forward, chain rule in fp64, store its 59 gradient floats.
template <int K>
__device__ __forceinline__ void project_bwd_one(int64_t i, int64_t vo, bool accum, const ProjParams& P, const float* __restrict__ means,
                                                const float* __restrict__ scales, const float* __restrict__ quats,
                                                const float* __restrict__ opac, const float* __restrict__ sh,
                                                const uint8_t* __restrict__ flags, const float* __restrict__ g_mean2d,
                                                const float* __restrict__ g_conic, const float* __restrict__ g_opac,
                                                const float* __restrict__ g_rgb, float* __restrict__ g_means,
                                                float* __restrict__ g_scales, float* __restrict__ g_quats,
                                                float* __restrict__ g_opacities, float* __restrict__ g_sh) {
    B g_mu[3] = {0, 0, 0}, g_s[3] = {0, 0, 0}, g_q[4] = {0, 0, 0, 0}, g_o = 0;
    // every load of this Gaussian is issued up front (the kernel is latency-bound: DESIGN.md 6.1)
    const uint8_t fl = flags[vo + i];        // per-view quantities live at v N + i (xpr_config.views)
    Fwd F;
    float mu[3], sc[3], q[4], o;
    mu[0] = __ldg(means + 3 * i); mu[1] = __ldg(means + 3 * i + 1); mu[2] = __ldg(means + 3 * i + 2);
    sc[0] = __ldg(scales + 3 * i); sc[1] = __ldg(scales + 3 * i + 1); sc[2] = __ldg(scales + 3 * i + 2);
    const float4 q4 = __ldg(reinterpret_cast<const float4*>(quats) + i);
    q[0] = q4.x; q[1] = q4.y; q[2] = q4.z; q[3] = q4.w;
    o = __ldg(opac + i);
    const int64_t vi = vo + i;
    const float2 gm_f = __ldg(reinterpret_cast<const float2*>(g_mean2d) + vi);
    const float gK_f[3] = {__ldg(g_conic + 3 * vi), __ldg(g_conic + 3 * vi + 1), __ldg(g_conic + 3 * vi + 2)};
    const float go_f = __ldg(g_opac + vi);
    const float grgb_f[3] = {__ldg(g_rgb + 3 * vi), __ldg(g_rgb + 3 * vi + 1), __ldg(g_rgb + 3 * vi + 2)};
    {   // colour first: rgb = max(0, 1/2 + sum_k Y_k(d) sh_k), d = (mu - cam_pos)/|mu - cam_pos|.  Its 3K
        // coefficient gradients are stored at once, so they do not occupy registers during the chain rule.
        float c[3 * K];
        load_sh<K>(sh, i, c);
        float dir[3], dnorm, Y[16];
        view_dir(P, mu, dir, dnorm);
        sh_basis(dir[0], dir[1], dir[2], Y);
        B dY[16][3];
        sh_basis_grad((B)dir[0], (B)dir[1], (B)dir[2], dY);
        B gd[3] = {0, 0, 0};
        float gsh[3 * K];
        // C16 mask saved by the forward; dL/dd = sum_k grad Y_k(d) w_k with w_k = sum_ch sh[k][ch] g_ch (three fp32
        // products per coefficient), accumulated over k in fp64
        const float gr = (fl & XPR_FLAG_RGB_POS_R) ? grgb_f[0] : 0.0f, gg = (fl & XPR_FLAG_RGB_POS_G) ? grgb_f[1] : 0.0f,
                    gb = (fl & XPR_FLAG_RGB_POS_B) ? grgb_f[2] : 0.0f;
#pragma unroll
        for (int k = 0; k < K; ++k) {
            gsh[3 * k] = Y[k] * gr; gsh[3 * k + 1] = Y[k] * gg; gsh[3 * k + 2] = Y[k] * gb;
            const B w = (B)fmaf(c[3 * k], gr, fmaf(c[3 * k + 1], gg, c[3 * k + 2] * gb));
#pragma unroll
            for (int j = 0; j < 3; ++j) gd[j] += dY[k][j] * w;
        }
        store_sh_grad<K>(g_sh, i, gsh, accum);
        const B dot = (B)dir[0] * gd[0] + (B)dir[1] * gd[1] + (B)dir[2] * gd[2];
#pragma unroll
        for (int j = 0; j < 3; ++j) g_mu[j] = (gd[j] - (B)dir[j] * dot) / (B)dnorm;
    }
    const bool vis = project_geometry(P, mu, sc, q, o, F);   // recompute; same decisions as forward
    if (vis) {
        const B gm[2] = {(B)gm_f.x, (B)gm_f.y};
        const B gK[3] = {(B)gK_f[0], (B)gK_f[1], (B)gK_f[2]};
        const B go_eff = (B)go_f;
        const float* W = P.W;
        // conic -> filtered covariance: G2 = -K G_K K (symmetric-matrix gradients)
        const B A = F.A, Bc = F.B, C = F.C;
        const B GK[2][2] = {{gK[0], 0.5 * gK[1]}, {0.5 * gK[1], gK[2]}};
        const B Km[2][2] = {{A, Bc}, {Bc, C}};
        B tmp[2][2], G2[2][2];
#pragma unroll
        for (int r = 0; r < 2; ++r)
#pragma unroll
            for (int j = 0; j < 2; ++j) tmp[r][j] = Km[r][0] * GK[0][j] + Km[r][1] * GK[1][j];
#pragma unroll
        for (int r = 0; r < 2; ++r)
#pragma unroll
            for (int j = 0; j < 2; ++j) G2[r][j] = -(tmp[r][0] * Km[0][j] + tmp[r][1] * Km[1][j]);
        B g_a = G2[0][0], g_b = 2.0 * G2[0][1], g_c = G2[1][1];
        if (P.antialias) {   // C19
            const B rho = F.rho;
            g_o = go_eff * rho;
            if (rho > 0.0) {
                const B g_rho = go_eff * (B)o;
                const B g_draw = g_rho * 0.5 * rho / (B)F.det_raw, g_det = -g_rho * 0.5 * rho / (B)F.det;
                g_a += g_draw * (B)F.c + g_det * (B)F.cp;
                g_c += g_draw * (B)F.a + g_det * (B)F.ap;
                g_b += -2.0 * (B)F.b * (g_draw + g_det);
            }
        } else g_o = go_eff;
        const B Gs[2][2] = {{g_a, 0.5 * g_b}, {0.5 * g_b, g_c}};
        B gM[3][3];
        if (P.projection == 0) {
            // dL/dSigma = T^T Gs T ; dL/dT = 2 Gs T Sigma ; dL/dJ = dL/dT W^T
            B GT[2][3];
#pragma unroll
            for (int r = 0; r < 2; ++r)
#pragma unroll
                for (int j = 0; j < 3; ++j) GT[r][j] = Gs[r][0] * (B)F.T[j] + Gs[r][1] * (B)F.T[3 + j];
            B gSig[3][3];
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int j = 0; j < 3; ++j) gSig[a][j] = (B)F.T[a] * GT[0][j] + (B)F.T[3 + a] * GT[1][j];
            B gT[2][3];
#pragma unroll
            for (int r = 0; r < 2; ++r)
#pragma unroll
                for (int j = 0; j < 3; ++j)
                    gT[r][j] = 2.0 * (GT[r][0] * (B)F.Sig[j] + GT[r][1] * (B)F.Sig[3 + j] + GT[r][2] * (B)F.Sig[6 + j]);
            B gJ[2][3];
#pragma unroll
            for (int r = 0; r < 2; ++r)
#pragma unroll
                for (int j = 0; j < 3; ++j)
                    gJ[r][j] = gT[r][0] * (B)W[3 * j] + gT[r][1] * (B)W[3 * j + 1] + gT[r][2] * (B)W[3 * j + 2];
            const B x = F.p[0], y = F.p[1], z = F.p[2], fx = P.fx, fy = P.fy, u = F.u, v = F.v;
            const B iz = 1.0 / z, iz2 = iz * iz;
            B g_p[3] = {0, 0, 0};
            g_p[2] += gJ[0][0] * (-fx * iz2) + gJ[1][1] * (-fy * iz2);
            g_p[2] += gJ[0][2] * (fx * u * iz2) + gJ[1][2] * (fy * v * iz2);
            const B g_u = gJ[0][2] * (-fx * iz), g_v = gJ[1][2] * (-fy * iz);
            if (!F.clamp_u) { g_p[0] += g_u * iz; g_p[2] += -g_u * x * iz2; }   // C16
            if (!F.clamp_v) { g_p[1] += g_v * iz; g_p[2] += -g_v * y * iz2; }
            g_p[0] += gm[0] * fx * iz; g_p[1] += gm[1] * fy * iz;
            g_p[2] += -gm[0] * fx * x * iz2 - gm[1] * fy * y * iz2;
#pragma unroll
            for (int j = 0; j < 3; ++j) g_mu[j] += (B)W[j] * g_p[0] + (B)W[3 + j] * g_p[1] + (B)W[6 + j] * g_p[2];
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int j = 0; j < 3; ++j)
                    gM[a][j] = 2.0 * (gSig[a][0] * (B)F.M[j] + gSig[a][1] * (B)F.M[3 + j] + gSig[a][2] * (B)F.M[6 + j]);
        } else {
            // UT: m = sum wm_k y_k ; cov = sum wc_k (y_k - m)(y_k - m)^T
            B gtot[2] = {gm[0], gm[1]};
            B dk[7][2], Gd[7][2];
#pragma unroll
            for (int k = 0; k < 7; ++k) {
                const B wc = (k == 0) ? (B)P.wc0 : (B)P.wk;
                dk[k][0] = (B)F.y[k][0] - (B)F.m[0]; dk[k][1] = (B)F.y[k][1] - (B)F.m[1];
#pragma unroll
                for (int r = 0; r < 2; ++r) {
                    Gd[k][r] = 2.0 * wc * (Gs[r][0] * dk[k][0] + Gs[r][1] * dk[k][1]);
                    gtot[r] -= Gd[k][r];
                }
            }
            B gx[7][3];
#pragma unroll
            for (int k = 0; k < 7; ++k) {
                const B wm = (k == 0) ? (B)P.wm0 : (B)P.wk;
                const B gy[2] = {wm * gtot[0] + Gd[k][0], wm * gtot[1] + Gd[k][1]};
                const B pc[3] = {(B)F.pc[k][0], (B)F.pc[k][1], (B)F.pc[k][2]};
                B Jp[2][3];
                camera_jac(P, pc, Jp);
                B gpc[3];
#pragma unroll
                for (int j = 0; j < 3; ++j) gpc[j] = Jp[0][j] * gy[0] + Jp[1][j] * gy[1];
#pragma unroll
                for (int j = 0; j < 3; ++j) {
                    gx[k][j] = (B)W[j] * gpc[0] + (B)W[3 + j] * gpc[1] + (B)W[6 + j] * gpc[2];
                    g_mu[j] += gx[k][j];
                }
            }
#pragma unroll
            for (int j = 0; j < 3; ++j)
#pragma unroll
                for (int d = 0; d < 3; ++d) gM[d][j] = (B)P.gamma * (gx[1 + 2 * j][d] - gx[2 + 2 * j][d]);
        }
        // M = R diag(s); R(q) with four free components (C17)
        B gR[3][3];
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int j = 0; j < 3; ++j) { g_s[j] += (B)F.R[3 * a + j] * gM[a][j]; gR[a][j] = (B)sc[j] * gM[a][j]; }
        {
            const B w = q[0], x = q[1], y = q[2], z = q[3];
            g_q[0] = 2.0 * (-z * gR[0][1] + y * gR[0][2] + z * gR[1][0] - x * gR[1][2] - y * gR[2][0] + x * gR[2][1]);
            g_q[1] = 2.0 * (y * gR[0][1] + z * gR[0][2] + y * gR[1][0] - 2.0 * x * gR[1][1] - w * gR[1][2] + z * gR[2][0] + w * gR[2][1] - 2.0 * x * gR[2][2]);
            g_q[2] = 2.0 * (-2.0 * y * gR[0][0] + x * gR[0][1] + w * gR[0][2] + x * gR[1][0] + z * gR[1][2] - w * gR[2][0] + z * gR[2][1] - 2.0 * y * gR[2][2]);
            g_q[3] = 2.0 * (-2.0 * z * gR[0][0] - w * gR[0][1] + x * gR[0][2] + w * gR[1][0] - 2.0 * z * gR[1][1] + y * gR[1][2] + x * gR[2][0] + y * gR[2][1]);
        }
    } else {   // cannot happen for a Gaussian the forward flagged visible (same arithmetic); keep the contract anyway
        float z[3 * K];
#pragma unroll
        for (int j = 0; j < 3 * K; ++j) z[j] = 0.0f;
        if (!accum) store_sh_grad<K>(g_sh, i, z);
        g_mu[0] = g_mu[1] = g_mu[2] = 0;
    }
    if (accum) {
#pragma unroll
        for (int j = 0; j < 3; ++j) { atomicAdd(g_means + 3 * i + j, (float)g_mu[j]); atomicAdd(g_scales + 3 * i + j, (float)g_s[j]); }
#pragma unroll
        for (int j = 0; j < 4; ++j) atomicAdd(g_quats + 4 * i + j, (float)g_q[j]);
        atomicAdd(g_opacities + i, (float)g_o);
        return;
    }
    g_means[3 * i] = (float)g_mu[0]; g_means[3 * i + 1] = (float)g_mu[1]; g_means[3 * i + 2] = (float)g_mu[2];
    g_scales[3 * i] = (float)g_s[0]; g_scales[3 * i + 1] = (float)g_s[1]; g_scales[3 * i + 2] = (float)g_s[2];
    reinterpret_cast<float4*>(g_quats)[i] = make_float4((float)g_q[0], (float)g_q[1], (float)g_q[2], (float)g_q[3]);
    g_opacities[i] = (float)g_o;
}

// Backward kernel.  Only a fraction of the Gaussians is visible (10 % in config 3, view 0) and they are
// scattered, so one thread per Gaussian would run the heavy chain rule with a handful of active lanes
// per warp.  Each CTA therefore owns PBWD_THREADS * ipt consecutive Gaussians: (1) it reads tile_count
// coalesced and compacts the visible indices into shared memory, (2) it runs the chain rule over the dense
// list.  The zeros of the culled Gaussians come from a cudaMemsetAsync issued by xpr_project_bwd before the
// launch (236 B per Gaussian at K = 16: most of the call's bytes, moved at fill bandwidth).
constexpr int PBWD_THREADS = 128, PBWD_MAX_IPT = 16;

#ifndef XPR_PBWD_MINB
#define XPR_PBWD_MINB 3
#endif
template <int K>
__global__ void __launch_bounds__(PBWD_THREADS, XPR_PBWD_MINB)
project_bwd_kernel(int64_t N, const __grid_constant__ ProjBatch PB, int ipt, const float* __restrict__ means, const float* __restrict__ scales,
                   const float* __restrict__ quats, const float* __restrict__ opac, const float* __restrict__ sh,
                   const uint32_t* __restrict__ tcount, const uint8_t* __restrict__ flags,
                   const float* __restrict__ g_mean2d, const float* __restrict__ g_conic,
                   const float* __restrict__ g_opac, const float* __restrict__ g_rgb, float* __restrict__ g_means,
                   float* __restrict__ g_scales, float* __restrict__ g_quats, float* __restrict__ g_opacities,
                   float* __restrict__ g_sh) {
    __shared__ uint16_t s_list[PBWD_THREADS * PBWD_MAX_IPT];
    __shared__ uint32_t s_cnt;
    const ProjParams& P = PB.p[blockIdx.y];            // batch of views: blockIdx.y is the view
    const int64_t vo = (int64_t)blockIdx.y * N;
    const bool accum = gridDim.y > 1;
    const int tid = threadIdx.x, lane = tid & 31;
    const int chunk = PBWD_THREADS * ipt;
    const int64_t base = (int64_t)blockIdx.x * chunk;
    const int n_here = (int)min((int64_t)chunk, N - base);
    if (tid == 0) s_cnt = 0u;
    __syncthreads();
    uint32_t tc[PBWD_MAX_IPT];                           // independent loads first (tile_count != 0 <=> visible)
#pragma unroll
    for (int k = 0; k < PBWD_MAX_IPT; ++k) {
        const int j = k * PBWD_THREADS + tid;
        tc[k] = (k < ipt && j < n_here) ? __ldg(tcount + vo + base + j) : 0u;
    }
    uint32_t vbits = 0;
#pragma unroll
    for (int k = 0; k < PBWD_MAX_IPT; ++k) vbits |= (tc[k] != 0u ? 1u : 0u) << k;
    for (int k = 0; k < ipt; ++k) {
        const int j = k * PBWD_THREADS + tid;
        const bool vis = (vbits >> k) & 1u;
        const uint32_t m = __ballot_sync(0xffffffffu, vis);
        uint32_t pos = 0;
        if (lane == 0 && m) pos = atomicAdd(&s_cnt, (uint32_t)__popc(m));
        pos = __shfl_sync(0xffffffffu, pos, 0);
        if (vis) s_list[pos + __popc(m & ((1u << lane) - 1u))] = (uint16_t)j;
    }
    __syncthreads();
    const int cnt = (int)s_cnt;
    // (the outputs were zero-filled by the host side of the call with cudaMemsetAsync -- a full-bandwidth fill instead of
    // zero stores issued from this 168-register, low-occupancy kernel: 236 B per culled Gaussian are 70 % of the bytes
    // of the call at 10 % visibility)
    for (int idx = tid; idx < cnt; idx += PBWD_THREADS)
        project_bwd_one<K>(base + s_list[idx], vo, accum, P, means, scales, quats, opac, sh, flags, g_mean2d, g_conic, g_opac,
                           g_rgb, g_means, g_scales, g_quats, g_opacities, g_sh);
}

// XPR-LinPrim projection backward (f4): dL/d(lin_rec) [N,20] -> parameter gradients.  One thread per primitive; the forward
// geometry is recomputed in fp32 exactly as lin_project_kernel does (same culling, same slabs), the chain rule runs in
// fp64:
//   slabs (kx, ky, h) -> n = c0 + e1 c1 + e2 c2 -> A^-1;  dL/dA = -A^-T (dL/dA^-1) A^-T;  A = J B: dL/dJ = dL/dA B^T,
//   dL/dB = J^T dL/dA;  B = W R diag(s);  sigma(o, min s);  J(p) and mu2D -> p = W mu + t;  colour as project_bwd.
// Every primitive's outputs are written (zeros when culled): no zero-fill, no atomics.
template <int K>
__global__ void __launch_bounds__(128)
lin_project_bwd_kernel(int64_t N, ProjParams P, const float* __restrict__ means, const float* __restrict__ scales,
                       const float* __restrict__ quats, const float* __restrict__ opac, const float* __restrict__ sh,
                       const uint32_t* __restrict__ tcount, const float4* __restrict__ lin_rec,
                       const float4* __restrict__ g_rec, float* __restrict__ g_means, float* __restrict__ g_scales,
                       float* __restrict__ g_quats, float* __restrict__ g_opacities, float* __restrict__ g_sh) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    B g_mu[3] = {0, 0, 0}, g_s[3] = {0, 0, 0}, g_q[4] = {0, 0, 0, 0}, g_o = 0;
    const float mu[3] = {__ldg(means + 3 * i), __ldg(means + 3 * i + 1), __ldg(means + 3 * i + 2)};
    float rec[20];
    int4 rc;
    uint32_t tc;
    LinGeom G;
    const bool vis = (tcount[i] != 0u) && lin_geometry(P, mu, scales, quats, opac, i, G, rec, rc, tc);
    if (!vis) {
        float z[3 * K];
#pragma unroll
        for (int j = 0; j < 3 * K; ++j) z[j] = 0.0f;
        store_sh_grad<K>(g_sh, i, z);
    } else {
        float gr[20];
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            const float4 v = __ldg(g_rec + 5 * i + k);
            gr[4 * k] = v.x; gr[4 * k + 1] = v.y; gr[4 * k + 2] = v.z; gr[4 * k + 3] = v.w;
        }
        {   // colour (C5, C16): the forward's clamp decision is the stored colour itself
            const float4 col = __ldg(lin_rec + 5 * i + 4);
            float c[3 * K];
            load_sh<K>(sh, i, c);
            float dir[3], dnorm, Y[16];
            view_dir(P, mu, dir, dnorm);
            sh_basis(dir[0], dir[1], dir[2], Y);
            B dY[16][3];
            sh_basis_grad((B)dir[0], (B)dir[1], (B)dir[2], dY);
            B gd[3] = {0, 0, 0};
            float gsh[3 * K];
            const float g0 = (col.x > 0.0f) ? gr[16] : 0.0f, g1 = (col.y > 0.0f) ? gr[17] : 0.0f, g2 = (col.z > 0.0f) ? gr[18] : 0.0f;
#pragma unroll
            for (int k = 0; k < K; ++k) {
                gsh[3 * k] = Y[k] * g0; gsh[3 * k + 1] = Y[k] * g1; gsh[3 * k + 2] = Y[k] * g2;
                const B w = (B)fmaf(c[3 * k], g0, fmaf(c[3 * k + 1], g1, c[3 * k + 2] * g2));
#pragma unroll
                for (int j = 0; j < 3; ++j) gd[j] += dY[k][j] * w;
            }
            store_sh_grad<K>(g_sh, i, gsh);
            const B dot = (B)dir[0] * gd[0] + (B)dir[1] * gd[1] + (B)dir[2] * gd[2];
#pragma unroll
            for (int j = 0; j < 3; ++j) g_mu[j] = (gd[j] - (B)dir[j] * dot) / (B)dnorm;
        }
        B Ai[3][3], gAi[3][3];
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b) { Ai[a][b] = (B)G.Ai[3 * a + b]; gAi[a][b] = 0; }
#pragma unroll
        for (int s = 0; s < 4; ++s) {
            const B e1 = (s < 2) ? 1.0 : -1.0, e2 = ((s & 1) == 0) ? 1.0 : -1.0;
            B n[3];
#pragma unroll
            for (int k = 0; k < 3; ++k) n[k] = Ai[0][k] + e1 * Ai[1][k] + e2 * Ai[2][k];
            if (!(fabs(n[2]) >= 1e-12)) continue;                                 // L4: constants
            const B inv = 1.0 / n[2], gkx = (B)gr[4 + 3 * s], gky = (B)gr[5 + 3 * s], gh = (B)gr[6 + 3 * s];
            const B gn[3] = {gkx * inv, gky * inv, -(gkx * n[0] + gky * n[1]) * inv * inv - gh * (n[2] > 0 ? 1.0 : -1.0) * inv * inv};
#pragma unroll
            for (int k = 0; k < 3; ++k) { gAi[0][k] += gn[k]; gAi[1][k] += e1 * gn[k]; gAi[2][k] += e2 * gn[k]; }
        }
        B tmp[3][3], gA[3][3];
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b) tmp[a][b] = Ai[0][a] * gAi[0][b] + Ai[1][a] * gAi[1][b] + Ai[2][a] * gAi[2][b];
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b) gA[a][b] = -(tmp[a][0] * Ai[b][0] + tmp[a][1] * Ai[b][1] + tmp[a][2] * Ai[b][2]);
        B gJ[3][3], gB[3][3], gM[3][3];
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b) {
                gJ[a][b] = gA[a][0] * (B)G.Bm[3 * b] + gA[a][1] * (B)G.Bm[3 * b + 1] + gA[a][2] * (B)G.Bm[3 * b + 2];
                gB[a][b] = (B)G.J[a] * gA[0][b] + (B)G.J[3 + a] * gA[1][b] + (B)G.J[6 + a] * gA[2][b];
            }
        const float* W = P.W;
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b) gM[a][b] = (B)W[a] * gB[0][b] + (B)W[3 + a] * gB[1][b] + (B)W[6 + a] * gB[2][b];
        const float sc[3] = {__ldg(scales + 3 * i), __ldg(scales + 3 * i + 1), __ldg(scales + 3 * i + 2)};
        B gR[3][3];
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int j = 0; j < 3; ++j) { g_s[j] += (B)G.R[3 * a + j] * gM[a][j]; gR[a][j] = (B)sc[j] * gM[a][j]; }
        {
            const float4 q4 = __ldg(reinterpret_cast<const float4*>(quats) + i);
            const B w = q4.x, x = q4.y, y = q4.z, z = q4.w;
            g_q[0] = 2.0 * (-z * gR[0][1] + y * gR[0][2] + z * gR[1][0] - x * gR[1][2] - y * gR[2][0] + x * gR[2][1]);
            g_q[1] = 2.0 * (y * gR[0][1] + z * gR[0][2] + y * gR[1][0] - 2.0 * x * gR[1][1] - w * gR[1][2] + z * gR[2][0] + w * gR[2][1] - 2.0 * x * gR[2][2]);
            g_q[2] = 2.0 * (-2.0 * y * gR[0][0] + x * gR[0][1] + w * gR[0][2] + x * gR[1][0] + z * gR[1][2] - w * gR[2][0] + z * gR[2][1] - 2.0 * y * gR[2][2]);
            g_q[3] = 2.0 * (-2.0 * z * gR[0][0] - w * gR[0][1] + x * gR[0][2] + w * gR[1][0] - 2.0 * z * gR[1][1] + y * gR[1][2] + x * gR[2][0] + y * gR[2][1]);
        }
        // density sigma = -log(1 - 0.99 o) / (2 min s)
        const B gsig = (B)gr[2], smin = (B)G.smin, od = (B)__ldg(opac + i);
        g_o = gsig * 0.99 / ((1.0 - 0.99 * od) * 2.0 * smin);
        {
            const B gsm = -gsig * (B)G.sigma / smin;
            if (G.jmin == 0) g_s[0] += gsm; else if (G.jmin == 1) g_s[1] += gsm; else g_s[2] += gsm;
        }
        // J(p) and mu2D
        const B x = G.p[0], y = G.p[1], z = G.p[2], d = (B)G.dist, fx = P.fx, fy = P.fy;
        B g_p[3] = {0, 0, 0};
        g_p[2] += gJ[0][0] * (-fx / (z * z)) + gJ[1][1] * (-fy / (z * z));
        g_p[0] += gJ[0][2] * (-fx / (z * z)); g_p[2] += gJ[0][2] * (2.0 * fx * x / (z * z * z));
        g_p[1] += gJ[1][2] * (-fy / (z * z)); g_p[2] += gJ[1][2] * (2.0 * fy * y / (z * z * z));
        const B r[3] = {x / d, y / d, z / d};
        const B rg = r[0] * gJ[2][0] + r[1] * gJ[2][1] + r[2] * gJ[2][2];
#pragma unroll
        for (int b = 0; b < 3; ++b) g_p[b] += (gJ[2][b] - r[b] * rg) / d;
        g_p[0] += (B)gr[0] * fx / z; g_p[1] += (B)gr[1] * fy / z;
        g_p[2] += -(B)gr[0] * fx * x / (z * z) - (B)gr[1] * fy * y / (z * z);
#pragma unroll
        for (int j = 0; j < 3; ++j) g_mu[j] += (B)W[j] * g_p[0] + (B)W[3 + j] * g_p[1] + (B)W[6 + j] * g_p[2];
    }
#pragma unroll
    for (int j = 0; j < 3; ++j) { g_means[3 * i + j] = (float)g_mu[j]; g_scales[3 * i + j] = (float)g_s[j]; }
    reinterpret_cast<float4*>(g_quats)[i] = make_float4((float)g_q[0], (float)g_q[1], (float)g_q[2], (float)g_q[3]);
    g_opacities[i] = (float)g_o;
}

int32_t make_params(const xpr_camera* cam, const xpr_config* cfg, ProjParams& P) {
    for (int i = 0; i < 3; ++i) {
        for (int j = 0; j < 3; ++j) P.W[3 * i + j] = cam->w2c[4 * i + j];
        P.t[i] = cam->w2c[4 * i + 3];
    }
    P.fx = cam->fx; P.fy = cam->fy; P.cx = cam->cx; P.cy = cam->cy;
    for (int i = 0; i < 4; ++i) P.k[i] = (double)cam->k[i];
    P.model = cam->model; P.projection = cfg->projection;
    P.K = (cfg->sh_degree + 1) * (cfg->sh_degree + 1);
    P.antialias = cfg->antialias;
    P.alpha_thresh = cfg->alpha_thresh; P.z_near = cfg->z_near; P.lowpass = cfg->lowpass;
    // C6: clamp x/z to [-(cx + 0.15 W)/fx, ((W - cx) + 0.15 W)/fx], likewise y (fp32, this order)
    volatile float wf = (float)cam->width, hf = (float)cam->height;
    volatile float extx = 0.15f * wf, exty = 0.15f * hf;
    volatile float nx = (wf - cam->cx), ny = (hf - cam->cy);
    volatile float sx = nx + extx, sy = ny + exty;
    volatile float mx = cam->cx + extx, my = cam->cy + exty;
    P.hix = sx / cam->fx; P.hiy = sy / cam->fy;
    volatile float lx = mx / cam->fx, ly = my / cam->fy;
    P.lox = -lx; P.loy = -ly;
    // UT weights: n = 3, lambda = alpha^2 (n + kappa) - n
    const double n = 3.0, al = (double)cfg->ut_alpha, lam = al * al * (n + (double)cfg->ut_kappa) - n;
    if (cfg->projection == 1 && !(n + lam > 0.0)) return XPR_ERR_INVALID_ARG;
    P.gamma = (float)sqrt(n + lam);
    const double wm0 = lam / (n + lam);
    P.wm0 = (float)wm0;
    P.wc0 = (float)(wm0 + (1.0 - al * al + (double)cfg->ut_beta));
    P.wk = (float)(1.0 / (2.0 * (n + lam)));
    for (int j = 0; j < 3; ++j) {
        volatile float s0 = P.W[j] * P.t[0], s1 = P.W[3 + j] * P.t[1], s2 = P.W[6 + j] * P.t[2];
        volatile float s01 = s0 + s1;
        volatile float s = s01 + s2;
        P.cpos[j] = -s;
    }
    P.TW = tiles_x(cam); P.TH = tiles_y(cam);
    return XPR_OK;
}

}  // namespace
}  // namespace xpr

using namespace xpr;

extern "C" int32_t xpr_project(int64_t N, const float* means, const float* scales, const float* quats,
                               const float* opacities, const float* sh, const xpr_camera* cam,
                               const xpr_config* cfg, float* mean2d, float* conic_opac, float* rgb, float* depth,
                               float* lnv, int32_t* tile_rect, uint32_t* tile_count, uint8_t* flags,
                               float* shade_rec, void* stream) {
    if (int32_t s = check_cam_cfg(cam, cfg)) return s;
    if (N < 0 || N > 0x7fffffffLL) return XPR_ERR_INVALID_ARG;
    if (N == 0) return XPR_OK;
    if (!aligned(means, 4) || !aligned(scales, 4) || !aligned(quats, 16) || !aligned(opacities, 4) ||
        !aligned(sh, 16) || !aligned(mean2d, 8) || !aligned(conic_opac, 16) || !aligned(rgb, 4) ||
        !aligned(depth, 4) || !aligned(lnv, 4) || !aligned(tile_rect, 16) || !aligned(tile_count, 4) || !flags ||
        (shade_rec && !aligned(shade_rec, 16)))
        return XPR_ERR_INVALID_ARG;
    ProjBatch P;
    const int V = num_views(cfg);
    for (int v = 0; v < V; ++v)
        if (int32_t s = make_params(cam + v, cfg, P.p[v])) return s;
    cudaStream_t st = (cudaStream_t)stream;
    const int threads = PROJ_THREADS;
    const dim3 blocks((unsigned)((N + PROJ_CHUNK - 1) / PROJ_CHUNK), (unsigned)V);
#define XPR_GO(KK)                                                                                              \
    project_kernel<KK><<<blocks, threads, 0, st>>>(N, P, means, scales, quats, opacities, sh, mean2d, conic_opac, \
                                                   rgb, depth, lnv, tile_rect, tile_count, flags,                \
                                                   reinterpret_cast<float4*>(shade_rec))
    switch (cfg->sh_degree) {
        case 0: XPR_GO(1); break;
        case 1: XPR_GO(4); break;
        case 2: XPR_GO(9); break;
        default: XPR_GO(16); break;
    }
#undef XPR_GO
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}

// zero-fill of the five parameter-gradient arrays: one memset when they are adjacent slices of one allocation, in this order
static int32_t fill_param_grads(int64_t N, const xpr_config* cfg, float* g_means, float* g_scales, float* g_quats,
                                float* g_opacities, float* g_sh, cudaStream_t st) {
    const size_t n = (size_t)N, K3 = 3 * (size_t)((cfg->sh_degree + 1) * (cfg->sh_degree + 1));
    if (g_scales == g_means + 3 * n && g_quats == g_scales + 3 * n && g_opacities == g_quats + 4 * n &&
        g_sh == g_opacities + n) {
        XPR_CUDA(cudaMemsetAsync(g_means, 0, sizeof(float) * (11 + K3) * n, st));
    } else {
        XPR_CUDA(cudaMemsetAsync(g_means, 0, sizeof(float) * 3 * n, st));
        XPR_CUDA(cudaMemsetAsync(g_scales, 0, sizeof(float) * 3 * n, st));
        XPR_CUDA(cudaMemsetAsync(g_quats, 0, sizeof(float) * 4 * n, st));
        XPR_CUDA(cudaMemsetAsync(g_opacities, 0, sizeof(float) * n, st));
        XPR_CUDA(cudaMemsetAsync(g_sh, 0, sizeof(float) * K3 * n, st));
    }
    return XPR_OK;
}

extern "C" int32_t xpr_project_bwd_fill(int64_t N, const xpr_config* cfg, float* g_means, float* g_scales, float* g_quats,
                                        float* g_opacities, float* g_sh, void* stream) {
    if (!cfg || cfg->sh_degree < 0 || cfg->sh_degree > 3 || N < 0 || N > 0x7fffffffLL) return XPR_ERR_INVALID_ARG;
    if (N == 0) return XPR_OK;
    if (!aligned(g_means, 4) || !aligned(g_scales, 4) || !aligned(g_quats, 16) || !aligned(g_opacities, 4) || !aligned(g_sh, 16))
        return XPR_ERR_INVALID_ARG;
    return fill_param_grads(N, cfg, g_means, g_scales, g_quats, g_opacities, g_sh, (cudaStream_t)stream);
}

static int32_t project_bwd_impl(bool fill, int64_t N, const float* means, const float* scales, const float* quats,
                                const float* opacities, const float* sh, const xpr_camera* cam,
                                const xpr_config* cfg, const uint32_t* tile_count, const uint8_t* flags,
                                const float* g_mean2d, const float* g_conic, const float* g_opac,
                                const float* g_rgb, float* g_means, float* g_scales, float* g_quats,
                                float* g_opacities, float* g_sh, void* stream) {
    if (int32_t s = check_cam_cfg(cam, cfg)) return s;
    if (N < 0 || N > 0x7fffffffLL) return XPR_ERR_INVALID_ARG;
    if (N == 0) return XPR_OK;
    if (!aligned(means, 4) || !aligned(scales, 4) || !aligned(quats, 16) || !aligned(opacities, 4) ||
        !aligned(sh, 16) || !aligned(tile_count, 4) || !flags || !aligned(g_mean2d, 8) || !aligned(g_conic, 4) ||
        !aligned(g_opac, 4) || !aligned(g_rgb, 4) || !aligned(g_means, 4) || !aligned(g_scales, 4) ||
        !aligned(g_quats, 16) || !aligned(g_opacities, 4) || !aligned(g_sh, 16))
        return XPR_ERR_INVALID_ARG;
    ProjBatch P;
    const int V = num_views(cfg);
    for (int v = 0; v < V; ++v)
        if (int32_t s = make_params(cam + v, cfg, P.p[v])) return s;
    cudaStream_t st = (cudaStream_t)stream;
    // Gaussians per CTA: enough CTAs for one full wave (148 SMs x 4 CTAs) before growing the chunk
#ifndef XPR_PBWD_WAVES
#define XPR_PBWD_WAVES 2
#endif
    int ipt = (int)(N / ((int64_t)148 * 4 * PBWD_THREADS * XPR_PBWD_WAVES));
    ipt = ipt < 1 ? 1 : (ipt > PBWD_MAX_IPT ? PBWD_MAX_IPT : ipt);
    const int64_t chunk = (int64_t)PBWD_THREADS * ipt;
    const dim3 blocks((unsigned)((N + chunk - 1) / chunk), (unsigned)V);
    if (fill)
        if (int32_t s = fill_param_grads(N, cfg, g_means, g_scales, g_quats, g_opacities, g_sh, st)) return s;
#define XPR_GO(KK)                                                                                                  \
    project_bwd_kernel<KK><<<blocks, PBWD_THREADS, 0, st>>>(N, P, ipt, means, scales, quats, opacities, sh, tile_count, \
                                                            flags, g_mean2d, g_conic, g_opac, g_rgb, g_means, g_scales, \
                                                            g_quats, g_opacities, g_sh)
    switch (cfg->sh_degree) {
        case 0: XPR_GO(1); break;
        case 1: XPR_GO(4); break;
        case 2: XPR_GO(9); break;
        default: XPR_GO(16); break;
    }
#undef XPR_GO
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}

extern "C" int32_t xpr_project_bwd(int64_t N, const float* means, const float* scales, const float* quats,
                                   const float* opacities, const float* sh, const xpr_camera* cam,
                                   const xpr_config* cfg, const uint32_t* tile_count, const uint8_t* flags,
                                   const float* g_mean2d, const float* g_conic, const float* g_opac,
                                   const float* g_rgb, float* g_means, float* g_scales, float* g_quats,
                                   float* g_opacities, float* g_sh, void* stream) {
    return project_bwd_impl(true, N, means, scales, quats, opacities, sh, cam, cfg, tile_count, flags, g_mean2d, g_conic,
                            g_opac, g_rgb, g_means, g_scales, g_quats, g_opacities, g_sh, stream);
}

extern "C" int32_t xpr_project_bwd_filled(int64_t N, const float* means, const float* scales, const float* quats,
                                          const float* opacities, const float* sh, const xpr_camera* cam,
                                          const xpr_config* cfg, const uint32_t* tile_count, const uint8_t* flags,
                                          const float* g_mean2d, const float* g_conic, const float* g_opac,
                                          const float* g_rgb, float* g_means, float* g_scales, float* g_quats,
                                          float* g_opacities, float* g_sh, void* stream) {
    return project_bwd_impl(false, N, means, scales, quats, opacities, sh, cam, cfg, tile_count, flags, g_mean2d, g_conic,
                            g_opac, g_rgb, g_means, g_scales, g_quats, g_opacities, g_sh, stream);
}

extern "C" int32_t xpr_lin_project(int64_t N, const float* means, const float* scales, const float* quats,
                                   const float* opacities, const float* sh, const xpr_camera* cam, const xpr_config* cfg,
                                   float* lin_rec, float* depth, int32_t* tile_rect, uint32_t* tile_count, void* stream) {
    if (int32_t s = check_cam_cfg(cam, cfg)) return s;
    if (cam->model != 0 || num_views(cfg) != 1) return XPR_ERR_UNSUPPORTED;      // LinPrim: pinhole, one view
    if (N < 0 || N > 0x7fffffffLL) return XPR_ERR_INVALID_ARG;
    if (N == 0) return XPR_OK;
    if (!aligned(means, 4) || !aligned(scales, 4) || !aligned(quats, 16) || !aligned(opacities, 4) || !aligned(sh, 16) ||
        !aligned(lin_rec, 16) || !aligned(depth, 4) || !aligned(tile_rect, 16) || !aligned(tile_count, 4))
        return XPR_ERR_INVALID_ARG;
    ProjParams P;
    if (int32_t s = make_params(cam, cfg, P)) return s;
    cudaStream_t st = (cudaStream_t)stream;
    const unsigned blocks = (unsigned)((N + 127) / 128);
#define XPR_GO(KK)                                                                                              \
    lin_project_kernel<KK><<<blocks, 128, 0, st>>>(N, P, means, scales, quats, opacities, sh,                    \
                                                   reinterpret_cast<float4*>(lin_rec), depth, tile_rect, tile_count)
    switch (cfg->sh_degree) {
        case 0: XPR_GO(1); break;
        case 1: XPR_GO(4); break;
        case 2: XPR_GO(9); break;
        default: XPR_GO(16); break;
    }
#undef XPR_GO
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}

extern "C" int32_t xpr_lin_project_bwd(int64_t N, const float* means, const float* scales, const float* quats,
                                       const float* opacities, const float* sh, const xpr_camera* cam, const xpr_config* cfg,
                                       const uint32_t* tile_count, const float* lin_rec, const float* g_lin_rec,
                                       float* g_means, float* g_scales, float* g_quats, float* g_opacities, float* g_sh,
                                       void* stream) {
    if (int32_t s = check_cam_cfg(cam, cfg)) return s;
    if (cam->model != 0 || num_views(cfg) != 1) return XPR_ERR_UNSUPPORTED;
    if (N < 0 || N > 0x7fffffffLL) return XPR_ERR_INVALID_ARG;
    if (N == 0) return XPR_OK;
    if (!aligned(means, 4) || !aligned(scales, 4) || !aligned(quats, 16) || !aligned(opacities, 4) || !aligned(sh, 16) ||
        !aligned(tile_count, 4) || !aligned(lin_rec, 16) || !aligned(g_lin_rec, 16) || !aligned(g_means, 4) ||
        !aligned(g_scales, 4) || !aligned(g_quats, 16) || !aligned(g_opacities, 4) || !aligned(g_sh, 16))
        return XPR_ERR_INVALID_ARG;
    ProjParams P;
    if (int32_t s = make_params(cam, cfg, P)) return s;
    cudaStream_t st = (cudaStream_t)stream;
    const unsigned blocks = (unsigned)((N + 127) / 128);
#define XPR_GO(KK)                                                                                                    \
    lin_project_bwd_kernel<KK><<<blocks, 128, 0, st>>>(N, P, means, scales, quats, opacities, sh, tile_count,          \
                                                       reinterpret_cast<const float4*>(lin_rec),                       \
                                                       reinterpret_cast<const float4*>(g_lin_rec), g_means, g_scales,  \
                                                       g_quats, g_opacities, g_sh)
    switch (cfg->sh_degree) {
        case 0: XPR_GO(1); break;
        case 1: XPR_GO(4); break;
        case 2: XPR_GO(9); break;
        default: XPR_GO(16); break;
    }
#undef XPR_GO
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}
