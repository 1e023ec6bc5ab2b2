// ray.cu -- the per-pixel and per-Gaussian maps of the XPR-3DGUT evaluation (PAPER A.1.2
// L437-444 Eq. 1, Listing 3): xpr_pixel_info (ray direction per pixel), xpr_project_ray (shader record
// M_c, o_c) and xpr_ray_bwd (chain rule from the record's gradient to mean, scale, quaternion).
//
// Reading C27: ray and Gaussian are expressed in the camera frame, p = W mu + t, ray origin 0:
//   M_c = S^-1 (W R)^T,  o_c = -M_c p,  d_c = M_c d.
// This translation unit is compiled with -fmad=false (rule R1): the record is fp32 with every operation
// individually rounded in the order written here; pixel_info runs in fp64 and rounds last (rule R2).
#include <math.h>

#include "common.cuh"

namespace xpr {
namespace {

struct RayCam {
    float W[9], t[3];
    double fx, fy, cx, cy, k[4];
    int model, width, height;
};

void make_ray_cam(const xpr_camera* cam, RayCam& C) {
    for (int i = 0; i < 3; ++i) {
        for (int j = 0; j < 3; ++j) C.W[3 * i + j] = cam->w2c[4 * i + j];
        C.t[i] = cam->w2c[4 * i + 3];
    }
    C.fx = cam->fx; C.fy = cam->fy; C.cx = cam->cx; C.cy = cam->cy;
    for (int i = 0; i < 4; ++i) C.k[i] = cam->k[i];
    C.model = cam->model; C.width = cam->width; C.height = cam->height;
}

// pixel_info: unit direction of the ray through (px + 1/2, py + 1/2), inverse of the camera model.
__global__ void __launch_bounds__(256) pixel_info_kernel(RayCam C, float* __restrict__ rays) {
    const int64_t pid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (pid >= (int64_t)C.width * C.height) return;
    const int px = (int)(pid % C.width), py = (int)(pid / C.width);
    const double xn = (((double)px + 0.5) - C.cx) / C.fx, yn = (((double)py + 0.5) - C.cy) / C.fy;
    double dx, dy, dz;
    if (C.model == 0) {
        const double n = sqrt((xn * xn + yn * yn) + 1.0);
        dx = xn / n; dy = yn / n; dz = 1.0 / n;
    } else {
        const double rd = sqrt(xn * xn + yn * yn);
        if (rd > 0.0) {
            double th = rd;   // theta (1 + k1 th^2 + k2 th^4 + k3 th^6 + k4 th^8) = rd, <= 12 Newton steps
            for (int it = 0; it < 12; ++it) {
                const double t2 = th * th;
                const double f = th * (1.0 + t2 * (C.k[0] + t2 * (C.k[1] + t2 * (C.k[2] + t2 * C.k[3])))) - rd;
                if (!(fabs(f) > 4e-16 * rd)) break;               // converged to fp64 rounding
                const double fp = 1.0 + t2 * (3.0 * C.k[0] + t2 * (5.0 * C.k[1] + t2 * (7.0 * C.k[2] + t2 * (9.0 * C.k[3]))));
                th = th - f / fp;
            }
            double sn, cs;
            sincos(th, &sn, &cs);
            const double s = sn / rd;
            dx = s * xn; dy = s * yn; dz = cs;
        } else { dx = 0.0; dy = 0.0; dz = 1.0; }
    }
    rays[3 * pid] = (float)dx; rays[3 * pid + 1] = (float)dy; rays[3 * pid + 2] = (float)dz;
}

struct RayFwd { float p[3], R[9], Mc[9], oc[3]; };

__device__ __forceinline__ void ray_record(const RayCam& C, const float mu[3], const float sc[3], const float q[4],
                                           RayFwd& F) {
    const float* W = C.W;
#pragma unroll
    for (int i = 0; i < 3; ++i) F.p[i] = ((W[3 * i] * mu[0] + W[3 * i + 1] * mu[1]) + W[3 * i + 2] * mu[2]) + C.t[i];
    {   // R(q), (w,x,y,z), not renormalised (C3)
        const float w = q[0], x = q[1], y = q[2], z = q[3];
        const float xx = x * x, yy = y * y, zz = z * z, xy = x * y, xz = x * z, yz = y * z;
        const float wx = w * x, wy = w * y, wz = w * z;
        F.R[0] = 1.0f - 2.0f * (yy + zz); F.R[1] = 2.0f * (xy - wz); F.R[2] = 2.0f * (xz + wy);
        F.R[3] = 2.0f * (xy + wz); F.R[4] = 1.0f - 2.0f * (xx + zz); F.R[5] = 2.0f * (yz - wx);
        F.R[6] = 2.0f * (xz - wy); F.R[7] = 2.0f * (yz + wx); F.R[8] = 1.0f - 2.0f * (xx + yy);
    }
    float WR[9];
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j)
            WR[3 * i + j] = (W[3 * i] * F.R[j] + W[3 * i + 1] * F.R[3 + j]) + W[3 * i + 2] * F.R[6 + j];
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) F.Mc[3 * i + j] = WR[3 * j + i] / sc[i];
#pragma unroll
    for (int i = 0; i < 3; ++i)
        F.oc[i] = -((F.Mc[3 * i] * F.p[0] + F.Mc[3 * i + 1] * F.p[1]) + F.Mc[3 * i + 2] * F.p[2]);
}

__global__ void __launch_bounds__(128)
project_ray_kernel(int64_t N, RayCam C, const float* __restrict__ means, const float* __restrict__ scales,
                   const float4* __restrict__ quats, const uint32_t* __restrict__ tile_count,
                   float4* __restrict__ ray_rec) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f), r1 = r0, r2 = r0;
    if (tile_count[i] != 0) {
        const float mu[3] = {means[3 * i], means[3 * i + 1], means[3 * i + 2]};
        const float sc[3] = {scales[3 * i], scales[3 * i + 1], scales[3 * i + 2]};
        const float4 qv = quats[i];
        const float q[4] = {qv.x, qv.y, qv.z, qv.w};
        RayFwd F;
        ray_record(C, mu, sc, q, F);
        bool finite = true;   // C30: a record that is not finite becomes zeros (never valid)
#pragma unroll
        for (int k = 0; k < 9; ++k) finite = finite && isfinite(F.Mc[k]);
#pragma unroll
        for (int k = 0; k < 3; ++k) finite = finite && isfinite(F.oc[k]);
        if (finite) {
            r0 = make_float4(F.Mc[0], F.Mc[1], F.Mc[2], F.Mc[3]);
            r1 = make_float4(F.Mc[4], F.Mc[5], F.Mc[6], F.Mc[7]);
            r2 = make_float4(F.Mc[8], F.oc[0], F.oc[1], F.oc[2]);
        }
    }
    ray_rec[3 * i] = r0; ray_rec[3 * i + 1] = r1; ray_rec[3 * i + 2] = r2;
}

// Chain rule record -> (mu, s, q), fp64 on the forward intermediates recomputed in fp32:
//   Gt = dL/dM_c - dL/do_c p^T, formed from the accumulators S_c, D of xpr_rasterize_ray_bwd;
//   dL/dp = -M_c^T dL/do_c;  dL/dmu = W^T dL/dp;
//   dL/d(WR)[j][i] = Gt[i][j] / s_i;  dL/ds_i = -sum_j Gt[i][j] M_c[i][j] / s_i;  dL/dR = W^T dL/d(WR);  R(q) (C17).
__global__ void __launch_bounds__(128)
ray_bwd_kernel(int64_t N, RayCam C, const float* __restrict__ means, const float* __restrict__ scales,
               const float4* __restrict__ quats, const uint32_t* __restrict__ tile_count,
               const float4* __restrict__ g_acc, float* __restrict__ g_means, float* __restrict__ g_scales,
               float4* __restrict__ g_quats) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    if (tile_count[i] == 0) return;
    const float4 a0 = g_acc[4 * i], a1 = g_acc[4 * i + 1], a2 = g_acc[4 * i + 2], a3 = g_acc[4 * i + 3];
    const double g[15] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w, a2.x, a2.y, a2.z, a2.w, a3.x, a3.y, a3.z};
    bool any = false;
#pragma unroll
    for (int k = 0; k < 15; ++k) any = any || (g[k] != 0.0);
    if (!any) return;
    const float mu[3] = {means[3 * i], means[3 * i + 1], means[3 * i + 2]};
    const float sc[3] = {scales[3 * i], scales[3 * i + 1], scales[3 * i + 2]};
    const float4 qv = quats[i];
    const float q[4] = {qv.x, qv.y, qv.z, qv.w};
    RayFwd F;
    ray_record(C, mu, sc, q, F);
    // dL/dM_c - dL/do_c p^T = -(S_c - tr(S_c) I) M_c^-T + M_c D  (rasterize_ray.cu), M_c^-T = cofactors / determinant
    // (the quaternion is not renormalised, C3, so W R need not be orthogonal)
    double M[9], MiT[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) M[k] = (double)F.Mc[k];
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const int a1i = (a + 1) % 3, a2i = (a + 2) % 3, b1i = (b + 1) % 3, b2i = (b + 2) % 3;
            MiT[3 * a + b] = M[3 * a1i + b1i] * M[3 * a2i + b2i] - M[3 * a1i + b2i] * M[3 * a2i + b1i];
        }
    const double rdet = 1.0 / (M[0] * MiT[0] + M[1] * MiT[1] + M[2] * MiT[2]);
    const double Sc[9] = {g[0], g[1], g[2], g[1], g[3], g[4], g[2], g[4], g[5]};
    const double D[9] = {g[6], g[7], g[8], g[7], g[9], g[10], g[8], g[10], g[11]};
    const double tr = g[0] + g[3] + g[5];
    double Gt[9], gp[3] = {0.0, 0.0, 0.0};
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            double u = 0.0, v = 0.0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                u += (Sc[3 * a + k] - (a == k ? tr : 0.0)) * MiT[3 * k + b];
                v += M[3 * a + k] * D[3 * k + b];
            }
            Gt[3 * a + b] = v - u * rdet;
            gp[b] -= M[3 * a + b] * g[12 + a];
        }
    double W[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) W[k] = (double)C.W[k];
    double gmu[3], gs[3], gWR[9], gR[9];
#pragma unroll
    for (int b = 0; b < 3; ++b) gmu[b] = W[b] * gp[0] + W[3 + b] * gp[1] + W[6 + b] * gp[2];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        gs[a] = 0.0;
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            gWR[3 * b + a] = Gt[3 * a + b] / (double)sc[a];
            gs[a] -= Gt[3 * a + b] * (double)F.Mc[3 * a + b] / (double)sc[a];
        }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k)
#pragma unroll
        for (int b = 0; b < 3; ++b) gR[3 * k + b] = W[k] * gWR[b] + W[3 + k] * gWR[3 + b] + W[6 + k] * gWR[6 + b];
    const double w = q[0], x = q[1], y = q[2], z = q[3];
    const double gq0 = 2.0 * (-z * gR[1] + y * gR[2] + z * gR[3] - x * gR[5] - y * gR[6] + x * gR[7]);
    const double gq1 = 2.0 * (y * gR[1] + z * gR[2] + y * gR[3] - 2.0 * x * gR[4] - w * gR[5] + z * gR[6] + w * gR[7] - 2.0 * x * gR[8]);
    const double gq2 = 2.0 * (-2.0 * y * gR[0] + x * gR[1] + w * gR[2] + x * gR[3] + z * gR[5] - w * gR[6] + z * gR[7] - 2.0 * y * gR[8]);
    const double gq3 = 2.0 * (-2.0 * z * gR[0] - w * gR[1] + x * gR[2] + w * gR[3] - 2.0 * z * gR[4] + y * gR[5] + x * gR[6] + y * gR[7]);
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        g_means[3 * i + b] = (float)((double)g_means[3 * i + b] + gmu[b]);
        g_scales[3 * i + b] = (float)((double)g_scales[3 * i + b] + gs[b]);
    }
    const float4 o = g_quats[i];
    g_quats[i] = make_float4((float)((double)o.x + gq0), (float)((double)o.y + gq1), (float)((double)o.z + gq2),
                             (float)((double)o.w + gq3));
}

int32_t check_cam(const xpr_camera* cam) {
    if (!cam) return XPR_ERR_INVALID_ARG;
    if (cam->width <= 0 || cam->height <= 0) return XPR_ERR_INVALID_ARG;
    if (cam->model != 0 && cam->model != 1) return XPR_ERR_INVALID_ARG;
    return XPR_OK;
}

}  // namespace
}  // namespace xpr

using namespace xpr;

extern "C" int32_t xpr_pixel_info(const xpr_camera* cam, float* pixel_rays, void* stream) {
    if (int32_t s = check_cam(cam)) return s;
    if (!aligned(pixel_rays, 4)) return XPR_ERR_INVALID_ARG;
    RayCam C;
    make_ray_cam(cam, C);
    const int64_t n = (int64_t)cam->width * cam->height;
    pixel_info_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(C, pixel_rays);
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}

extern "C" int32_t xpr_project_ray(int64_t N, const float* means, const float* scales, const float* quats,
                                   const xpr_camera* cam, const uint32_t* tile_count, float* ray_rec, void* stream) {
    if (int32_t s = check_cam(cam)) return s;
    if (N < 0 || N > 0x7fffffffLL) return XPR_ERR_INVALID_ARG;
    if (N == 0) return XPR_OK;
    if (!aligned(means, 4) || !aligned(scales, 4) || !aligned(quats, 16) || !aligned(tile_count, 4) ||
        !aligned(ray_rec, 16))
        return XPR_ERR_INVALID_ARG;
    RayCam C;
    make_ray_cam(cam, C);
    project_ray_kernel<<<(unsigned)((N + 127) / 128), 128, 0, (cudaStream_t)stream>>>(
        N, C, means, scales, reinterpret_cast<const float4*>(quats), tile_count, reinterpret_cast<float4*>(ray_rec));
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}

extern "C" int32_t xpr_ray_bwd(int64_t N, const float* means, const float* scales, const float* quats,
                               const xpr_camera* cam, const uint32_t* tile_count, const float* g_ray_acc,
                               float* g_means, float* g_scales, float* g_quats, void* stream) {
    if (int32_t s = check_cam(cam)) return s;
    if (N < 0 || N > 0x7fffffffLL) return XPR_ERR_INVALID_ARG;
    if (N == 0) return XPR_OK;
    if (!aligned(means, 4) || !aligned(scales, 4) || !aligned(quats, 16) || !aligned(tile_count, 4) ||
        !aligned(g_ray_acc, 16) || !aligned(g_means, 4) || !aligned(g_scales, 4) || !aligned(g_quats, 16))
        return XPR_ERR_INVALID_ARG;
    RayCam C;
    make_ray_cam(cam, C);
    ray_bwd_kernel<<<(unsigned)((N + 127) / 128), 128, 0, (cudaStream_t)stream>>>(
        N, C, means, scales, reinterpret_cast<const float4*>(quats), tile_count,
        reinterpret_cast<const float4*>(g_ray_acc), g_means, g_scales, reinterpret_cast<float4*>(g_quats));
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}
