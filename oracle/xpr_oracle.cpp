// xpr_oracle.cpp -- CPU ORACLE (test infrastructure, NOT the product; see xpr_oracle.h).
//
// Plain, slow, obviously-correct restatement of the tile-based splatting forward + backward
// pass of PAPER.md (XPR, arxiv 2606.11529), following DESIGN.md readings C1..C26 and the
// arithmetic rules R1..R3.  No blocking, fusion or reordering beyond what those state.
// Shares no code with paper_2606_11529_b200/csrc.  Build: oracle/build.py
// (g++ -O2 -ffp-contract=off -fno-fast-math -fopenmp).
//
// Template parameter S: float = parity mode, double = self-check mode.
#include "xpr_oracle.h"

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <numeric>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---------------------------------------------------------------------------------------------
// Real spherical harmonics, degree <= 3 (reading C5: index k = l^2+l+m, Condon-Shortley sign).
// ---------------------------------------------------------------------------------------------
constexpr double SH_c0 = 0.28209479177387814;  // 1/(2 sqrt(pi))
constexpr double SH_c1 = 0.4886025119029199;   // sqrt(3/(4 pi))
constexpr double SH_a2 = 1.0925484305920792;   // sqrt(15/pi)/2
constexpr double SH_b2 = 0.31539156525252005;  // sqrt(5/pi)/4
constexpr double SH_c2 = 0.5462742152960396;   // sqrt(15/pi)/4
constexpr double SH_a3 = 0.5900435899266435;   // sqrt(35/(2 pi))/4
constexpr double SH_b3 = 2.890611442640554;    // sqrt(105/pi)/2
constexpr double SH_c3 = 0.4570457994644658;   // sqrt(21/(2 pi))/4
constexpr double SH_d3 = 0.3731763325901154;   // sqrt(7/pi)/4
constexpr double SH_e3 = 1.445305721320277;    // sqrt(105/pi)/4

template <class S>
void sh_basis(const S d[3], S Y[16]) {
    const S x = d[0], y = d[1], z = d[2];
    const S c0 = S(SH_c0), c1 = S(SH_c1), a2 = S(SH_a2), b2 = S(SH_b2), c2 = S(SH_c2);
    const S a3 = S(SH_a3), b3 = S(SH_b3), c3 = S(SH_c3), d3 = S(SH_d3), e3 = S(SH_e3);
    const S xx = x * x, yy = y * y, zz = z * z, xy = x * y, yz = y * z, xz = x * z;
    Y[0] = c0;
    Y[1] = (-c1) * y;
    Y[2] = c1 * z;
    Y[3] = (-c1) * x;
    Y[4] = a2 * xy;
    Y[5] = (-a2) * yz;
    Y[6] = b2 * ((S(2) * zz - xx) - yy);
    Y[7] = (-a2) * xz;
    Y[8] = c2 * (xx - yy);
    Y[9] = ((-a3) * y) * (S(3) * xx - yy);
    Y[10] = (b3 * xy) * z;
    Y[11] = ((-c3) * y) * ((S(4) * zz - xx) - yy);
    Y[12] = (d3 * z) * ((S(2) * zz - S(3) * xx) - S(3) * yy);
    Y[13] = ((-c3) * x) * ((S(4) * zz - xx) - yy);
    Y[14] = (e3 * z) * (xx - yy);
    Y[15] = ((-a3) * x) * (xx - S(3) * yy);
}

// Gradient of each basis polynomial w.r.t. the (free) components of d; fp64 (backward only).
void sh_basis_grad(const double d[3], double dY[16][3]) {
    const double x = d[0], y = d[1], z = d[2];
    const double xx = x * x, yy = y * y, zz = z * z, xy = x * y, yz = y * z, xz = x * z;
    for (int k = 0; k < 16; ++k) dY[k][0] = dY[k][1] = dY[k][2] = 0.0;
    dY[1][1] = -SH_c1;
    dY[2][2] = SH_c1;
    dY[3][0] = -SH_c1;
    dY[4][0] = SH_a2 * y;  dY[4][1] = SH_a2 * x;
    dY[5][1] = -SH_a2 * z; dY[5][2] = -SH_a2 * y;
    dY[6][0] = -2 * SH_b2 * x; dY[6][1] = -2 * SH_b2 * y; dY[6][2] = 4 * SH_b2 * z;
    dY[7][0] = -SH_a2 * z; dY[7][2] = -SH_a2 * x;
    dY[8][0] = 2 * SH_c2 * x; dY[8][1] = -2 * SH_c2 * y;
    dY[9][0] = -6 * SH_a3 * xy; dY[9][1] = -SH_a3 * (3 * xx - 3 * yy);
    dY[10][0] = SH_b3 * yz; dY[10][1] = SH_b3 * xz; dY[10][2] = SH_b3 * xy;
    dY[11][0] = 2 * SH_c3 * xy; dY[11][1] = -SH_c3 * (4 * zz - xx - 3 * yy); dY[11][2] = -8 * SH_c3 * yz;
    dY[12][0] = -6 * SH_d3 * xz; dY[12][1] = -6 * SH_d3 * yz; dY[12][2] = SH_d3 * (6 * zz - 3 * xx - 3 * yy);
    dY[13][0] = -SH_c3 * (4 * zz - 3 * xx - yy); dY[13][1] = 2 * SH_c3 * xy; dY[13][2] = -8 * SH_c3 * xz;
    dY[14][0] = 2 * SH_e3 * xz; dY[14][1] = -2 * SH_e3 * yz; dY[14][2] = SH_e3 * (xx - yy);
    dY[15][0] = -SH_a3 * (3 * xx - 3 * yy); dY[15][1] = 6 * SH_a3 * xy;
}

// ---------------------------------------------------------------------------------------------
// Camera model pi (readings C1, C2, C18): camera-space point -> continuous pixel coordinates.
// Pinhole: (fx x/z + cx, fy y/z + cy).  Fisheye-equidistant: r = sqrt(x^2+y^2),
// theta = atan2(r,z), theta_d = theta (1 + k1 th^2 + k2 th^4 + k3 th^6 + k4 th^8),
// pix = (fx theta_d x/r + cx, fy theta_d y/r + cy), limit theta_d/r -> 1/z as r -> 0.
// R2: atan2 and the radial polynomial go through fp64 in both modes.
// ---------------------------------------------------------------------------------------------
template <class S>
void camera_project(const xo_camera& cam, const S p[3], S pix[2]) {
    const S fx = S(cam.fx), fy = S(cam.fy), cx = S(cam.cx), cy = S(cam.cy);
    if (cam.model == 0) {
        pix[0] = fx * (p[0] / p[2]) + cx;
        pix[1] = fy * (p[1] / p[2]) + cy;
        return;
    }
    if (cam.model == 2) {   // affine (orthographic) map, oracle-only: lets pin P7 check the UT exactly
        pix[0] = fx * p[0] + cx;
        pix[1] = fy * p[1] + cy;
        return;
    }
    const S r = std::sqrt(p[0] * p[0] + p[1] * p[1]);
    S s;
    if (r > S(0)) {
        const double th = std::atan2((double)r, (double)p[2]);
        const double t2 = th * th;
        const double poly = 1.0 + t2 * (cam.k[0] + t2 * (cam.k[1] + t2 * (cam.k[2] + t2 * cam.k[3])));
        s = S((th * poly) / (double)r);
    } else {
        s = S(1.0 / (double)p[2]);
    }
    pix[0] = fx * (s * p[0]) + cx;
    pix[1] = fy * (s * p[1]) + cy;
}

// d pix / d p (2x3), fp64, for the UT backward.
void camera_project_jac(const xo_camera& cam, const double p[3], double Jp[2][3]) {
    const double x = p[0], y = p[1], z = p[2];
    if (cam.model == 0) {
        Jp[0][0] = cam.fx / z; Jp[0][1] = 0; Jp[0][2] = -cam.fx * x / (z * z);
        Jp[1][0] = 0; Jp[1][1] = cam.fy / z; Jp[1][2] = -cam.fy * y / (z * z);
        return;
    }
    if (cam.model == 2) {
        Jp[0][0] = cam.fx; Jp[0][1] = 0; Jp[0][2] = 0;
        Jp[1][0] = 0; Jp[1][1] = cam.fy; Jp[1][2] = 0;
        return;
    }
    const double r2 = x * x + y * y, r = std::sqrt(r2);
    if (!(r > 0)) {  // on-axis limit: s = 1/z, ds/dr = 0
        Jp[0][0] = cam.fx / z; Jp[0][1] = 0; Jp[0][2] = 0;
        Jp[1][0] = 0; Jp[1][1] = cam.fy / z; Jp[1][2] = 0;
        return;
    }
    const double th = std::atan2(r, z), t2 = th * th;
    const double k1 = cam.k[0], k2 = cam.k[1], k3 = cam.k[2], k4 = cam.k[3];
    const double thd = th * (1.0 + t2 * (k1 + t2 * (k2 + t2 * (k3 + t2 * k4))));
    const double dthd = 1.0 + t2 * (3 * k1 + t2 * (5 * k2 + t2 * (7 * k3 + t2 * 9 * k4)));
    const double dth_dr = z / (r2 + z * z), dth_dz = -r / (r2 + z * z);
    const double s = thd / r;
    const double ds_dr = (dthd * dth_dr * r - thd) / r2;
    const double ds_dz = dthd * dth_dz / r;
    const double ds_dx = ds_dr * x / r, ds_dy = ds_dr * y / r;
    Jp[0][0] = cam.fx * (s + x * ds_dx); Jp[0][1] = cam.fx * x * ds_dy; Jp[0][2] = cam.fx * x * ds_dz;
    Jp[1][0] = cam.fy * y * ds_dx; Jp[1][1] = cam.fy * (s + y * ds_dy); Jp[1][2] = cam.fy * y * ds_dz;
}

// ---------------------------------------------------------------------------------------------
// Forward intermediates of one primitive (kept for the backward pass).
// ---------------------------------------------------------------------------------------------
template <class S>
struct Proj {
    bool visible = false;
    S p[3];                 // camera-space mean
    S u0, v0, u, v;         // x/z, y/z and their clamped versions (C6)
    bool clamp_u = false, clamp_v = false;
    S R[3][3], M[3][3], Sig[3][3];
    S J00, J11, J02, J12, T[2][3];
    S m[2];                 // mean2d
    S a, b, c;              // raw 2D covariance
    S ap, cp, det, det_raw, rho, o_eff;
    S A, B, C, lnv, ex, ey;
    int32_t rect[4];
    uint32_t tc = 0;
    S dvec[3], dnorm, dir[3], Y[16], raw[3], rgb[3];
    uint8_t flags = 0;
    // UT
    S sig[7][3], pc[7][3], y[7][2], wm[7], wc[7], gamma;
};

template <class S>
void rotation(const S q[4], S R[3][3]) {   // reading C3: (w,x,y,z), not renormalised
    const S w = q[0], x = q[1], y = q[2], z = q[3];
    const S xx = x * x, yy = y * y, zz = z * z, xy = x * y, xz = x * z, yz = y * z;
    const S wx = w * x, wy = w * y, wz = w * z;
    R[0][0] = S(1) - S(2) * (yy + zz); R[0][1] = S(2) * (xy - wz); R[0][2] = S(2) * (xz + wy);
    R[1][0] = S(2) * (xy + wz); R[1][1] = S(1) - S(2) * (xx + zz); R[1][2] = S(2) * (yz - wx);
    R[2][0] = S(2) * (xz - wy); R[2][1] = S(2) * (yz + wx); R[2][2] = S(1) - S(2) * (xx + yy);
}

// project for one primitive: PAPER Listing 1 L239-262 (EWA) / Listing 3 L447-486 (UT).
template <class S>
void project_one(const S mu[3], const S sc[3], const S q[4], S o, const S* sh, const xo_camera& cam,
                 const xo_config& cfg, Proj<S>& P) {
    P.visible = false; P.tc = 0; P.flags = 0;
    const double* Wt = cam.w2c;
    S W[3][3], t[3];
    for (int i = 0; i < 3; ++i) { for (int j = 0; j < 3; ++j) W[i][j] = S(Wt[4 * i + j]); t[i] = S(Wt[4 * i + 3]); }
    const S fx = S(cam.fx), fy = S(cam.fy), cx = S(cam.cx), cy = S(cam.cy);
    // world -> camera (L241-242): p = W mu + t, left-to-right sums
    for (int i = 0; i < 3; ++i) P.p[i] = ((W[i][0] * mu[0] + W[i][1] * mu[1]) + W[i][2] * mu[2]) + t[i];
    if (!(P.p[2] > S(cfg.z_near))) return;                      // (mu_c[2] > z_near), L262
    // Sigma = R S S^T R^T (L78)
    rotation(q, P.R);
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) P.M[i][j] = P.R[i][j] * sc[j];
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j)
        P.Sig[i][j] = (P.M[i][0] * P.M[j][0] + P.M[i][1] * P.M[j][1]) + P.M[i][2] * P.M[j][2];

    if (cfg.projection == 0) {
        // EWA (L244-246, L435): mean through the pinhole, covariance through the clamped Jacobian
        P.u0 = P.p[0] / P.p[2]; P.v0 = P.p[1] / P.p[2];
        P.m[0] = fx * P.u0 + cx; P.m[1] = fy * P.v0 + cy;
        const S wf = S(cam.width), hf = S(cam.height);
        const S extx = S(0.15) * wf, exty = S(0.15) * hf;         // C6
        const S hix = ((wf - cx) + extx) / fx, lox = -((cx + extx) / fx);
        const S hiy = ((hf - cy) + exty) / fy, loy = -((cy + exty) / fy);
        P.clamp_u = !(P.u0 >= lox && P.u0 <= hix);
        P.clamp_v = !(P.v0 >= loy && P.v0 <= hiy);
        P.u = std::min(std::max(P.u0, lox), hix);
        P.v = std::min(std::max(P.v0, loy), hiy);
        P.J00 = fx / P.p[2]; P.J11 = fy / P.p[2];
        P.J02 = -(P.J00 * P.u); P.J12 = -(P.J11 * P.v);
        for (int j = 0; j < 3; ++j) {
            P.T[0][j] = P.J00 * W[0][j] + P.J02 * W[2][j];
            P.T[1][j] = P.J11 * W[1][j] + P.J12 * W[2][j];
        }
        S V[2][3];
        for (int r = 0; r < 2; ++r) for (int j = 0; j < 3; ++j)
            V[r][j] = (P.T[r][0] * P.Sig[0][j] + P.T[r][1] * P.Sig[1][j]) + P.T[r][2] * P.Sig[2][j];
        P.a = (V[0][0] * P.T[0][0] + V[0][1] * P.T[0][1]) + V[0][2] * P.T[0][2];
        P.b = (V[0][0] * P.T[1][0] + V[0][1] * P.T[1][1]) + V[0][2] * P.T[1][2];
        P.c = (V[1][0] * P.T[1][0] + V[1][1] * P.T[1][1]) + V[1][2] * P.T[1][2];
    } else {
        // Unscented transform, 2*3+1 sigma points (L437, L452-463); weights alpha,beta,kappa
        const double n = 3.0, lam = cfg.ut_alpha * cfg.ut_alpha * (n + cfg.ut_kappa) - n;
        P.gamma = S(std::sqrt(n + lam));
        const double wm0 = lam / (n + lam), wc0 = wm0 + (1.0 - cfg.ut_alpha * cfg.ut_alpha + cfg.ut_beta);
        const double wk = 1.0 / (2.0 * (n + lam));
        P.wm[0] = S(wm0); P.wc[0] = S(wc0);
        for (int k = 1; k < 7; ++k) { P.wm[k] = S(wk); P.wc[k] = S(wk); }
        for (int d = 0; d < 3; ++d) P.sig[0][d] = mu[d];
        for (int j = 0; j < 3; ++j) for (int d = 0; d < 3; ++d) {
            const S off = P.gamma * P.M[d][j];                   // gamma * s_j * R[:,j]
            P.sig[1 + 2 * j][d] = mu[d] + off;
            P.sig[2 + 2 * j][d] = mu[d] - off;
        }
        for (int k = 0; k < 7; ++k) {
            for (int i = 0; i < 3; ++i)
                P.pc[k][i] = ((W[i][0] * P.sig[k][0] + W[i][1] * P.sig[k][1]) + W[i][2] * P.sig[k][2]) + t[i];
            if (!(P.pc[k][2] > S(0))) return;                    // C18: any sigma point behind the camera
            camera_project(cam, P.pc[k], P.y[k]);
        }
        S mx = P.wm[0] * P.y[0][0], my = P.wm[0] * P.y[0][1];
        for (int k = 1; k < 7; ++k) { mx = mx + P.wm[k] * P.y[k][0]; my = my + P.wm[k] * P.y[k][1]; }
        P.m[0] = mx; P.m[1] = my;
        S a = S(0), b = S(0), c = S(0);
        for (int k = 0; k < 7; ++k) {
            const S dx = P.y[k][0] - mx, dy = P.y[k][1] - my;
            a = a + P.wc[k] * (dx * dx); b = b + P.wc[k] * (dx * dy); c = c + P.wc[k] * (dy * dy);
        }
        P.a = a; P.b = b; P.c = c;
    }
    // low-pass (C4; L467-470), determinant, conic = inverse covariance (L435)
    P.ap = P.a + S(cfg.lowpass); P.cp = P.c + S(cfg.lowpass);
    P.det = P.ap * P.cp - P.b * P.b;
    if (!(P.det > S(0))) return;                                 // (det > 0), L262
    P.det_raw = P.a * P.c - P.b * P.b;
    if (cfg.antialias) {                                         // C19, L472-473
        P.rho = std::sqrt(std::max(S(0), P.det_raw / P.det));
        P.o_eff = o * P.rho;
    } else { P.rho = S(1); P.o_eff = o; }
    // C9: >= for EWA (L262), > for UT (L482), exactly as printed
    if (cfg.projection == 0) { if (!(P.o_eff >= S(cfg.alpha_thresh))) return; }
    else                     { if (!(P.o_eff >  S(cfg.alpha_thresh))) return; }
    P.A = P.cp / P.det; P.B = (-P.b) / P.det; P.C = P.ap / P.det;
    // extents (C7), R2: the logarithm goes through fp64
    P.lnv = S(std::log((double)P.o_eff / (double)S(cfg.alpha_thresh)));
    P.ex = std::sqrt((S(2) * P.lnv) * P.ap);
    P.ey = std::sqrt((S(2) * P.lnv) * P.cp);
    if (!(std::max(P.ex, P.ey) > S(0))) return;                  // (r > 0), L262
    // tile-space bounding box, half-open (L147); tile count (L258)
    const S ts = S(cfg.tile);
    const int32_t TW = (cam.width + cfg.tile - 1) / cfg.tile, TH = (cam.height + cfg.tile - 1) / cfg.tile;
    // fmin/fmax (IEEE: a NaN operand is ignored) so that any input gives an in-range rectangle (C26)
    auto lo = [&](S x, int32_t lim) { return (int32_t)std::fmin(std::fmax(std::floor(x / ts), S(0)), S(lim)); };
    auto hi = [&](S x, int32_t lim) { return (int32_t)std::fmin(std::fmax(std::ceil(x / ts), S(0)), S(lim)); };
    P.rect[0] = lo(P.m[0] - P.ex, TW); P.rect[1] = lo(P.m[1] - P.ey, TH);
    P.rect[2] = hi(P.m[0] + P.ex, TW); P.rect[3] = hi(P.m[1] + P.ey, TH);
    const int64_t tc = (int64_t)(P.rect[2] - P.rect[0]) * (int64_t)(P.rect[3] - P.rect[1]);
    if (!(tc > 0)) return;                                       // (tc > 0), L262
    P.tc = (uint32_t)tc;
    // view-dependent colour (L263, L481; formula absent -> C5)
    S cpos[3];
    for (int j = 0; j < 3; ++j) cpos[j] = -((W[0][j] * t[0] + W[1][j] * t[1]) + W[2][j] * t[2]);
    for (int j = 0; j < 3; ++j) P.dvec[j] = mu[j] - cpos[j];
    P.dnorm = std::sqrt((P.dvec[0] * P.dvec[0] + P.dvec[1] * P.dvec[1]) + P.dvec[2] * P.dvec[2]);
    for (int j = 0; j < 3; ++j) P.dir[j] = P.dvec[j] / P.dnorm;
    sh_basis(P.dir, P.Y);
    const int K = (cfg.sh_degree + 1) * (cfg.sh_degree + 1);
    uint8_t fl = XO_VISIBLE;
    if (P.clamp_u) fl |= XO_CLAMP_U;
    if (P.clamp_v) fl |= XO_CLAMP_V;
    for (int ch = 0; ch < 3; ++ch) {
        S acc = P.Y[0] * sh[ch];
        for (int k = 1; k < K; ++k) acc = acc + P.Y[k] * sh[3 * k + ch];
        P.raw[ch] = acc + S(0.5);
        P.rgb[ch] = std::max(S(0), P.raw[ch]);
        if (P.raw[ch] > S(0)) fl |= (uint8_t)(XO_RGB_POS_R << ch);
    }
    P.flags = fl;
    P.visible = true;
}

template <class S>
void project_all(int64_t N, const S* means, const S* scales, const S* quats, const S* opac, const S* sh,
                 const xo_camera* cam, const xo_config* cfg, S* mean2d, S* conic, S* opac_eff, S* rgb,
                 S* depth, S* lnv, int32_t* rect, uint32_t* tcount, uint8_t* flags) {
    const int K = (cfg->sh_degree + 1) * (cfg->sh_degree + 1);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; ++i) {
        Proj<S> P;
        project_one<S>(means + 3 * i, scales + 3 * i, quats + 4 * i, opac[i], sh + (int64_t)3 * K * i, *cam, *cfg, P);
        if (P.visible) {
            mean2d[2 * i] = P.m[0]; mean2d[2 * i + 1] = P.m[1];
            conic[3 * i] = P.A; conic[3 * i + 1] = P.B; conic[3 * i + 2] = P.C;
            opac_eff[i] = P.o_eff; depth[i] = P.p[2]; lnv[i] = P.lnv;
            for (int c = 0; c < 3; ++c) rgb[3 * i + c] = P.rgb[c];
            for (int c = 0; c < 4; ++c) rect[4 * i + c] = P.rect[c];
            tcount[i] = P.tc; flags[i] = P.flags;
        } else {   // filtered primitive (L82): tile count 0, everything else zero
            mean2d[2 * i] = mean2d[2 * i + 1] = S(0);
            conic[3 * i] = conic[3 * i + 1] = conic[3 * i + 2] = S(0);
            opac_eff[i] = depth[i] = lnv[i] = S(0);
            for (int c = 0; c < 3; ++c) rgb[3 * i + c] = S(0);
            for (int c = 0; c < 4; ++c) rect[4 * i + c] = 0;
            tcount[i] = 0; flags[i] = 0;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// evaluate (PAPER Listing 1) with the pre-scaled conic (C25) and the R3 order:
//   power = fma(fma(qa, dx, qb*dy), dx, (qc*dy)*dy),  qa=-A/2, qb=-B, qc=-C/2.
// ---------------------------------------------------------------------------------------------
template <class S>
inline S eval_power(S A, S B, S C, S mx, S my, S pxc, S pyc, S& dx, S& dy) {
    const S qa = S(-0.5) * A, qb = -B, qc = S(-0.5) * C;
    dx = pxc - mx; dy = pyc - my;
    return std::fma(std::fma(qa, dx, qb * dy), dx, (qc * dy) * dy);
}

// One pixel, front to back over `list[0..len)` (Alg. 1; C12 test-before-blend).
// Optionally records the contributing sequence for the backward pass.
template <class S>
struct Contrib { uint32_t pos, g; S alpha, T, G, dx, dy; bool clamped; };

template <class S>
void composite_pixel(const xo_config& cfg, const S* mean2d, const S* conic, const S* opac, const S* rgb,
                     const S* lnv, const uint32_t* list, uint32_t len, S pxc, S pyc, S out_rgb[3], S& out_T,
                     uint32_t& out_n, uint8_t* fragile, int64_t* visit, int64_t* pass,
                     std::vector<Contrib<S>>* rec, uint32_t limit) {
    S T = S(1), C[3] = {S(0), S(0), S(0)};
    uint32_t last = 0;
    uint8_t frag = 0;
    const S amax = S(cfg.alpha_max), tmin = S(cfg.t_min);
    const double fr = cfg.fragile_rel;
    const uint32_t stop = std::min(len, limit);
    for (uint32_t k = 0; k < stop; ++k) {
        const uint32_t g = list[k];
        S dx, dy;
        const S power = eval_power<S>(conic[3 * g], conic[3 * g + 1], conic[3 * g + 2], mean2d[2 * g],
                                      mean2d[2 * g + 1], pxc, pyc, dx, dy);
        if (visit) ++*visit;
        const S thr = -lnv[g];
        {   // margins of the power-based decisions (only used by precision-changing pins)
            const double scale = std::max({std::fabs((double)conic[3 * g] * dx * dx), std::fabs((double)conic[3 * g + 2] * dy * dy),
                                           std::fabs((double)conic[3 * g + 1] * dx * dy), 1e-30});
            if (std::fabs((double)power - (double)thr) <= fr * std::max(scale, std::fabs((double)thr))) frag |= XO_FRAG_GATE;
        }
        if (power > S(0)) continue;                       // valid = power <= 0 (L289, C20)
        if (power < thr) continue;                        // alpha < alpha_thresh (L679, C12)
        if (pass) ++*pass;
        const S G = std::exp(power);
        const S og = opac[g] * G;
        const S alpha = std::min(amax, og);               // C11
        if (std::fabs((double)og - (double)amax) <= fr * (double)amax) frag |= XO_FRAG_CLAMP;
        const S Tn = T * (S(1) - alpha);
        if (std::fabs((double)Tn - (double)tmin) <= fr * (double)tmin) frag |= XO_FRAG_EXIT;
        if (Tn < tmin) break;                             // C12: stop without blending
        const S w = alpha * T;
        for (int c = 0; c < 3; ++c) C[c] = C[c] + rgb[3 * g + c] * w;
        if (rec) rec->push_back({k, g, alpha, T, G, dx, dy, !(og < amax)});
        T = Tn;
        last = k + 1;
    }
    for (int c = 0; c < 3; ++c) out_rgb[c] = C[c] + T * S(cfg.bg[c]);   // C13
    out_T = T; out_n = last;
    if (fragile) *fragile = frag;
}

template <class S>
void rasterize_fwd(const xo_camera* cam, const xo_config* cfg, const S* mean2d, const S* conic, const S* opac,
                   const S* rgb, const S* lnv, const uint32_t* vals, const uint32_t* ranges, S* image, S* final_T,
                   uint32_t* n_contrib, uint8_t* fragile, int64_t* counters) {
    const int W = cam->width, H = cam->height, ts = cfg->tile;
    const int TW = (W + ts - 1) / ts, TH = (H + ts - 1) / ts;
    int64_t visit = 0, pass = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : visit, pass)
    for (int t = 0; t < TW * TH; ++t) {
        const int tx = t % TW, ty = t / TW;
        const uint32_t b = ranges[2 * t], e = ranges[2 * t + 1];
        for (int py = ty * ts; py < std::min(H, (ty + 1) * ts); ++py)
            for (int px = tx * ts; px < std::min(W, (tx + 1) * ts); ++px) {
                const int64_t pid = (int64_t)py * W + px;
                S c[3], T; uint32_t n; uint8_t fr = 0; int64_t v = 0, p = 0;
                composite_pixel<S>(*cfg, mean2d, conic, opac, rgb, lnv, vals + b, e - b, S(px) + S(0.5),
                                   S(py) + S(0.5), c, T, n, &fr, &v, &p, nullptr, 0xffffffffu);
                for (int k = 0; k < 3; ++k) image[3 * pid + k] = c[k];
                final_T[pid] = T; n_contrib[pid] = n;
                if (fragile) fragile[pid] = fr;
                visit += v; pass += p;
            }
    }
    if (counters) { counters[0] = visit; counters[1] = pass; }
}

// Strict mode: the pixel's own list = all visible primitives whose tile rectangle contains the
// pixel's tile, sorted by (depth, index) (L84 "depth-sorted list of contributing primitives").
template <class S>
void rasterize_fwd_strict(const xo_camera* cam, const xo_config* cfg, int64_t N, const S* mean2d, const S* conic,
                          const S* opac, const S* rgb, const S* lnv, const S* depth, const int32_t* rect,
                          const uint32_t* tcount, S* image, S* final_T, uint32_t* n_contrib) {
    const int W = cam->width, H = cam->height, ts = cfg->tile;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t pid = 0; pid < (int64_t)W * H; ++pid) {
        const int px = (int)(pid % W), py = (int)(pid / W);
        const int tx = px / ts, ty = py / ts;
        std::vector<uint32_t> list;
        for (int64_t g = 0; g < N; ++g)
            if (tcount[g] > 0 && tx >= rect[4 * g] && tx < rect[4 * g + 2] && ty >= rect[4 * g + 1] && ty < rect[4 * g + 3])
                list.push_back((uint32_t)g);
        std::stable_sort(list.begin(), list.end(), [&](uint32_t x, uint32_t y) {
            if (depth[x] != depth[y]) return depth[x] < depth[y];
            return x < y;
        });
        S c[3], T; uint32_t n;
        composite_pixel<S>(*cfg, mean2d, conic, opac, rgb, lnv, list.data(), (uint32_t)list.size(), S(px) + S(0.5),
                           S(py) + S(0.5), c, T, n, nullptr, nullptr, nullptr, nullptr, 0xffffffffu);
        for (int k = 0; k < 3; ++k) image[3 * pid + k] = c[k];
        final_T[pid] = T; n_contrib[pid] = n;
    }
}

// Reverse mode through compositing.  For the contributing sequence k = 1..n of a pixel with
// c(x,y) = sum_k c_k alpha_k T_k + T_final bg (L86, C13), and S_k = sum_{j>k} c_j alpha_j T_j + T_final bg:
//   dL/dc_k = alpha_k T_k g;   dL/dalpha_k = sum_ch g_ch (c_k T_k - S_k / (1 - alpha_k));
//   alpha = min(amax, o G): clamp active -> no gradient to o, power (C14); G = exp(power);
//   dL/do = G dL/dalpha;  dL/dpower = o G dL/dalpha;
//   power = -1/2 (A dx^2 + C dy^2) - B dx dy, dx = px - m_x:
//   dL/dA = -1/2 dx^2 dL/dpower, dL/dB = -dx dy dL/dpower, dL/dC = -1/2 dy^2 dL/dpower,
//   dL/dm_x = (A dx + B dy) dL/dpower, dL/dm_y = (B dx + C dy) dL/dpower.
// Gates and the exit are piecewise constant (C15).
// MASS = true accumulates |addend| instead of the addend: the "mass" sum_pixels |term| of every
// gradient element, i.e. the scale an fp32 sum of those terms is conditioned on (used only to
// derive the cancellation-aware part of the gradient tolerance).
// ACC = float: every sum of this function (per list position over the tile's pixels, then over the tiles) is kept in
// fp32 instead of fp64, in this function's fixed order -- what a careful fp32 CPU implementation would return.  Used
// only to put the GPU's fp32 summation error beside that of a CPU fp32 sum (tests/test_gpu_parity.py).
template <class S, bool MASS = false, class ACC = double>
void rasterize_bwd(const xo_camera* cam, const xo_config* cfg, int64_t N, const S* mean2d, const S* conic, const S* opac,
                   const S* rgb, const S* lnv, const uint32_t* vals, const uint32_t* ranges, const uint32_t* n_contrib,
                   const S* dL, double* g_mean2d, double* g_conic, double* g_opac, double* g_rgb) {
    const int W = cam->width, H = cam->height, ts = cfg->tile;
    const int TW = (W + ts - 1) / ts, TH = (H + ts - 1) / ts;
    std::fill(g_mean2d, g_mean2d + 2 * N, 0.0); std::fill(g_conic, g_conic + 3 * N, 0.0);
    std::fill(g_opac, g_opac + N, 0.0); std::fill(g_rgb, g_rgb + 3 * N, 0.0);
#pragma omp parallel for schedule(dynamic, 1)
    for (int t = 0; t < TW * TH; ++t) {
        const int tx = t % TW, ty = t / TW;
        const uint32_t b = ranges[2 * t], e = ranges[2 * t + 1];
        if (e <= b) continue;
        std::vector<ACC> acc((size_t)(e - b) * 9, ACC(0));   // per list position: m(2) conic(3) o(1) rgb(3)
        std::vector<Contrib<S>> rec;
        for (int py = ty * ts; py < std::min(H, (ty + 1) * ts); ++py)
            for (int px = tx * ts; px < std::min(W, (tx + 1) * ts); ++px) {
                const int64_t pid = (int64_t)py * W + px;
                rec.clear();
                S c[3], T; uint32_t n;
                composite_pixel<S>(*cfg, mean2d, conic, opac, rgb, lnv, vals + b, e - b, S(px) + S(0.5), S(py) + S(0.5), c,
                                   T, n, nullptr, nullptr, nullptr, &rec, n_contrib[pid]);
                const double g[3] = {(double)dL[3 * pid], (double)dL[3 * pid + 1], (double)dL[3 * pid + 2]};
                double Sb[3] = {(double)T * cfg->bg[0], (double)T * cfg->bg[1], (double)T * cfg->bg[2]};
                for (size_t r = rec.size(); r-- > 0;) {
                    const Contrib<S>& q = rec[r];
                    const double al = (double)q.alpha, Tk = (double)q.T;
                    ACC* a9 = &acc[(size_t)q.pos * 9];
                    double dalpha = 0.0;
                    for (int ch = 0; ch < 3; ++ch) {
                        const double ck = (double)rgb[3 * q.g + ch];
                        a9[6 + ch] += ACC(MASS ? std::fabs(al * Tk * g[ch]) : al * Tk * g[ch]);
                        dalpha += g[ch] * (ck * Tk - Sb[ch] / (1.0 - al));
                    }
                    for (int ch = 0; ch < 3; ++ch) Sb[ch] += (double)rgb[3 * q.g + ch] * al * Tk;
                    if (q.clamped) continue;
                    const double G = (double)q.G, o = (double)opac[q.g];
                    const double dpow = o * G * dalpha;
                    const double A = (double)conic[3 * q.g], B = (double)conic[3 * q.g + 1], C = (double)conic[3 * q.g + 2];
                    const double dx = (double)q.dx, dy = (double)q.dy;
                    const double add[6] = {(A * dx + B * dy) * dpow, (B * dx + C * dy) * dpow,   // d power / d m = A dx + B dy, ..
                                           -0.5 * dx * dx * dpow, -dx * dy * dpow, -0.5 * dy * dy * dpow, G * dalpha};
                    for (int j = 0; j < 6; ++j) a9[j] += ACC(MASS ? std::fabs(add[j]) : add[j]);
                }
            }
        for (uint32_t k = 0; k < e - b; ++k) {
            const uint32_t gi = vals[b + k];
            const ACC* a9 = &acc[(size_t)k * 9];
            bool any = false;
            for (int j = 0; j < 9; ++j) any |= (a9[j] != ACC(0));
            if (!any) continue;
            if (sizeof(ACC) == 4) {   // fp32 sum over the tiles too, serialised (order = whichever tile arrives first)
#pragma omp critical(xo_acc32)
                {
                    g_mean2d[2 * gi] = (double)((float)g_mean2d[2 * gi] + (float)a9[0]);
                    g_mean2d[2 * gi + 1] = (double)((float)g_mean2d[2 * gi + 1] + (float)a9[1]);
                    for (int j = 0; j < 3; ++j) g_conic[3 * gi + j] = (double)((float)g_conic[3 * gi + j] + (float)a9[2 + j]);
                    g_opac[gi] = (double)((float)g_opac[gi] + (float)a9[5]);
                    for (int j = 0; j < 3; ++j) g_rgb[3 * gi + j] = (double)((float)g_rgb[3 * gi + j] + (float)a9[6 + j]);
                }
                continue;
            }
#pragma omp atomic
            g_mean2d[2 * gi] += a9[0];
#pragma omp atomic
            g_mean2d[2 * gi + 1] += a9[1];
#pragma omp atomic
            g_conic[3 * gi] += a9[2];
#pragma omp atomic
            g_conic[3 * gi + 1] += a9[3];
#pragma omp atomic
            g_conic[3 * gi + 2] += a9[4];
#pragma omp atomic
            g_opac[gi] += a9[5];
#pragma omp atomic
            g_rgb[3 * gi] += a9[6];
#pragma omp atomic
            g_rgb[3 * gi + 1] += a9[7];
#pragma omp atomic
            g_rgb[3 * gi + 2] += a9[8];
        }
    }
}

// Reverse mode through projection + SH; all chain-rule arithmetic in fp64 on the forward
// intermediates recomputed in S (so that clamps / culling decisions equal the forward's).
template <class S>
void project_bwd_one(const S mu[3], const S sc[3], const S q[4], S o, const S* sh, const xo_camera& cam,
                     const xo_config& cfg, const double gm[2], const double gK[3], double go_eff, const double grgb[3],
                     double g_mu[3], double g_s[3], double g_q[4], double& g_o, double* g_sh) {
    const int K = (cfg.sh_degree + 1) * (cfg.sh_degree + 1);
    for (int j = 0; j < 3; ++j) g_mu[j] = g_s[j] = 0.0;
    for (int j = 0; j < 4; ++j) g_q[j] = 0.0;
    g_o = 0.0;
    for (int j = 0; j < 3 * K; ++j) g_sh[j] = 0.0;
    Proj<S> P;
    project_one<S>(mu, sc, q, o, sh, cam, cfg, P);
    if (!P.visible) return;                                      // culled -> exactly zero (P11)
    double W[3][3];
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) W[i][j] = cam.w2c[4 * i + j];
    // conic -> filtered covariance:  G2 = -K G_K K  (K = cov'^-1, symmetric-matrix gradients)
    const double A = P.A, B = P.B, C = P.C;
    const double GK[2][2] = {{gK[0], 0.5 * gK[1]}, {0.5 * gK[1], gK[2]}};
    const double Km[2][2] = {{A, B}, {B, C}};
    double tmp[2][2], G2[2][2];
    for (int i = 0; i < 2; ++i) for (int j = 0; j < 2; ++j) tmp[i][j] = Km[i][0] * GK[0][j] + Km[i][1] * GK[1][j];
    for (int i = 0; i < 2; ++i) for (int j = 0; j < 2; ++j) G2[i][j] = -(tmp[i][0] * Km[0][j] + tmp[i][1] * Km[1][j]);
    double g_a = G2[0][0], g_b = 2.0 * G2[0][1], g_c = G2[1][1];   // w.r.t. scalars a, b, c of cov_raw
    // opacity (C19)
    if (cfg.antialias) {
        const double rho = P.rho, a = P.a, b = P.b, c = P.c, ap = P.ap, cp = P.cp;
        g_o = go_eff * rho;
        if (rho > 0.0) {
            const double g_rho = go_eff * (double)o;
            const double g_draw = g_rho * 0.5 * rho / (double)P.det_raw, g_det = -g_rho * 0.5 * rho / (double)P.det;
            g_a += g_draw * c + g_det * cp; g_c += g_draw * a + g_det * ap; g_b += -2.0 * b * (g_draw + g_det);
        }
    } else g_o = go_eff;
    const double Gs[2][2] = {{g_a, 0.5 * g_b}, {0.5 * g_b, g_c}};   // dL/dcov_raw as a symmetric matrix
    double gSig[3][3] = {{0}}, gM[3][3] = {{0}};
    double g_p[3] = {0, 0, 0};                                      // dL/d(camera-space mean)
    if (cfg.projection == 0) {
        double T[2][3], Sig[3][3];
        for (int r = 0; r < 2; ++r) for (int j = 0; j < 3; ++j) T[r][j] = P.T[r][j];
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) Sig[i][j] = P.Sig[i][j];
        // dL/dSigma = T^T Gs T ; dL/dT = 2 Gs T Sigma ; dL/dJ = dL/dT W^T
        double GT[2][3];
        for (int r = 0; r < 2; ++r) for (int j = 0; j < 3; ++j) GT[r][j] = Gs[r][0] * T[0][j] + Gs[r][1] * T[1][j];
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) gSig[i][j] = T[0][i] * GT[0][j] + T[1][i] * GT[1][j];
        double gT[2][3];
        for (int r = 0; r < 2; ++r) for (int j = 0; j < 3; ++j)
            gT[r][j] = 2.0 * (GT[r][0] * Sig[0][j] + GT[r][1] * Sig[1][j] + GT[r][2] * Sig[2][j]);
        double gJ[2][3];
        for (int r = 0; r < 2; ++r) for (int j = 0; j < 3; ++j) gJ[r][j] = gT[r][0] * W[j][0] + gT[r][1] * W[j][1] + gT[r][2] * W[j][2];
        const double x = P.p[0], y = P.p[1], z = P.p[2], fx = cam.fx, fy = cam.fy, u = P.u, v = P.v;
        // J00 = fx/z, J11 = fy/z, J02 = -fx u/z, J12 = -fy v/z
        g_p[2] += gJ[0][0] * (-fx / (z * z)) + gJ[1][1] * (-fy / (z * z));
        g_p[2] += gJ[0][2] * (fx * u / (z * z)) + gJ[1][2] * (fy * v / (z * z));
        const double g_u = gJ[0][2] * (-fx / z), g_v = gJ[1][2] * (-fy / z);
        if (!P.clamp_u) { g_p[0] += g_u / z; g_p[2] += -g_u * x / (z * z); }   // C16
        if (!P.clamp_v) { g_p[1] += g_v / z; g_p[2] += -g_v * y / (z * z); }
        // mean2d = (fx x/z + cx, fy y/z + cy), unclamped
        g_p[0] += gm[0] * fx / z; g_p[1] += gm[1] * fy / z;
        g_p[2] += -gm[0] * fx * x / (z * z) - gm[1] * fy * y / (z * z);
        for (int j = 0; j < 3; ++j) g_mu[j] += W[0][j] * g_p[0] + W[1][j] * g_p[1] + W[2][j] * g_p[2];
        // Sigma = M M^T  ->  dL/dM = 2 dL/dSigma M (dL/dSigma symmetric)
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j)
            gM[i][j] = 2.0 * (gSig[i][0] * (double)P.M[0][j] + gSig[i][1] * (double)P.M[1][j] + gSig[i][2] * (double)P.M[2][j]);
    } else {
        // UT: m = sum wm_k y_k ; cov = sum wc_k (y_k - m)(y_k - m)^T
        //   g_tot = g_m - 2 sum_j wc_j Gs (y_j - m);  dL/dy_k = wm_k g_tot + 2 wc_k Gs (y_k - m)
        double gtot[2] = {gm[0], gm[1]};
        double dk[7][2];
        for (int k = 0; k < 7; ++k) {
            dk[k][0] = (double)P.y[k][0] - (double)P.m[0]; dk[k][1] = (double)P.y[k][1] - (double)P.m[1];
            for (int r = 0; r < 2; ++r) gtot[r] -= 2.0 * (double)P.wc[k] * (Gs[r][0] * dk[k][0] + Gs[r][1] * dk[k][1]);
        }
        double gx[7][3];
        for (int k = 0; k < 7; ++k) {
            double gy[2];
            for (int r = 0; r < 2; ++r) gy[r] = (double)P.wm[k] * gtot[r] + 2.0 * (double)P.wc[k] * (Gs[r][0] * dk[k][0] + Gs[r][1] * dk[k][1]);
            const double pc[3] = {(double)P.pc[k][0], (double)P.pc[k][1], (double)P.pc[k][2]};
            double Jp[2][3];
            camera_project_jac(cam, pc, Jp);
            double gpc[3];
            for (int j = 0; j < 3; ++j) gpc[j] = Jp[0][j] * gy[0] + Jp[1][j] * gy[1];
            for (int j = 0; j < 3; ++j) gx[k][j] = W[0][j] * gpc[0] + W[1][j] * gpc[1] + W[2][j] * gpc[2];
            for (int j = 0; j < 3; ++j) g_mu[j] += gx[k][j];
        }
        // x_{+-j} = mu +- gamma M[:,j]  ->  dL/dM[:,j] = gamma (gx_{+j} - gx_{-j})
        for (int j = 0; j < 3; ++j) for (int d = 0; d < 3; ++d)
            gM[d][j] = (double)P.gamma * (gx[1 + 2 * j][d] - gx[2 + 2 * j][d]);
    }
    // M = R diag(s)
    double gR[3][3];
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) { g_s[j] += (double)P.R[i][j] * gM[i][j]; gR[i][j] = (double)sc[j] * gM[i][j]; }
    // R(q), four free components (C17)
    const double w = q[0], x = q[1], y = q[2], z = q[3];
    g_q[0] = 2.0 * (-z * gR[0][1] + y * gR[0][2] + z * gR[1][0] - x * gR[1][2] - y * gR[2][0] + x * gR[2][1]);
    g_q[1] = 2.0 * (y * gR[0][1] + z * gR[0][2] + y * gR[1][0] - 2.0 * x * gR[1][1] - w * gR[1][2] + z * gR[2][0] + w * gR[2][1] - 2.0 * x * gR[2][2]);
    g_q[2] = 2.0 * (-2.0 * y * gR[0][0] + x * gR[0][1] + w * gR[0][2] + x * gR[1][0] + z * gR[1][2] - w * gR[2][0] + z * gR[2][1] - 2.0 * y * gR[2][2]);
    g_q[3] = 2.0 * (-2.0 * z * gR[0][0] - w * gR[0][1] + x * gR[0][2] + w * gR[1][0] - 2.0 * z * gR[1][1] + y * gR[1][2] + x * gR[2][0] + y * gR[2][1]);
    // colour: rgb = max(0, 1/2 + sum_k Y_k(d) sh_k), d = (mu - cam_pos)/|mu - cam_pos|
    double gd[3] = {0, 0, 0}, dY[16][3];
    const double dir[3] = {(double)P.dir[0], (double)P.dir[1], (double)P.dir[2]};
    sh_basis_grad(dir, dY);
    for (int ch = 0; ch < 3; ++ch) {
        if (!(P.raw[ch] > S(0))) continue;                         // C16 mask
        for (int k = 0; k < K; ++k) {
            g_sh[3 * k + ch] = (double)P.Y[k] * grgb[ch];
            for (int j = 0; j < 3; ++j) gd[j] += dY[k][j] * (double)sh[3 * k + ch] * grgb[ch];
        }
    }
    const double dot = dir[0] * gd[0] + dir[1] * gd[1] + dir[2] * gd[2];
    for (int j = 0; j < 3; ++j) g_mu[j] += (gd[j] - dir[j] * dot) / (double)P.dnorm;
}

template <class S>
void project_bwd_all(int64_t N, const S* means, const S* scales, const S* quats, const S* opac, const S* sh,
                     const xo_camera* cam, const xo_config* cfg, const double* g_mean2d, const double* g_conic,
                     const double* g_opac_eff, const double* g_rgb, double* g_means, double* g_scales, double* g_quats,
                     double* g_opac, double* g_sh) {
    const int K = (cfg->sh_degree + 1) * (cfg->sh_degree + 1);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; ++i)
        project_bwd_one<S>(means + 3 * i, scales + 3 * i, quats + 4 * i, opac[i], sh + (int64_t)3 * K * i, *cam, *cfg,
                           g_mean2d + 2 * i, g_conic + 3 * i, g_opac_eff[i], g_rgb + 3 * i, g_means + 3 * i,
                           g_scales + 3 * i, g_quats + 4 * i, g_opac[i], g_sh + (int64_t)3 * K * i);
}

inline uint32_t float_bits(float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; }

}  // namespace

// ---------------------------------------------------------------------------------------------
// C entry points
// ---------------------------------------------------------------------------------------------
#define XO_DEF(SFX, T)                                                                                              \
    extern "C" void xpr_oracle_project_##SFX(int64_t N, const T* means, const T* scales, const T* quats,            \
                                             const T* opacities, const T* sh, const xo_camera* cam,                 \
                                             const xo_config* cfg, T* mean2d, T* conic, T* opac_eff, T* rgb,        \
                                             T* depth, T* lnv, int32_t* tile_rect, uint32_t* tile_count,            \
                                             uint8_t* flags) {                                                      \
        project_all<T>(N, means, scales, quats, opacities, sh, cam, cfg, mean2d, conic, opac_eff, rgb, depth, lnv,  \
                       tile_rect, tile_count, flags);                                                               \
    }                                                                                                               \
    extern "C" void xpr_oracle_rasterize_fwd_##SFX(const xo_camera* cam, const xo_config* cfg, int64_t N,           \
                                                   const T* mean2d, const T* conic, const T* opac_eff,              \
                                                   const T* rgb, const T* lnv, const uint32_t* vals_sorted,         \
                                                   const uint32_t* tile_ranges, T* image, T* final_T,               \
                                                   uint32_t* n_contrib, uint8_t* fragile, int64_t* counters) {      \
        (void)N;                                                                                                    \
        rasterize_fwd<T>(cam, cfg, mean2d, conic, opac_eff, rgb, lnv, vals_sorted, tile_ranges, image, final_T,     \
                         n_contrib, fragile, counters);                                                             \
    }                                                                                                               \
    extern "C" void xpr_oracle_rasterize_fwd_strict_##SFX(                                                          \
        const xo_camera* cam, const xo_config* cfg, int64_t N, const T* mean2d, const T* conic, const T* opac_eff,  \
        const T* rgb, const T* lnv, const T* depth, const int32_t* tile_rect, const uint32_t* tile_count, T* image, \
        T* final_T, uint32_t* n_contrib) {                                                                          \
        rasterize_fwd_strict<T>(cam, cfg, N, mean2d, conic, opac_eff, rgb, lnv, depth, tile_rect, tile_count,       \
                                image, final_T, n_contrib);                                                         \
    }                                                                                                               \
    extern "C" void xpr_oracle_rasterize_bwd_##SFX(                                                                 \
        const xo_camera* cam, const xo_config* cfg, int64_t N, const T* mean2d, const T* conic, const T* opac_eff,  \
        const T* rgb, const T* lnv, const uint32_t* vals_sorted, const uint32_t* tile_ranges,                       \
        const uint32_t* n_contrib, const T* dL_dimage, double* g_mean2d, double* g_conic, double* g_opac_eff,       \
        double* g_rgb) {                                                                                            \
        rasterize_bwd<T>(cam, cfg, N, mean2d, conic, opac_eff, rgb, lnv, vals_sorted, tile_ranges, n_contrib,       \
                         dL_dimage, g_mean2d, g_conic, g_opac_eff, g_rgb);                                          \
    }                                                                                                               \
    extern "C" void xpr_oracle_rasterize_bwd_mass_##SFX(                                                            \
        const xo_camera* cam, const xo_config* cfg, int64_t N, const T* mean2d, const T* conic, const T* opac_eff,  \
        const T* rgb, const T* lnv, const uint32_t* vals_sorted, const uint32_t* tile_ranges,                       \
        const uint32_t* n_contrib, const T* dL_dimage, double* g_mean2d, double* g_conic, double* g_opac_eff,       \
        double* g_rgb) {                                                                                            \
        rasterize_bwd<T, true>(cam, cfg, N, mean2d, conic, opac_eff, rgb, lnv, vals_sorted, tile_ranges, n_contrib, \
                               dL_dimage, g_mean2d, g_conic, g_opac_eff, g_rgb);                                    \
    }                                                                                                               \
    extern "C" void xpr_oracle_rasterize_bwd_acc32_##SFX(                                                           \
        const xo_camera* cam, const xo_config* cfg, int64_t N, const T* mean2d, const T* conic, const T* opac_eff,  \
        const T* rgb, const T* lnv, const uint32_t* vals_sorted, const uint32_t* tile_ranges,                       \
        const uint32_t* n_contrib, const T* dL_dimage, double* g_mean2d, double* g_conic, double* g_opac_eff,       \
        double* g_rgb) {                                                                                            \
        rasterize_bwd<T, false, float>(cam, cfg, N, mean2d, conic, opac_eff, rgb, lnv, vals_sorted, tile_ranges,    \
                                       n_contrib, dL_dimage, g_mean2d, g_conic, g_opac_eff, g_rgb);                 \
    }                                                                                                               \
    extern "C" void xpr_oracle_project_bwd_##SFX(                                                                   \
        int64_t N, const T* means, const T* scales, const T* quats, const T* opacities, const T* sh,                \
        const xo_camera* cam, const xo_config* cfg, const double* g_mean2d, const double* g_conic,                  \
        const double* g_opac_eff, const double* g_rgb, double* g_means, double* g_scales, double* g_quats,          \
        double* g_opacities, double* g_sh) {                                                                        \
        project_bwd_all<T>(N, means, scales, quats, opacities, sh, cam, cfg, g_mean2d, g_conic, g_opac_eff, g_rgb,  \
                           g_means, g_scales, g_quats, g_opacities, g_sh);                                          \
    }                                                                                                               \
    extern "C" void xpr_oracle_sh_basis_##SFX(const T* dir, T* out16) { sh_basis<T>(dir, out16); }                  \
    extern "C" void xpr_oracle_camera_project_##SFX(const xo_camera* cam, const T* p_cam, T* pix2) {                \
        camera_project<T>(*cam, p_cam, pix2);                                                                       \
    }

XO_DEF(f32, float)
XO_DEF(f64, double)

// Replicate + assign tile id: primitive i appears tc_i times; for local offset r,
// w_i = x_max - x_min, x = x_min + (r mod w_i), y = y_min + floor(r / w_i), t = y W' + x.
// key = tile << 32 | float bits of depth (BASELINE.json:north_star, C10); value = i.
extern "C" int64_t xpr_oracle_emit(int64_t N, const float* depth, const int32_t* rect, const uint32_t* tcount,
                                   int32_t tiles_x, int64_t capacity, uint64_t* keys, uint32_t* vals) {
    int64_t I = 0;
    for (int64_t i = 0; i < N; ++i) {
        const uint32_t tc = tcount[i];
        if (tc == 0) continue;
        const int32_t w = rect[4 * i + 2] - rect[4 * i];
        for (uint32_t r = 0; r < tc; ++r) {
            if (I < capacity) {
                const int32_t x = rect[4 * i] + (int32_t)(r % (uint32_t)w);
                const int32_t y = rect[4 * i + 1] + (int32_t)(r / (uint32_t)w);
                const uint64_t t = (uint64_t)y * (uint64_t)tiles_x + (uint64_t)x;
                keys[I] = (t << 32) | (uint64_t)float_bits(depth[i]);
                vals[I] = (uint32_t)i;
            }
            ++I;
        }
    }
    return I;
}

// ---------------------------------------------------------------------------------------------
// tile_cull of XPR-3DGS ("Cull", Listing 1, A.1.1 L435; StopThePop): keep the pair
// (primitive, tile) iff the maximum of alpha = o G_2D(x) over the tile reaches alpha_thresh, i.e. iff
//   min_{x in tile} 1/2 (x - mu)^T K (x - mu) <= ln(o / alpha_thresh) = lnv,   K = [[A, B], [B, C]].
// "Tile" is the hull of the tile's pixel centres [ts*tx + 1/2, ts*tx + ts - 1/2]^2 (reading C8, C1).
// The minimiser is mu when mu is inside, else it lies on an edge facing mu (the response falls off
// along every ray from mu, L435): on the vertical edge x = xe the minimiser over y is
// dy = clamp(-B dx / C, ...), on the horizontal edge y = ye it is dx = clamp(-B dy / A, ...).
// fp32 evaluation order and the conservative margin are fixed in DESIGN.md reading C8: a pair is
// dropped only if q > lnv + 2^-18 (|a| + |b| + |c| + lnv), with q = (a + b) + c,
// a = ((A/2) dx) dx, b = (B dx) dy, c = ((C/2) dy) dy.  Written so that a NaN keeps the pair.
// ---------------------------------------------------------------------------------------------
template <class S>
bool tile_keep(S mx, S my, S A, S B, S C, S lnv, int32_t tx, int32_t ty, int32_t ts) {
    const S x0 = S(ts) * S(tx) + S(0.5), x1 = (S(ts) * S(tx) + S(ts)) - S(0.5);
    const S y0 = S(ts) * S(ty) + S(0.5), y1 = (S(ts) * S(ty) + S(ts)) - S(0.5);
    const bool in_x = (mx >= x0) && (mx <= x1), in_y = (my >= y0) && (my <= y1);
    if (in_x && in_y) return true;
    const S margin = S(1.0 / 262144.0);   // 2^-18
    auto drop = [&](S dx, S dy) {
        const S a = ((S(0.5) * A) * dx) * dx, b = (B * dx) * dy, c = ((S(0.5) * C) * dy) * dy;
        const S q = (a + b) + c;
        const S mag = ((std::fabs(a) + std::fabs(b)) + std::fabs(c)) + lnv;
        return q > lnv + mag * margin;
    };
    bool dropped = true;                   // dropped by every facing edge
    if (!in_x) {
        const S dx = ((mx < x0) ? x0 : x1) - mx;
        S dy = (-(B * dx)) / C;
        const S lo = y0 - my, hi = y1 - my;
        dy = (dy < lo) ? lo : dy; dy = (hi < dy) ? hi : dy;
        dropped = dropped && drop(dx, dy);
    }
    if (!in_y) {
        const S dy = ((my < y0) ? y0 : y1) - my;
        S dx = (-(B * dy)) / A;
        const S lo = x0 - mx, hi = x1 - mx;
        dx = (dx < lo) ? lo : dx; dx = (hi < dx) ? hi : dx;
        dropped = dropped && drop(dx, dy);
    }
    return !dropped;
}

#define XO_KEEP(S, T)                                                                                     \
    extern "C" void xpr_oracle_tile_keep_##S(int64_t n, const T* mean2d, const T* conic, const T* lnv,     \
                                             const int32_t* tile_xy, int32_t ts, uint8_t* keep) {          \
        for (int64_t i = 0; i < n; ++i)                                                                   \
            keep[i] = tile_keep<T>(mean2d[2 * i], mean2d[2 * i + 1], conic[3 * i], conic[3 * i + 1],       \
                                   conic[3 * i + 2], lnv[i], tile_xy[2 * i], tile_xy[2 * i + 1], ts) ? 1 : 0; \
    }
XO_KEEP(f32, float)
XO_KEEP(f64, double)

// Replicate + assign tile id + cull: as xpr_oracle_emit, but a pair that fails tile_cull
// is not emitted (the paper keeps its slot with tile id T so that it sorts behind every tile and
// belongs to no segment; dropping it gives the same per-tile segments).  Decisions in fp32.
extern "C" int64_t xpr_oracle_emit_cull(int64_t N, const float* depth, const int32_t* rect, const uint32_t* tcount,
                                        const float* mean2d, const float* conic, const float* lnv, int32_t tiles_x,
                                        int32_t ts, int64_t capacity, uint64_t* keys, uint32_t* vals) {
    int64_t I = 0;
    for (int64_t i = 0; i < N; ++i) {
        const uint32_t tc = tcount[i];
        if (tc == 0) continue;
        const int32_t w = rect[4 * i + 2] - rect[4 * i];
        for (uint32_t r = 0; r < tc; ++r) {
            const int32_t x = rect[4 * i] + (int32_t)(r % (uint32_t)w);
            const int32_t y = rect[4 * i + 1] + (int32_t)(r / (uint32_t)w);
            if (!tile_keep<float>(mean2d[2 * i], mean2d[2 * i + 1], conic[3 * i], conic[3 * i + 1], conic[3 * i + 2],
                                  lnv[i], x, y, ts))
                continue;
            if (I < capacity) {
                const uint64_t t = (uint64_t)y * (uint64_t)tiles_x + (uint64_t)x;
                keys[I] = (t << 32) | (uint64_t)float_bits(depth[i]);
                vals[I] = (uint32_t)i;
            }
            ++I;
        }
    }
    return I;
}

// Sort by (tile, depth) and identify bounds.  Stable sort on index-ordered emission
// gives the tie-break "lower primitive index first" (C10).  Empty tiles get (0, 0).
static void sort_and_bounds(int64_t I, const std::vector<uint64_t>& keys, const std::vector<uint32_t>& vals,
                            int32_t tiles_x, int32_t tiles_y, uint64_t* keys_sorted, uint32_t* vals_sorted,
                            uint32_t* ranges) {
    std::vector<uint32_t> perm((size_t)I);
    std::iota(perm.begin(), perm.end(), 0u);
    std::stable_sort(perm.begin(), perm.end(), [&](uint32_t x, uint32_t y) { return keys[x] < keys[y]; });
    for (int64_t j = 0; j < I; ++j) { keys_sorted[j] = keys[perm[j]]; vals_sorted[j] = vals[perm[j]]; }
    const int64_t T = (int64_t)tiles_x * tiles_y;
    for (int64_t t = 0; t < 2 * T; ++t) ranges[t] = 0;
    for (int64_t j = 0; j < I; ++j) {
        const uint64_t t = keys_sorted[j] >> 32;
        if (j == 0 || (keys_sorted[j - 1] >> 32) != t) ranges[2 * t] = (uint32_t)j;
        if (j == I - 1 || (keys_sorted[j + 1] >> 32) != t) ranges[2 * t + 1] = (uint32_t)(j + 1);
    }
}

extern "C" int64_t xpr_oracle_bin_sort(int64_t N, const float* depth, const int32_t* rect, const uint32_t* tcount,
                                       int32_t tiles_x, int32_t tiles_y, int64_t capacity, uint64_t* keys_sorted,
                                       uint32_t* vals_sorted, uint32_t* ranges) {
    const int64_t I = xpr_oracle_emit(N, depth, rect, tcount, tiles_x, 0, nullptr, nullptr);
    if (capacity < I) return I;
    std::vector<uint64_t> keys((size_t)I);
    std::vector<uint32_t> vals((size_t)I);
    xpr_oracle_emit(N, depth, rect, tcount, tiles_x, I, keys.data(), vals.data());
    sort_and_bounds(I, keys, vals, tiles_x, tiles_y, keys_sorted, vals_sorted, ranges);
    return I;
}

// The same with tile_cull ("Cull"): returns the number of surviving pairs.
extern "C" int64_t xpr_oracle_bin_sort_cull(int64_t N, const float* depth, const int32_t* rect, const uint32_t* tcount,
                                            const float* mean2d, const float* conic, const float* lnv, int32_t tiles_x,
                                            int32_t tiles_y, int32_t ts, int64_t capacity, uint64_t* keys_sorted,
                                            uint32_t* vals_sorted, uint32_t* ranges) {
    const int64_t I = xpr_oracle_emit_cull(N, depth, rect, tcount, mean2d, conic, lnv, tiles_x, ts, 0, nullptr, nullptr);
    if (capacity < I) return I;
    std::vector<uint64_t> keys((size_t)I);
    std::vector<uint32_t> vals((size_t)I);
    xpr_oracle_emit_cull(N, depth, rect, tcount, mean2d, conic, lnv, tiles_x, ts, I, keys.data(), vals.data());
    sort_and_bounds(I, keys, vals, tiles_x, tiles_y, keys_sorted, vals_sorted, ranges);
    return I;
}

extern "C" int32_t xpr_oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// XPR-3DGUT ray evaluation
#include "xpr_oracle_ray.inc"

// rendered depth and accumulated opacity
#include "xpr_oracle_feat.inc"

// XPR-LinPrim
#include "xpr_oracle_lin.inc"
