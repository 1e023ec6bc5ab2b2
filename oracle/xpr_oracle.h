/*
 * xpr_oracle.h -- C interface of the CPU ORACLE for the tile-based splatting hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call anything under oracle/.
 * It shares no code with the CUDA path (paper_2606_11529_b200/csrc, include/xpr.h): the structs
 * below are the oracle's own, every field a double, and all pointers are HOST pointers.
 *
 * What it computes: the plain definition of tile-based 3DGS rendering and its exact reverse-mode
 * derivative, written from /root/reference/PAPER.md (XPR, arxiv 2606.11529) and the readings
 * C1..C31 / rules R1..R3 in DESIGN.md.  Each function cites the passage it follows
 * ("PAPER L<line>").  Scalar type: *_f32 = parity mode (every operation individually rounded in
 * fp32, in the order DESIGN.md section 3 fixes; compiled with -ffp-contract=off), *_f64 =
 * self-check mode (closed forms, finite differences).  Gradients are accumulated and returned
 * in fp64 in both modes.
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"): P1 closed form single Gaussian, P2
 * transmittance/opacity invariants, P3 brute-force binning, P4 tiling invariance, P5 sort
 * invariants, P6 central finite differences (fp64), P7 UT exact for affine maps, P8 UT~EWA limit,
 * P9 fisheye special cases, P10 SH orthonormality/degree-0, P11 linearity, P12 fp32-vs-fp64,
 * P13 tile_cull (dense-sampling maximum, no passing pixel in a dropped pair, image unchanged),
 * P14 3DGUT ray evaluation (brute-force maximum along the ray in the world frame, isotropic closed form,
 * pixel_info as the inverse of the camera model, finite differences),
 * P15 rendered depth / accumulated opacity (equal to the pinned colour pass with rgb := (z, 1, .) and bg = 0,
 * A = 1 - T_final, finite differences).
 * No function here is "parity unpinned".
 */
#ifndef XPR_ORACLE_H
#define XPR_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    int32_t model;              /* 0 pinhole, 1 fisheye-equidistant, 2 affine/orthographic (pin P7 only) */
    int32_t width, height;
    double fx, fy, cx, cy;
    double k[4];
    double w2c[12];             /* row-major [W|t] */
} xo_camera;

typedef struct {
    int32_t projection;         /* 0 EWA, 1 UT */
    int32_t sh_degree;          /* 0..3 */
    int32_t tile;               /* tile edge in pixels (16; 8 allowed for pin P4) */
    int32_t antialias;          /* Mip-Splatting opacity factor */
    double alpha_thresh, alpha_max, t_min, z_near, lowpass;
    double ut_alpha, ut_beta, ut_kappa;
    double bg[3];
    double fragile_rel;         /* relative margin of the fragile-pixel protocol */
    int32_t tile_cull;          /* 1: drop (primitive, tile) pairs that fail tile_cull */
} xo_config;

/* flags byte written by project */
enum { XO_VISIBLE = 1, XO_CLAMP_U = 2, XO_CLAMP_V = 4, XO_RGB_POS_R = 8, XO_RGB_POS_G = 16, XO_RGB_POS_B = 32 };
/* fragile bits written by rasterize_fwd */
enum { XO_FRAG_EXIT = 1, XO_FRAG_CLAMP = 2, XO_FRAG_GATE = 4 };

#define XO_DECL(S, T)                                                                                   \
    /* Preprocess (Listing 1; UT: L437, Listing 3). */         \
    void xpr_oracle_project_##S(int64_t N, const T* means, const T* scales, const T* quats,             \
                                const T* opacities, const T* sh, const xo_camera* cam,                  \
                                const xo_config* cfg, T* mean2d, T* conic, T* opac_eff, T* rgb,         \
                                T* depth, T* lnv, int32_t* tile_rect, uint32_t* tile_count,             \
                                uint8_t* flags);                                                        \
    /* Shader, Algorithm 1 (Listing 1), tile lists from bin_sort. */      \
    void xpr_oracle_rasterize_fwd_##S(const xo_camera* cam, const xo_config* cfg, int64_t N,            \
                                      const T* mean2d, const T* conic, const T* opac_eff, const T* rgb, \
                                      const T* lnv, const uint32_t* vals_sorted,                        \
                                      const uint32_t* tile_ranges, T* image, T* final_T,                \
                                      uint32_t* n_contrib, uint8_t* fragile, int64_t* counters);        \
    /* Strict per-pixel mode: each pixel's own list sorted by (depth, index); no binning used. */       \
    void xpr_oracle_rasterize_fwd_strict_##S(const xo_camera* cam, const xo_config* cfg, int64_t N,     \
                                             const T* mean2d, const T* conic, const T* opac_eff,        \
                                             const T* rgb, const T* lnv, const T* depth,                \
                                             const int32_t* tile_rect, const uint32_t* tile_count,      \
                                             T* image, T* final_T, uint32_t* n_contrib);                \
    /* Reverse mode through compositing (hand-derived; the paper relies on AD, L106). */                \
    void xpr_oracle_rasterize_bwd_##S(const xo_camera* cam, const xo_config* cfg, int64_t N,            \
                                      const T* mean2d, const T* conic, const T* opac_eff, const T* rgb, \
                                      const T* lnv, const uint32_t* vals_sorted,                        \
                                      const uint32_t* tile_ranges, const uint32_t* n_contrib,           \
                                      const T* dL_dimage, double* g_mean2d, double* g_conic,            \
                                      double* g_opac_eff, double* g_rgb);                               \
    /* Same loop with every sum kept in fp32 (a CPU fp32 implementation; reported beside the GPU) */ \
    void xpr_oracle_rasterize_bwd_acc32_##S(const xo_camera* cam, const xo_config* cfg, int64_t N,      \
                                      const T* mean2d, const T* conic, const T* opac_eff, const T* rgb, \
                                      const T* lnv, const uint32_t* vals_sorted,                        \
                                      const uint32_t* tile_ranges, const uint32_t* n_contrib,           \
                                      const T* dL_dimage, double* g_mean2d, double* g_conic,            \
                                      double* g_opac_eff, double* g_rgb);                               \
    /* Same loop with |addend| accumulated: per-element mass sum_pixels |term| (tolerance scale only). */ \
    void xpr_oracle_rasterize_bwd_mass_##S(const xo_camera* cam, const xo_config* cfg, int64_t N,       \
                                      const T* mean2d, const T* conic, const T* opac_eff, const T* rgb, \
                                      const T* lnv, const uint32_t* vals_sorted,                        \
                                      const uint32_t* tile_ranges, const uint32_t* n_contrib,           \
                                      const T* dL_dimage, double* g_mean2d, double* g_conic,            \
                                      double* g_opac_eff, double* g_rgb);                               \
    /* Reverse mode through projection + SH (hand-derived). */                                          \
    void xpr_oracle_project_bwd_##S(int64_t N, const T* means, const T* scales, const T* quats,         \
                                    const T* opacities, const T* sh, const xo_camera* cam,              \
                                    const xo_config* cfg, const double* g_mean2d, const double* g_conic,\
                                    const double* g_opac_eff, const double* g_rgb, double* g_means,     \
                                    double* g_scales, double* g_quats, double* g_opacities,             \
                                    double* g_sh);                                                      \
    /* Real SH basis, degree <= 3 (reading C5); out[16]. */                                             \
    void xpr_oracle_sh_basis_##S(const T* dir, T* out16);                                               \
    /* Camera model pi: camera-space point -> pixel (readings C1, C2, C18). */                          \
    void xpr_oracle_camera_project_##S(const xo_camera* cam, const T* p_cam, T* pix2);

XO_DECL(f32, float)
XO_DECL(f64, double)

/* Rasterizer: replicate, assign tile id, stable sort by (tile, depth), bounds.
 * depth is fp32 (its bit pattern is the low key word, BASELINE.json:north_star).  Returns the
 * number of pairs I; writes at most `capacity` entries (pass capacity=0 to count only). */
int64_t xpr_oracle_bin_sort(int64_t N, const float* depth, const int32_t* tile_rect,
                            const uint32_t* tile_count, int32_t tiles_x, int32_t tiles_y,
                            int64_t capacity, uint64_t* keys_sorted, uint32_t* vals_sorted,
                            uint32_t* tile_ranges);

/* Unsorted emission only (pin P3 / parity of the emit step). */
int64_t xpr_oracle_emit(int64_t N, const float* depth, const int32_t* tile_rect,
                        const uint32_t* tile_count, int32_t tiles_x, int64_t capacity,
                        uint64_t* keys, uint32_t* vals);

/* tile_cull of XPR-3DGS ("Cull", L268-281, L435): keep[i] = 1 iff the maximum of alpha over the
 * hull of the pixel centres of tile tile_xy[i] reaches alpha_thresh (conservative margin: DESIGN.md C8). */
void xpr_oracle_tile_keep_f32(int64_t n, const float* mean2d, const float* conic, const float* lnv,
                              const int32_t* tile_xy, int32_t ts, uint8_t* keep);
void xpr_oracle_tile_keep_f64(int64_t n, const double* mean2d, const double* conic, const double* lnv,
                              const int32_t* tile_xy, int32_t ts, uint8_t* keep);
/* Emission and binning with tile_cull: pairs that fail it are not emitted.  Return the surviving count. */
int64_t xpr_oracle_emit_cull(int64_t N, const float* depth, const int32_t* tile_rect, const uint32_t* tile_count,
                             const float* mean2d, const float* conic, const float* lnv, int32_t tiles_x,
                             int32_t ts, int64_t capacity, uint64_t* keys, uint32_t* vals);
int64_t xpr_oracle_bin_sort_cull(int64_t N, const float* depth, const int32_t* tile_rect,
                                 const uint32_t* tile_count, const float* mean2d, const float* conic,
                                 const float* lnv, int32_t tiles_x, int32_t tiles_y, int32_t ts, int64_t capacity,
                                 uint64_t* keys_sorted, uint32_t* vals_sorted, uint32_t* tile_ranges);

/* ---- XPR-3DGUT evaluation, SURVEY 8(f) f2 (xpr_oracle_ray.inc; PAPER A.1.2 L437-444 Eq. 1, Listing 3).
 * Reading C27: ray and Gaussian live in the camera frame.  pixel_rays [H*W*3]: unit ray directions (camera frame)
 * through the pixel centres; ray_rec [N*12]: M_c = S^-1 (W R)^T row-major (9), o_c = -M_c p (3).  Pin P14. */
#define XO_RAY_DECL(S, T)                                                                                \
    void xpr_oracle_pixel_info_##S(const xo_camera* cam, T* pixel_rays);                                 \
    void xpr_oracle_pixel_ray_##S(const xo_camera* cam, double u, double v, T* d3);                      \
    void xpr_oracle_project_ray_##S(int64_t N, const T* means, const T* scales, const T* quats,          \
                                    const xo_camera* cam, const uint32_t* tile_count, T* ray_rec);       \
    /* out3 = {power = nhq/dd, nhq = -1/2 |o_c x d_c|^2, dd = |d_c|^2} for one record and one ray */     \
    void xpr_oracle_ray_power_##S(const T* rec12, const T* d3, T* out3);                                 \
    void xpr_oracle_rasterize_ray_fwd_##S(const xo_camera* cam, const xo_config* cfg, int64_t N,         \
                                          const T* ray_rec, const T* opac_eff, const T* rgb,             \
                                          const T* lnv, const T* pixel_rays, const uint32_t* vals_sorted,\
                                          const uint32_t* tile_ranges, T* image, T* final_T,             \
                                          uint32_t* n_contrib, uint8_t* fragile, int64_t* counters);     \
    /* g_ray_rec [N*12] = dL/dM_c (9), dL/do_c (3) */                                                    \
    void xpr_oracle_rasterize_ray_bwd_##S(const xo_camera* cam, const xo_config* cfg, int64_t N,         \
                                          const T* ray_rec, const T* opac_eff, const T* rgb,             \
                                          const T* lnv, const T* pixel_rays, const uint32_t* vals_sorted,\
                                          const uint32_t* tile_ranges, const uint32_t* n_contrib,        \
                                          const T* dL_dimage, double* g_ray_rec, double* g_opac_eff,     \
                                          double* g_rgb);                                                \
    void xpr_oracle_rasterize_ray_bwd_mass_##S(const xo_camera* cam, const xo_config* cfg, int64_t N,    \
                                          const T* ray_rec, const T* opac_eff, const T* rgb,             \
                                          const T* lnv, const T* pixel_rays, const uint32_t* vals_sorted,\
                                          const uint32_t* tile_ranges, const uint32_t* n_contrib,        \
                                          const T* dL_dimage, double* g_ray_rec, double* g_opac_eff,     \
                                          double* g_rgb);                                                \
    /* chain rule record -> (mu, s, q); WRITES its outputs (the caller adds them to project_bwd's) */    \
    /* the same sums in the form the GPU accumulates: g_ray_acc [N*16] = S_c = sum k c c^T (6), D = sum 2 dL/ddd  \
       d d^T (6), sum dL/do_c (3), unused (1); mass != 0: sums of |addend|.  xpr_oracle_ray_bwd_acc applies the     \
       chain rule to them; the two routes are equal (pin P14f) */                                                   \
    void xpr_oracle_rasterize_ray_bwd_acc_##S(const xo_camera* cam, const xo_config* cfg, int64_t N,     \
                                          const T* ray_rec, const T* opac_eff, const T* rgb,             \
                                          const T* lnv, const T* pixel_rays, const uint32_t* vals_sorted,\
                                          const uint32_t* tile_ranges, const uint32_t* n_contrib,        \
                                          const T* dL_dimage, int32_t mass, double* g_ray_acc,           \
                                          double* g_opac_eff, double* g_rgb);                            \
    void xpr_oracle_ray_bwd_acc_##S(int64_t N, const T* means, const T* scales, const T* quats,          \
                                const xo_camera* cam, const uint32_t* tile_count,                        \
                                const double* g_ray_acc, double* g_means, double* g_scales,              \
                                double* g_quats);                                                        \
    void xpr_oracle_ray_bwd_##S(int64_t N, const T* means, const T* scales, const T* quats,              \
                                const xo_camera* cam, const uint32_t* tile_count,                        \
                                const double* g_ray_rec, double* g_means, double* g_scales,              \
                                double* g_quats);

XO_RAY_DECL(f32, float)
XO_RAY_DECL(f64, double)

/* ---- Rendered features beyond colour, SURVEY 8(f) f3 (xpr_oracle_feat.inc; Table 2; reading C31):
 * depth image D = sum_k z_k alpha_k T_k and accumulated opacity A = sum_k alpha_k T_k over the colour pass's own
 * contributing sequence, no background; depth [N] = camera-space z of the centres (project's output).  The
 * backward takes dL/dimage, dL/dD, dL/dA and returns rasterize_bwd's outputs plus g_depth [N].  Pin P15. */
#define XO_FEAT_DECL(S, T)                                                                               \
    void xpr_oracle_rasterize_fwd_da_##S(const xo_camera* cam, const xo_config* cfg, int64_t N,          \
                                         const T* mean2d, const T* conic, const T* opac_eff,             \
                                         const T* rgb, const T* lnv, const T* depth,                     \
                                         const uint32_t* vals_sorted, const uint32_t* tile_ranges,       \
                                         T* depth_img, T* alpha_img);                                    \
    void xpr_oracle_rasterize_bwd_da_##S(const xo_camera* cam, const xo_config* cfg, int64_t N,          \
                                         const T* mean2d, const T* conic, const T* opac_eff,             \
                                         const T* rgb, const T* lnv, const T* depth,                     \
                                         const uint32_t* vals_sorted, const uint32_t* tile_ranges,       \
                                         const uint32_t* n_contrib, const T* dL_dimage,                  \
                                         const T* dL_ddepth, const T* dL_dalpha, double* g_mean2d,       \
                                         double* g_conic, double* g_opac_eff, double* g_rgb,             \
                                         double* g_depth);                                               \
    /* sum of |addend| per element (tolerance aid, like xpr_oracle_rasterize_bwd_mass_*) */             \
    void xpr_oracle_rasterize_bwd_da_mass_##S(const xo_camera* cam, const xo_config* cfg, int64_t N,     \
                                         const T* mean2d, const T* conic, const T* opac_eff,             \
                                         const T* rgb, const T* lnv, const T* depth,                     \
                                         const uint32_t* vals_sorted, const uint32_t* tile_ranges,       \
                                         const uint32_t* n_contrib, const T* dL_dimage,                  \
                                         const T* dL_ddepth, const T* dL_dalpha, double* g_mean2d,       \
                                         double* g_conic, double* g_opac_eff, double* g_rgb,             \
                                         double* g_depth);

XO_FEAT_DECL(f32, float)
XO_FEAT_DECL(f64, double)

/* N-channel features (same section; pin P16): feat [N*C], feat_img [H*W*C] = sum_k feat[g_k,:] alpha_k T_k over the
 * colour pass's contributing sequence, no background (rgb is only an argument of the shared walk and does not
 * influence the result).  The backward takes dL/dfeat_img ALONE and returns that part of g_mean2d, g_conic, g_opac_eff
 * plus g_feat [N*C]; colour / D / A parts of a loss add (every step is linear in the incoming gradient). */
#define XO_FEATN_DECL(S, T)                                                                              \
    void xpr_oracle_rasterize_fwd_featn_##S(const xo_camera* cam, const xo_config* cfg, int64_t N,       \
                                            const T* mean2d, const T* conic, const T* opac_eff,          \
                                            const T* rgb, const T* lnv, const T* feat, int32_t C,        \
                                            const uint32_t* vals_sorted, const uint32_t* tile_ranges,    \
                                            T* feat_img);                                                \
    void xpr_oracle_rasterize_bwd_featn_##S(const xo_camera* cam, const xo_config* cfg, int64_t N,       \
                                            const T* mean2d, const T* conic, const T* opac_eff,          \
                                            const T* rgb, const T* lnv, const T* feat, int32_t C,        \
                                            const uint32_t* vals_sorted, const uint32_t* tile_ranges,    \
                                            const uint32_t* n_contrib, const T* dL_dfeat,                \
                                            double* g_mean2d, double* g_conic, double* g_opac_eff,       \
                                            double* g_feat);

XO_FEATN_DECL(f32, float)
XO_FEATN_DECL(f64, double)

/* z = (W mu + t)_z: WRITES g_means [N*3] = W[2,:] g_depth (zeros where tile_count == 0); the caller adds it to
 * project_bwd's g_means. */
void xpr_oracle_depth_bwd(int64_t N, const xo_camera* cam, const uint32_t* tile_count, const double* g_depth,
                          double* g_means);

int32_t xpr_oracle_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
