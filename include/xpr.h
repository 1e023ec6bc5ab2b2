/*
 * xpr.h -- C-ABI boundary of libxpr.so: the tile-based splatting forward + backward hot path of
 * "XPR: An Extensible Cross-Platform Point-Based Differentiable Renderer" (arxiv 2606.11529),
 * hand-written CUDA for NVIDIA B200 (sm_100a).  Citations are PAPER.md line numbers ("PAPER L..")
 * plus the readings C1..C32, L1..L6 and arithmetic rules R1..R3 listed in DESIGN.md section 3.
 *
 * Conventions
 *  - Every function returns an int32_t status (XPR_OK == 0).  No exceptions, no global state other
 *    than the last CUDA error code (thread-local), re-entrant.
 *  - Unless a parameter says HOST, every array pointer is a DEVICE pointer owned by the caller
 *    (e.g. a PyTorch allocation), contiguous, row-major, 16-byte aligned.  The library allocates
 *    no persistent device memory; scratch comes from the caller-provided workspace.
 *  - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  All work is
 *    enqueued on it.  The only call that synchronises the stream is xpr_bin_sort, at its end (8-byte
 *    read-back of the pair count I), and only when num_pairs_host != NULL.
 *  - xpr_camera / xpr_config are HOST structs, read during the call.
 *  - Arguments are validated before any launch: NULL or misaligned pointer, negative size, bad
 *    enum -> XPR_ERR_INVALID_ARG; tile != 16, sh_degree > 3 -> XPR_ERR_UNSUPPORTED; a CUDA runtime
 *    failure -> XPR_ERR_CUDA (code via xpr_last_cuda_error()).
 *  - `scales`, `opacities`, `quats` are ACTIVATED values (positive scales, opacity in (0,1), unit
 *    quaternion (w,x,y,z), not renormalised inside) exactly as the paper's PrimitiveParams
 *    (PAPER L425-431).  Activations and the loss live outside the library.
 *  - Pixel (i,j) is sampled at (i+0.5, j+0.5); mean2d is in continuous pixel coordinates (C1).
 *    Tile t = ty*tiles_x + tx covers pixels [16 tx, 16 tx+16) x [16 ty, 16 ty+16).
 */
#ifndef XPR_H
#define XPR_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum { XPR_OK = 0, XPR_ERR_INVALID_ARG = 1, XPR_ERR_CAPACITY = 2, XPR_ERR_CUDA = 3, XPR_ERR_UNSUPPORTED = 4,
       XPR_ERR_SCRATCH_LIMIT = 5 /* xpr_bin_sort_static: the sizes need more than XPR_STATIC_SCRATCH_BYTES of workspace */ };

/* flags byte written per Gaussian by xpr_project */
enum { XPR_FLAG_VISIBLE = 1, XPR_FLAG_CLAMP_U = 2, XPR_FLAG_CLAMP_V = 4,
       XPR_FLAG_RGB_POS_R = 8, XPR_FLAG_RGB_POS_G = 16, XPR_FLAG_RGB_POS_B = 32 };

typedef struct {
    int32_t model;          /* 0 pinhole, 1 fisheye-equidistant (C18) */
    int32_t width, height;  /* pixels */
    float fx, fy, cx, cy;   /* intrinsics (C2) */
    float k[4];             /* fisheye radial distortion k1..k4 */
    float w2c[12];          /* row-major 3x4 [W|t]: x_cam = W x_world + t, +z forward, x right, y down */
} xpr_camera;

typedef struct {
    int32_t projection;     /* 0 EWA (PAPER Listing 1), 1 UT with 7 sigma points */
    int32_t sh_degree;      /* 0..3, K = (sh_degree+1)^2 coefficients per channel */
    int32_t tile;           /* tile edge in pixels; must be 16 */
    int32_t antialias;      /* Mip-Splatting opacity factor (C19) */
    float alpha_thresh;     /* 1/255 */
    float alpha_max;        /* 0.99 (C11) */
    float t_min;            /* 1e-4 transmittance exit (C12) */
    float z_near;           /* 0.2 (C9) */
    float lowpass;          /* 0.3 added to the 2D covariance diagonal (C4) */
    float ut_alpha, ut_beta, ut_kappa;  /* unscented-transform weights: 1, 2, 0 */
    float bg[3];            /* background colour (C13) */
    int32_t tile_cull;      /* 1: xpr_bin_sort_cull drops (Gaussian, tile) pairs that fail tile_cull */
    uint32_t* tile_order;   /* DEVICE uint32[T] or NULL.  Scheduling only, no effect on any result: when set,
                               xpr_bin_sort[_cull] also writes the tile indices by decreasing list length (1024
                               length classes) and the four rasterize calls walk the tiles in that order, so that
                               the tail of a launch consists of short tiles */
    int32_t views;          /* 0 or 1: one view.  V in 2..8: ONE call renders a batch of V views of the same Gaussians (PAPER
                               L19, Table 2 "batched views"; BASELINE.json configs[4]): `cam` then points to V cameras of
                               equal model, width and height; per-Gaussian outputs of xpr_project (and the inputs of the later
                               calls) are [V*N, ...] view-major, index v*N + i; tile_rect rows are offset by v*tiles_y, so that
                               the tile id of a pair is v*T + t and one xpr_bin_sort[_cull] call (its N = V*N) sorts all views
                               (keys = (v*T + t) << 32 | depth bits; tile_ranges [V*T, 2]); images are [V, H, W, .], the
                               compositing calls launch V*T tiles; xpr_project_bwd SUMS the parameter gradients over the views.
                               xpr_rasterize_feat_fwd / _bwd take the batch too (depth_img, alpha_img, dL_ddepth, dL_dalpha are
                               [V, H, W]; g_depth [V*N]).  xpr_pixel_info, xpr_project_ray, xpr_ray_bwd, the featn calls and
                               xpr_depth_bwd take one view (call xpr_depth_bwd once per view on that view's slices: it adds) */
} xpr_config;
enum { XPR_MAX_VIEWS = 8 };

const char* xpr_status_string(int32_t status);
int32_t xpr_last_cuda_error(void);   /* cudaError_t of the last XPR_ERR_CUDA on this thread */
int32_t xpr_version(void);           /* 10000*major + 100*minor + patch */

/*
 * xpr_project -- Preprocess stage (Listing 1; A.1.1 L435; UT: L437,
 * Listing 3) fused with SH -> RGB (C5).  One thread per Gaussian.
 *   in : means[N,3] scales[N,3] quats[N,4] opacities[N] sh[N,K,3]  (fp32)
 *   out: mean2d[N,2], conic_opac[N,4] = (A,B,C,o_eff) with (A,B,C) the inverse of the low-passed
 *        2D covariance, rgb[N,3], depth[N] (camera z of the mean), lnv[N] = ln(o_eff/alpha_thresh),
 *        tile_rect[N,4] = (x_min,y_min,x_max,y_max) half-open in tile units,
 *        tile_count[N] = rectangle area if visible else 0, flags[N];
 *        shade_rec[N,12] (may be NULL) = the shader data p_sd of the primitive packed as the
 *        compositing calls read it, 3 x float4, 16-byte aligned:
 *          (mx, my, -A/2, -B | -C/2, lnv, log2 o_eff, depth | r, g, b, o_eff)
 *        -- the pre-scaled conic of reading C25 (exact in fp32); log2 by lg2.approx (it only feeds exp()).  lnv > 0 in
 *        every record xpr_project writes (a Gaussian with lnv <= 0 has an empty extent and is culled); the compositing
 *        kernels rely on it: they test both gates of a list entry (power <= 0, power >= -lnv) as ONE unsigned compare
 *        bits(-power) <= bits(lnv), so a record built by the caller (xpr_shade_record) must come from such a Gaussian.
 *   For a culled Gaussian only tile_count (=0) and flags (=0) are written; its other outputs are
 *   left untouched (they are never read downstream).
 *   Arithmetic follows rule R1: fp32, every operation individually rounded, no FMA contraction,
 *   so that depth bits, rectangles and tile counts are bit-reproducible.
 *   Two readings the paper does not fix and nothing can pin: the EWA Jacobian is evaluated at
 *   x/z clamped to [-(cx + 0.15 W)/fx, ((W - cx) + 0.15 W)/fx] (likewise y; C6), and with the UT a Gaussian is culled
 *   when any of its 7 sigma points has z <= 0 (C18).
 */
int32_t xpr_project(int64_t N, const float* means, const float* scales, const float* quats,
                    const float* opacities, const float* sh, const xpr_camera* cam, const xpr_config* cfg,
                    float* mean2d, float* conic_opac, float* rgb, float* depth, float* lnv,
                    int32_t* tile_rect, uint32_t* tile_count, uint8_t* flags, float* shade_rec, void* stream);

/*
 * xpr_shade_record -- builds shade_rec[N,12] (layout above) from the separate projection outputs, for a caller
 * whose projection did not come from xpr_project; depth may be NULL (slot 7 is then 0; it is only read by the
 * rendered-depth feature).  Records of culled Gaussians (tile_count == 0) are not written.
 */
int32_t xpr_shade_record(int64_t N, const float* mean2d, const float* conic_opac, const float* rgb, const float* lnv,
                         const float* depth, const uint32_t* tile_count, float* shade_rec, void* stream);

/*
 * xpr_bin_sort -- Rasterizer stage: prefix-sum of tile counts, replication,
 * tile-id assignment  x = x_min + (r mod w), y = y_min + floor(r / w), t = y*tiles_x + x,
 * key = (uint64)t << 32 | float_bits(depth) (BASELINE.json:north_star, C10), value = Gaussian
 * index; the result of the stable LSD radix sort by key, produced by hand-written kernels (onesweep passes on the
 * depth bits of the Gaussians and on the supertile ids, then one pass that writes every pair at its final position,
 * DESIGN.md 6.2); per-tile bounds.
 *   in : depth[N], tile_rect[N,4], tile_count[N] from xpr_project; pair_capacity = length of the
 *        output arrays (must be < 2^30; 0 is allowed and makes the call a size probe: with any visible
 *        Gaussian it reports XPR_ERR_CAPACITY and the capacity that suffices, in both modes below).
 *        N must be < 2^30 (XPR_ERR_UNSUPPORTED otherwise: the sort's look-back words carry 30-bit counts).
 *   out: keys_sorted[I] u64, vals_sorted[I] u32, tile_ranges[T,2] = (start,end) per tile, (0,0)
 *        for an empty tile; *num_pairs_host (HOST int64) = I.
 *   Capacity: besides the I output pairs, the output arrays serve as scratch for the (Gaussian, tile row) rows
 *   (4 bytes each) and for the (Gaussian, 8 x 8-tile supertile) words the call sorts first (8 bytes each, two
 *   buffers): pair_capacity >= max(I, rows + 1, 2 x words).  rows and words are at most sum of tile_count; for
 *   Gaussians that cover a few tiles each 2 x words can exceed I.
 *   Nothing inside the call waits for the host: every count stays on the device and every kernel
 *   reads it there.  With num_pairs_host != NULL the call ends with a 16-byte read-back of the counts
 *   and a stream synchronisation; if the capacity does not suffice -> XPR_ERR_CAPACITY with
 *   *num_pairs_host = the capacity that suffices (max(I, rows + 1, 2 x words)).
 *   With num_pairs_host == NULL the call is fully asynchronous (capturable in a CUDA graph): it
 *   returns XPR_OK after enqueueing; once the stream has run, workspace bytes [0,8) hold (uint64) the
 *   number of sorted pairs, or the capacity that suffices when it exceeds pair_capacity -- the caller
 *   must compare it with pair_capacity before trusting the outputs -- and bytes [8,16) the number of
 *   sorted pairs (0 on overflow).
 *   In both modes, when the capacity does not suffice nothing out of bounds is written, tile_ranges
 *   is (0,0) for every tile (a following xpr_rasterize_fwd renders the background) and keys/vals are
 *   unspecified.  keys_sorted and vals_sorted are also used as scratch during the call.
 *   workspace: DEVICE scratch of at least xpr_bin_sort_workspace() bytes, 256-byte aligned.
 *   Equal keys keep emission order = ascending Gaussian index.
 */
int32_t xpr_bin_sort_workspace(int64_t N, int64_t pair_capacity, int32_t num_tiles, size_t* bytes);
int32_t xpr_bin_sort(int64_t N, const float* depth, const int32_t* tile_rect, const uint32_t* tile_count,
                     const xpr_camera* cam, const xpr_config* cfg, int64_t pair_capacity,
                     uint64_t* keys_sorted, uint32_t* vals_sorted, uint32_t* tile_ranges,
                     int64_t* num_pairs_host, void* workspace, size_t workspace_bytes, void* stream);

/*
 * xpr_bin_sort_cull -- xpr_bin_sort with the optional "Cull" step of the paper's rasterizer (
 * tile_cull of XPR-3DGS: Listing 1, A.1.1 L435, after StopThePop).  With cfg->tile_cull != 0 a
 * candidate pair (Gaussian, tile) is kept iff the maximum of alpha = o G_2D(x) over the hull of the
 * tile's pixel centres reaches alpha_thresh, i.e. iff min 1/2 d^T K d <= lnv; the minimiser is the mean
 * if it lies inside, else a point on an edge facing the mean.  The decision is conservative (margin
 * 2^-18 of the magnitude of the terms, reading C8), so every dropped pair has alpha <
 * alpha_thresh at all of its pixels and the image, final_T and the gradients are those of xpr_bin_sort
 * (PAPER L683); n_contrib, which counts list positions, refers to the shorter lists.
 * The paper keeps a rejected pair in its slot with tile id T; here it is not written at all: the
 * survivors are compacted in emission order and only they are sorted.
 *   in : as xpr_bin_sort + the tile-cull data p_tcd of xpr_project: mean2d[N,2], conic_opac[N,4], lnv[N].
 *   out: as xpr_bin_sort; *num_pairs_host = number of SURVIVING pairs (= length of the sorted arrays).
 *   pair_capacity as for xpr_bin_sort, with I the SURVIVING pairs (rejected pairs are never generated, so the
 *   candidate count sum of tile_count need not fit); otherwise XPR_ERR_CAPACITY with *num_pairs_host = the capacity
 *   that suffices.
 *   With cfg->tile_cull == 0 the call is xpr_bin_sort; xpr_bin_sort itself rejects cfg->tile_cull != 0.
 */
int32_t xpr_bin_sort_cull(int64_t N, const float* depth, const int32_t* tile_rect, const uint32_t* tile_count,
                          const float* mean2d, const float* conic_opac, const float* lnv,
                          const xpr_camera* cam, const xpr_config* cfg, int64_t pair_capacity,
                          uint64_t* keys_sorted, uint32_t* vals_sorted, uint32_t* tile_ranges,
                          int64_t* num_pairs_host, void* workspace, size_t workspace_bytes, void* stream);

/*
 * xpr_bin_sort_static -- xpr_bin_sort / xpr_bin_sort_cull WITHOUT a caller workspace and without any allocation, for
 * callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
 * The scratch is a static device array of XPR_STATIC_SCRATCH_BYTES (16 MiB) inside the library: every GPU that loads
 * libxpr.so holds it until the process exits.  The call itself issues no cudaMalloc, cudaFree or allocating library
 * routine; its first call on a device looks the array's address up (cudaGetSymbolAddress, with the current device) --
 * make that first call at set-up, outside any stream capture.
 *   Arguments and results exactly as xpr_bin_sort_cull (mean2d, conic_opac, lnv are read only when cfg->tile_cull != 0
 *   and may be NULL otherwise: the call is then xpr_bin_sort), minus workspace / workspace_bytes.
 *   Limit: the sizes must satisfy xpr_bin_sort_workspace(N, pair_capacity, tiles) <= XPR_STATIC_SCRATCH_BYTES, about
 *   20 N + 9 pair_capacity + 272 tiles bytes -- e.g. N = 200 000 (view x Gaussian entries) with pair_capacity
 *   = 1 048 576, or N = 262 144 with pair_capacity = 786 432, at 1920 x 1080 (8160 tiles); beyond it ->
 *   XPR_ERR_SCRATCH_LIMIT before anything is launched (use xpr_bin_sort with a workspace of your own).
 *   Sharing: all calls on a device use the SAME array, which keeps the previous call's contents.  Every call zero-fills
 *   the part that must start at zero and writes every other part before reading it, so calls in stream order are
 *   independent of each other; calls that OVERLAP on the GPU (two streams with no ordering between them, or this call
 *   in two graphs replayed concurrently) race on the array and give undefined results.  In the asynchronous mode
 *   (num_pairs_host == NULL) the counts xpr_bin_sort leaves in workspace bytes [0,16) stay inside the library: size
 *   pair_capacity from an earlier synchronous call.
 */
enum { XPR_STATIC_SCRATCH_BYTES = 16 * 1024 * 1024 };
int32_t xpr_bin_sort_static(int64_t N, const float* depth, const int32_t* tile_rect, const uint32_t* tile_count,
                            const float* mean2d, const float* conic_opac, const float* lnv,
                            const xpr_camera* cam, const xpr_config* cfg, int64_t pair_capacity,
                            uint64_t* keys_sorted, uint32_t* vals_sorted, uint32_t* tile_ranges,
                            int64_t* num_pairs_host, void* stream);

/*
 * xpr_rasterize_fwd -- Shader stage (Algorithm 1, Listing 1).
 * Per pixel, front to back over its tile's list:
 *   power = -1/2 (A dx^2 + C dy^2) - B dx dy   (order fixed by R3);
 *   skip if power > 0 (L289) or power < -lnv (alpha < alpha_thresh, L679, C12);
 *   alpha = min(alpha_max, o_eff exp(power));  T' = T (1 - alpha);  stop WITHOUT blending if
 *   T' < t_min;  C += rgb alpha T;  T = T'.   Finally C += T bg.
 *   in : shade_rec[N,12] of xpr_project (or xpr_shade_record), the lists of xpr_bin_sort[_cull].
 *   out: image[H,W,3], final_T[H,W], n_contrib[H,W] = 1 + list position of the last blended entry.
 *   The records of a tile's list are gathered into shared memory by cp.async (three-stage ring).
 */
int32_t xpr_rasterize_fwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* shade_rec,
                          const uint32_t* vals_sorted, const uint32_t* tile_ranges,
                          float* image, float* final_T, uint32_t* n_contrib, void* stream);

/*
 * xpr_rasterize_stats -- measurement aid (SURVEY.md 8(d) roofline accounting): the same walk as
 * xpr_rasterize_fwd without writing an image; stats[0..3] (DEVICE uint64[4], overwritten) =
 * {pixel-pairs visited, pixel-pairs passing both gates, pixel-pairs blended, sum of n_contrib}.
 */
int32_t xpr_rasterize_stats(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* shade_rec,
                            const uint32_t* vals_sorted, const uint32_t* tile_ranges, uint64_t* stats,
                            void* stream);

/*
 * xpr_rasterize_bwd -- reverse mode through compositing (the paper relies on AD, L106; formulas
 * in DESIGN.md section 3, readings C14-C15).  Replays each tile back to front from n_contrib.
 *   in : forward inputs + final_T, n_contrib, dL_dimage[H,W,3].
 *   out: g_mean2d[N,2], g_conic[N,3] (w.r.t. A,B,C), g_opac[N] (w.r.t. o_eff), g_rgb[N,3];
 *        ACCUMULATED with fp32 atomics; zero-filled first by this call when zero_init != 0.
 *        (with one fill instead of four when the four arrays are adjacent slices of one allocation, in this order).
 */
int32_t xpr_rasterize_bwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* shade_rec,
                          const uint32_t* vals_sorted, const uint32_t* tile_ranges,
                          const float* final_T, const uint32_t* n_contrib, const float* dL_dimage,
                          float* g_mean2d, float* g_conic, float* g_opac, float* g_rgb,
                          int32_t zero_init, void* stream);
/*
 * xpr_rasterize_bwd_loss -- xpr_rasterize_bwd for the two losses BASELINE.json's configs name, with the loss gradient
 * formed inside the kernel: dL/dimage = sign(I - target) (loss_kind 0, L = sum |I - target|) or 2 (I - target)
 * (loss_kind 1, L = sum (I - target)^2) from `image` (the output of xpr_rasterize_fwd) and `target`, both [H,W,3]
 * ([V,H,W,3] for a batch of views) -- the values xpr_loss_grad would write, so every result is that of xpr_loss_grad
 * followed by xpr_rasterize_bwd, one pass over the image and one launch less.  Other arguments and errors as
 * xpr_rasterize_bwd; loss_kind outside {0, 1} -> XPR_ERR_INVALID_ARG.
 */
int32_t xpr_rasterize_bwd_loss(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* shade_rec,
                               const uint32_t* vals_sorted, const uint32_t* tile_ranges, const float* image,
                               const float* final_T, const uint32_t* n_contrib, int32_t loss_kind, const float* target,
                               float* g_mean2d, float* g_conic, float* g_opac, float* g_rgb, int32_t zero_init,
                               void* stream);

/*
 * xpr_project_bwd -- reverse mode through projection (EWA or UT) and SH (DESIGN.md section 3,
 * readings C16-C19).  One thread per Gaussian; a culled Gaussian (tile_count == 0) gets zeros.
 *   out (fully overwritten): g_means[N,3] g_scales[N,3] g_quats[N,4] g_opacities[N] g_sh[N,K,3].
 *   The call is a zero-fill of the five outputs (one cudaMemsetAsync when they are adjacent slices of one allocation,
 *   in this order) followed by a kernel over the visible Gaussians only.  The fill (59 floats per Gaussian at degree 3)
 *   is pure HBM traffic with no input: xpr_project_bwd_fill issues it alone -- e.g. on a second stream, under the
 *   ALU-bound xpr_rasterize_bwd -- and xpr_project_bwd_filled is xpr_project_bwd without it (the caller orders the two:
 *   the fill must have completed, and nothing may have written the arrays since).
 */
int32_t xpr_project_bwd(int64_t N, const float* means, const float* scales, const float* quats,
                        const float* opacities, const float* sh, const xpr_camera* cam, const xpr_config* cfg,
                        const uint32_t* tile_count, const uint8_t* flags,
                        const float* g_mean2d, const float* g_conic, const float* g_opac, const float* g_rgb,
                        float* g_means, float* g_scales, float* g_quats, float* g_opacities, float* g_sh,
                        void* stream);
int32_t xpr_project_bwd_fill(int64_t N, const xpr_config* cfg, float* g_means, float* g_scales, float* g_quats,
                             float* g_opacities, float* g_sh, void* stream);
int32_t xpr_project_bwd_filled(int64_t N, const float* means, const float* scales, const float* quats,
                               const float* opacities, const float* sh, const xpr_camera* cam, const xpr_config* cfg,
                               const uint32_t* tile_count, const uint8_t* flags,
                               const float* g_mean2d, const float* g_conic, const float* g_opac, const float* g_rgb,
                               float* g_means, float* g_scales, float* g_quats, float* g_opacities, float* g_sh,
                               void* stream);

/*
 * ---- XPR-3DGUT evaluation (PAPER A.1.2 L437-444 Eq. 1, Listing 3) -----------------
 * The 2D footprint of xpr_project (UT or EWA) only tiles and culls; a pixel evaluates the 3D Gaussian at the
 * point of maximum response along its camera ray.  Reading C27: ray and Gaussian are expressed in the camera
 * frame (ray origin 0, p = W mu + t):  M_c = S^-1 (W R)^T,  o_c = -M_c p,  d_c = M_c d,
 *   response = exp(-1/2 |o_c x d_c|^2 / |d_c|^2),  alpha = min(alpha_max, o_eff response),
 *   valid = response > 0.0113 (L500) and alpha >= alpha_thresh, both decided on products (rule R3):
 *   nhq = -1/2 |o_c x d_c|^2, dd = |d_c|^2:  nhq > ln(0.0113) dd  and  nhq >= -lnv dd.
 *
 * xpr_pixel_info -- pixel_info of Listing 3: pixel_rays[H,W,3] = unit direction (camera frame) of the ray through
 *   the pixel centre (i+0.5, j+0.5), the inverse of the camera model (fisheye: at most 12 Newton steps on the
 *   radial polynomial); fp64 inside, rounded to fp32 last (rule R2).  Depends on the intrinsics only.
 * xpr_project_ray -- shader record p_sd: ray_rec[N,12] = M_c row-major (9), o_c (3); zeros for a culled Gaussian
 *   (tile_count == 0) and for a record that is not finite (C30).  fp32, rule R1.
 * xpr_rasterize_ray_fwd / _bwd -- xpr_rasterize_fwd / _bwd with this evaluation; opacity o_eff is read from
 *   conic_opac[.,3].  bwd ACCUMULATES g_ray_acc[N,16] (16-byte aligned), g_opac[N], g_rgb[N,3]; g_ray_acc holds the
 *   record gradient as sums that do not cancel in fp32: with k = -dL/dpower / |d_c|^2, c = o_c x d_c per pixel,
 *   S_c = sum k c c^T (xx xy xz yy yz zz), D = sum 2 dL/d|d_c|^2 d d^T (same order), sum dL/do_c (3), one unused
 *   slot; dL/dM_c - dL/do_c p^T = -(S_c - tr(S_c) I) M_c^-T + M_c D exactly
 *   (zero-filled first when zero_init != 0).
 * xpr_ray_bwd -- chain rule from g_ray_acc to (mu, s, q), fp64 inside; ADDS to g_means[N,3], g_scales[N,3],
 *   g_quats[N,4] (call it after xpr_project_bwd, which is given zero g_mean2d / g_conic: the footprint carries
 *   no gradient, the opacity factor and the colour do).
 */
int32_t xpr_pixel_info(const xpr_camera* cam, float* pixel_rays, void* stream);
int32_t xpr_project_ray(int64_t N, const float* means, const float* scales, const float* quats,
                        const xpr_camera* cam, const uint32_t* tile_count, float* ray_rec, void* stream);
int32_t xpr_rasterize_ray_fwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* ray_rec,
                              const float* conic_opac, const float* rgb, const float* lnv, const float* pixel_rays,
                              const uint32_t* vals_sorted, const uint32_t* tile_ranges,
                              float* image, float* final_T, uint32_t* n_contrib, void* stream);
int32_t xpr_rasterize_ray_stats(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* ray_rec,
                                const float* conic_opac, const float* rgb, const float* lnv, const float* pixel_rays,
                                const uint32_t* vals_sorted, const uint32_t* tile_ranges, uint64_t* stats,
                                void* stream);
int32_t xpr_rasterize_ray_bwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* ray_rec,
                              const float* conic_opac, const float* rgb, const float* lnv, const float* pixel_rays,
                              const uint32_t* vals_sorted, const uint32_t* tile_ranges,
                              const float* final_T, const uint32_t* n_contrib, const float* dL_dimage,
                              float* g_ray_acc, float* g_opac, float* g_rgb, int32_t zero_init, void* stream);
int32_t xpr_ray_bwd(int64_t N, const float* means, const float* scales, const float* quats,
                    const xpr_camera* cam, const uint32_t* tile_count, const float* g_ray_acc,
                    float* g_means, float* g_scales, float* g_quats, void* stream);

/*
 * ---- Rendered features beyond colour ("rendered features such as depth", Table 2) ----
 * Reading C31: a rendered feature is blended with the colour's weights over the pixel's contributing
 * sequence, without a background term:
 *   depth image D[H,W] = sum_k z_k alpha_k T_k  (z_k = `depth` of xpr_project, the depth of the sort key, L149),
 *   accumulated opacity A[H,W] = sum_k alpha_k T_k.
 * xpr_rasterize_feat_fwd -- xpr_rasterize_fwd that also writes depth_img and alpha_img in the same walk (image,
 *   final_T, n_contrib as xpr_rasterize_fwd: same gates, clamp and exit).  z_k is slot 7 of shade_rec.
 * xpr_rasterize_feat_bwd -- xpr_rasterize_bwd with the two extra incoming gradients dL_ddepth[H,W], dL_dalpha[H,W]
 *   and the extra output g_depth[N] = dL/dz; ACCUMULATES like xpr_rasterize_bwd, zero-filled first when
 *   zero_init != 0 (one fill when g_mean2d, g_conic, g_opac, g_rgb, g_depth are adjacent slices, in this order).
 * xpr_depth_bwd -- z = (W mu + t)_z: ADDS W[2,:] g_depth[i] to g_means[i,:] for every Gaussian with
 *   tile_count[i] > 0 (call it after xpr_project_bwd, which overwrites g_means).
 * xpr_rasterize_ray_feat_fwd / _bwd -- the same two features with the XPR-3DGUT ray evaluation (f2 x f3): C31 blends a
 *   feature with the weights alpha_k T_k of the colour pass whichever evaluation produced alpha_k (Eq. 1 L439-444 here).
 *   Arguments of xpr_rasterize_ray_fwd / _bwd plus depth[N] (of xpr_project), depth_img / alpha_img, dL_ddepth /
 *   dL_dalpha and g_depth[N]; zero_init: one fill when g_ray_acc, g_opac, g_rgb, g_depth are adjacent slices in this order.
 * Errors as the colour calls: null / misaligned pointer, N < 0 -> XPR_ERR_INVALID_ARG before any launch.
 */
int32_t xpr_rasterize_ray_feat_fwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* ray_rec,
                                   const float* conic_opac, const float* rgb, const float* lnv, const float* depth,
                                   const float* pixel_rays, const uint32_t* vals_sorted, const uint32_t* tile_ranges,
                                   float* image, float* final_T, uint32_t* n_contrib, float* depth_img, float* alpha_img,
                                   void* stream);
int32_t xpr_rasterize_ray_feat_bwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* ray_rec,
                                   const float* conic_opac, const float* rgb, const float* lnv, const float* depth,
                                   const float* pixel_rays, const uint32_t* vals_sorted, const uint32_t* tile_ranges,
                                   const float* final_T, const uint32_t* n_contrib, const float* dL_dimage,
                                   const float* dL_ddepth, const float* dL_dalpha, float* g_ray_acc, float* g_opac,
                                   float* g_rgb, float* g_depth, int32_t zero_init, void* stream);
int32_t xpr_rasterize_feat_fwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* shade_rec,
                               const uint32_t* vals_sorted, const uint32_t* tile_ranges,
                               float* image, float* final_T, uint32_t* n_contrib, float* depth_img,
                               float* alpha_img, void* stream);
int32_t xpr_rasterize_feat_bwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* shade_rec,
                               const uint32_t* vals_sorted, const uint32_t* tile_ranges,
                               const float* final_T, const uint32_t* n_contrib, const float* dL_dimage,
                               const float* dL_ddepth, const float* dL_dalpha,
                               float* g_mean2d, float* g_conic, float* g_opac, float* g_rgb, float* g_depth,
                               int32_t zero_init, void* stream);
int32_t xpr_depth_bwd(int64_t N, const xpr_camera* cam, const uint32_t* tile_count, const float* g_depth,
                      float* g_means, void* stream);

/*
 * N-channel features (same reading C31; SURVEY 8(f) f3 "N-channel feature outputs"): feat [N,C] row-major, any C >= 1;
 *   feat_img[H,W,C] = sum_k feat[g_k,:] alpha_k T_k over the colour pass's contributing sequence, no background.
 * xpr_rasterize_featn_fwd -- REPLAYS the walk of a finished colour pass (xpr_rasterize_fwd or xpr_rasterize_feat_fwd on
 *   the same lists): in n_contrib[H,W]; out feat_img (fully overwritten).  One launch, grid = (tiles, ceil(C / 8)).
 * xpr_rasterize_featn_bwd -- reverse mode for dL_dfeat[H,W,C] ALONE: ADDS that part to g_mean2d[N,2], g_conic[N,3],
 *   g_opac[N] (so it can follow xpr_rasterize_bwd / _feat_bwd, whose parts it completes: every step is linear in the
 *   incoming gradient) and to g_feat[N,C].  zero_init bit 0: zero-fill g_mean2d, g_conic, g_opac first; bit 1: zero-fill
 *   g_feat first.  in: final_T, n_contrib of the colour pass.
 * Errors: C < 1, N < 0, null / misaligned pointer -> XPR_ERR_INVALID_ARG before any launch.
 */
int32_t xpr_rasterize_featn_fwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* mean2d,
                                const float* conic_opac, const float* lnv, const float* feat, int32_t C,
                                const uint32_t* vals_sorted, const uint32_t* tile_ranges,
                                const uint32_t* n_contrib, float* feat_img, void* stream);
int32_t xpr_rasterize_featn_bwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* mean2d,
                                const float* conic_opac, const float* lnv, const float* feat, int32_t C,
                                const uint32_t* vals_sorted, const uint32_t* tile_ranges,
                                const float* final_T, const uint32_t* n_contrib, const float* dL_dfeat,
                                float* g_mean2d, float* g_conic, float* g_opac, float* g_feat,
                                int32_t zero_init, void* stream);

/*
 * ---- XPR-LinPrim (PAPER A.1.3 L506-697, Listings 4-5, Eq. 2): forward and backward path ----
 * Primitive: the octahedron {x : |S^-1 R^T (x - mu)|_1 <= 1} with homogeneous density
 * sigma = -log(1 - 0.99 o) / (2 min(s)) (L506-524); alpha = 1 - exp(-sigma (tau_exit - tau_enter)) (L528).
 * The body of the paper's `project` listing is lost in the extraction (L545-560); DESIGN.md section 3 readings L1-L6
 * fill it and both sides (oracle/xpr_oracle_lin.inc, these kernels) follow them.
 *
 * xpr_lin_project -- Vertex-shader stage: p = W mu + t, dist = |p| (the sort depth, "Euclidean depth" L532, L2),
 *   A = J W R diag(s) with J = (d pixel / dp of the pinhole; p^T / |p|) (L534-536, L1), the projected octahedron
 *   {|A^-1 (p2D - mu2D, tau)|_1 <= 1} written as four slab pairs with normals n = c0 +- c1 +- c2, c_k the rows of
 *   A^-1 (L538-542): tau in [m_i - h_i, m_i + h_i], m_i = -(kx_i dx + ky_i dy), kx = n_x / n_z, ky = n_y / n_z,
 *   h = 1 / |n_z| (h = +inf when |n_z| < 1e-12: the slab does not bound tau, L566, L4); footprint = the exact
 *   axis-aligned box of the shadow, half extents max_j |A[0][j]|, max_j |A[1][j]| (L3); colour as xpr_project (C5).
 *   in : means[N,3], scales[N,3] (activated, > 0), quats[N,4] (w,x,y,z), opacities[N] in [0,1),
 *        sh[N,K,3] as xpr_project (quaternions are not renormalised, C3); cam: ONE pinhole camera (fisheye, cfg->views > 1 -> XPR_ERR_UNSUPPORTED).
 *   out: lin_rec[N,20] fp32, 16-byte aligned = (mu2D.x, mu2D.y, sigma, dist | (kx_i, ky_i, h_i) i = 0..3 | r, g, b, 0),
 *        all 0 for a culled primitive; depth[N] = dist; tile_rect[N,4], tile_count[N] as xpr_project.
 *   Culled: p_z <= z_near, non-finite record, empty rectangle.
 *
 * xpr_bin_sort_lin -- xpr_bin_sort for LinPrim pairs; with cfg->tile_cull != 0 a candidate (primitive, tile) is kept
 *   iff Eq. 2's upper bound of the chord over the tile (corners x0 = 16 tx + 1/2, x1 = 16 (tx + 1) + 1/2 as the listing
 *   prints them, L6; bound = max(0, min_{i,j} max_corners (m_i - m_j) + h_i + h_j)) gives sigma dtau >= -log(1 -
 *   alpha_thresh) (L589-612, L633-676).  The bound is a minimum of functions convex in the tile position, so along one
 *   tile row the kept tiles form ONE interval: the call shrinks each row of the rectangle from both ends.
 *   Arguments, capacity contract and error behaviour as xpr_bin_sort_cull, with lin_rec in place of the tile-cull data.
 *
 * xpr_lin_rasterize_fwd -- Shader stage (Alg. 1; evaluate L618-629): per pixel, front to back over the tile's
 *   list: x = sigma (min_i (m_i + h_i) - max_i (m_i - h_i)) or 0 when that is not positive; skip when
 *   x < -log(1 - alpha_thresh) (decided on x, rule R3); alpha = min(alpha_max, 1 - exp(-x)); T' = T (1 - alpha); stop
 *   WITHOUT blending if T' < t_min; C += rgb alpha T; T = T'; finally C += T bg (L5: the common rules C11-C13).
 *   out: image[H,W,3], final_T[H,W], n_contrib[H,W] (1-based list position of the last blended primitive).
 * xpr_lin_rasterize_stats -- the same walk, no image: stats[4] (DEVICE uint64) = {(pixel, primitive) evaluations,
 *   those that pass the gate, those blended, sum of n_contrib}.
 * Errors (all four): null cam / cfg, N < 0, misaligned pointer -> XPR_ERR_INVALID_ARG; cfg->tile != 16, a fisheye
 *   camera or cfg->views > 1 -> XPR_ERR_UNSUPPORTED; nothing is launched in either case.
 *
 * xpr_lin_rasterize_bwd -- reverse mode through the loop above (the paper relies on AD): back to front from
 *   n_contrib, T_k = T_{k+1} / (1 - alpha_k); dL/dalpha_k as xpr_rasterize_bwd; alpha = min(alpha_max, 1 - exp(-x)): no
 *   gradient where the clamp is active (C14), else G = dL/dx = exp(-x) dL/dalpha; with en / ex the slab pairs the ray
 *   enters / leaves through (the first one on ties): dL/dsigma += dtau G, and with gm = sigma G: dL/dh_ex += gm,
 *   dL/dh_en += gm, dL/dkx_ex -= dx gm, dL/dkx_en += dx gm (ky with dy), dL/dmu2D += gm ((kx, ky)_ex - (kx, ky)_en);
 *   gates, exit and the choice of en / ex are piecewise constant (C15).
 *   in : lin_rec, vals_sorted, tile_ranges as the forward; final_T[H,W], n_contrib[H,W] of the forward; dL_dimage[H,W,3].
 *   out: g_lin_rec[N,20] fp32, 16-byte aligned, in the layout of lin_rec (slots 3 and 19 stay 0): zero-filled by the
 *        call, then accumulated with fp32 atomics (summation order not fixed: DESIGN.md section 5).
 * xpr_lin_project_bwd -- reverse mode through xpr_lin_project: slabs -> A^-1 (dL/dA = -A^-T dL/dA^-1 A^-T) -> A = J W R
 *   diag(s) -> (mu, s, q); sigma(o, min s) (the first shortest half-axis on ties); J(p) and mu2D -> mu; colour as
 *   xpr_project_bwd (clamped channels carry none, C16).  The forward is recomputed in fp32, the chain rule runs in fp64.
 *   in : the parameters, tile_count[N] and lin_rec[N,20] of the forward, g_lin_rec[N,20].
 *   out: g_means[N,3], g_scales[N,3], g_quats[N,4] (16-byte aligned), g_opacities[N], g_sh[N,K,3] (16-byte aligned):
 *        every element written, zeros for culled primitives.  depth (sort only) and the footprint carry no gradient.
 * Errors as above.
 */
int32_t xpr_lin_project(int64_t N, const float* means, const float* scales, const float* quats, const float* opacities,
                        const float* sh, const xpr_camera* cam, const xpr_config* cfg, float* lin_rec, float* depth,
                        int32_t* tile_rect, uint32_t* tile_count, void* stream);
int32_t xpr_bin_sort_lin(int64_t N, const float* depth, const int32_t* tile_rect, const uint32_t* tile_count,
                         const float* lin_rec, const xpr_camera* cam, const xpr_config* cfg, int64_t pair_capacity,
                         uint64_t* keys_sorted, uint32_t* vals_sorted, uint32_t* tile_ranges, int64_t* num_pairs_host,
                         void* workspace, size_t workspace_bytes, void* stream);
int32_t xpr_lin_rasterize_fwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* lin_rec,
                              const uint32_t* vals_sorted, const uint32_t* tile_ranges, float* image, float* final_T,
                              uint32_t* n_contrib, void* stream);
int32_t xpr_lin_rasterize_stats(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* lin_rec,
                                const uint32_t* vals_sorted, const uint32_t* tile_ranges, uint64_t* stats, void* stream);
int32_t xpr_lin_rasterize_bwd(const xpr_camera* cam, const xpr_config* cfg, int64_t N, const float* lin_rec,
                              const uint32_t* vals_sorted, const uint32_t* tile_ranges, const float* final_T,
                              const uint32_t* n_contrib, const float* dL_dimage, float* g_lin_rec, void* stream);
int32_t xpr_lin_project_bwd(int64_t N, const float* means, const float* scales, const float* quats, const float* opacities,
                            const float* sh, const xpr_camera* cam, const xpr_config* cfg, const uint32_t* tile_count,
                            const float* lin_rec, const float* g_lin_rec, float* g_means, float* g_scales, float* g_quats,
                            float* g_opacities, float* g_sh, void* stream);

/*
 * xpr_loss_grad -- convenience for the caller's side of the step (reading C21: the loss lives outside the path):
 * dL/dimage of the two losses BASELINE.json's configs name, as sums over all n = H*W*3 values, in one pass:
 *   kind 0: L = sum |I - target|    -> dL = sign(I - target);      kind 1: L = sum (I - target)^2 -> dL = 2 (I - target).
 * image, target, dL_dimage: DEVICE fp32 [n], 16-byte aligned.
 */
int32_t xpr_loss_grad(int32_t kind, int64_t n, const float* image, const float* target, float* dL_dimage,
                      void* stream);

#ifdef __cplusplus
}
#endif
#endif /* XPR_H */
