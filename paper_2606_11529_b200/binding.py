"""Thin ctypes binding of libxpr.so (include/xpr.h): same names, argument marshalling only.

Every step of the hot path runs inside the CUDA library; PyTorch is used for device memory and
streams.  There is no CPU fallback: if libxpr.so is missing or a call fails, an exception is raised.
Nothing here imports ``oracle/``.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libxpr.so")

XPR_OK, XPR_ERR_INVALID_ARG, XPR_ERR_CAPACITY, XPR_ERR_CUDA, XPR_ERR_UNSUPPORTED = 0, 1, 2, 3, 4
XPR_ERR_SCRATCH_LIMIT = 5
XPR_STATIC_SCRATCH_BYTES = 16 * 1024 * 1024
FLAG_VISIBLE, FLAG_CLAMP_U, FLAG_CLAMP_V, FLAG_RGB_POS_R, FLAG_RGB_POS_G, FLAG_RGB_POS_B = 1, 2, 4, 8, 16, 32

SYMBOLS = ("xpr_status_string", "xpr_last_cuda_error", "xpr_version", "xpr_project", "xpr_bin_sort_workspace",
           "xpr_shade_record", "xpr_bin_sort", "xpr_bin_sort_cull", "xpr_rasterize_fwd", "xpr_rasterize_stats", "xpr_rasterize_bwd", "xpr_project_bwd",
           "xpr_pixel_info", "xpr_project_ray", "xpr_rasterize_ray_fwd", "xpr_rasterize_ray_stats", "xpr_rasterize_ray_bwd",
           "xpr_ray_bwd", "xpr_rasterize_feat_fwd", "xpr_rasterize_feat_bwd", "xpr_depth_bwd", "xpr_rasterize_featn_fwd", "xpr_rasterize_featn_bwd", "xpr_loss_grad",
           "xpr_lin_project", "xpr_bin_sort_lin", "xpr_lin_rasterize_fwd", "xpr_lin_rasterize_stats",
           "xpr_lin_rasterize_bwd", "xpr_lin_project_bwd", "xpr_rasterize_ray_feat_fwd", "xpr_rasterize_ray_feat_bwd",
           "xpr_project_bwd_fill", "xpr_project_bwd_filled", "xpr_bin_sort_static", "xpr_rasterize_bwd_loss")


class XprCamera(C.Structure):
    _fields_ = [("model", C.c_int32), ("width", C.c_int32), ("height", C.c_int32),
                ("fx", C.c_float), ("fy", C.c_float), ("cx", C.c_float), ("cy", C.c_float),
                ("k", C.c_float * 4), ("w2c", C.c_float * 12)]


class XprConfig(C.Structure):
    _fields_ = [("projection", C.c_int32), ("sh_degree", C.c_int32), ("tile", C.c_int32), ("antialias", C.c_int32),
                ("alpha_thresh", C.c_float), ("alpha_max", C.c_float), ("t_min", C.c_float), ("z_near", C.c_float),
                ("lowpass", C.c_float), ("ut_alpha", C.c_float), ("ut_beta", C.c_float), ("ut_kappa", C.c_float),
                ("bg", C.c_float * 3), ("tile_cull", C.c_int32), ("tile_order", C.c_void_p), ("views", C.c_int32)]


class XprError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = lib().xpr_status_string(C.c_int32(status)).decode()
        if status == XPR_ERR_CUDA:
            msg += f" [cudaError {lib().xpr_last_cuda_error()}]"
        super().__init__(f"{where}: {msg}")


_lib = None


def lib():
    """Load libxpr.so (built in-tree by ``python -m paper_2606_11529_b200.build``); fail loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} not found: build it with `python -m paper_2606_11529_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.xpr_status_string.restype = C.c_char_p
        for name in SYMBOLS[1:]:
            getattr(L, name).restype = C.c_int32
        _lib = L
    return _lib


def make_camera(cam) -> XprCamera:
    """cam: any object with model,width,height,fx,fy,cx,cy,k,w2c (e.g. scenes.Camera)."""
    c = XprCamera()
    c.model, c.width, c.height = int(cam.model), int(cam.width), int(cam.height)
    c.fx, c.fy, c.cx, c.cy = float(cam.fx), float(cam.fy), float(cam.cx), float(cam.cy)
    for i in range(4):
        c.k[i] = float(cam.k[i])
    w = [float(v) for row in cam.w2c for v in row]
    for i in range(12):
        c.w2c[i] = w[i]
    return c


def make_config(d: dict) -> XprConfig:
    c = XprConfig()
    c.projection, c.sh_degree, c.tile, c.antialias = int(d["projection"]), int(d["sh_degree"]), int(d["tile"]), int(d["antialias"])
    c.alpha_thresh, c.alpha_max, c.t_min = float(d["alpha_thresh"]), float(d["alpha_max"]), float(d["t_min"])
    c.z_near, c.lowpass = float(d["z_near"]), float(d["lowpass"])
    c.ut_alpha, c.ut_beta, c.ut_kappa = float(d["ut_alpha"]), float(d["ut_beta"]), float(d["ut_kappa"])
    for i in range(3):
        c.bg[i] = float(d["bg"][i])
    c.tile_cull = int(d.get("tile_cull", 0))
    c.tile_order = None      # the pipeline sets tile_order to a device buffer of T uint32 (scheduling only)
    c.views = int(d.get("views", 1))
    return c


def make_cameras(cams):
    """A contiguous array of xpr_camera for a batch of views (xpr_config.views)."""
    arr = (XprCamera * len(cams))()
    for i, cam in enumerate(cams):
        C.memmove(C.byref(arr[i]), C.byref(make_camera(cam)), C.sizeof(XprCamera))
    return arr


def num_tiles(cam: XprCamera, cfg: XprConfig):
    ts = int(cfg.tile)
    return (int(cam.width) + ts - 1) // ts, (int(cam.height) + ts - 1) // ts


_F32, _I32, _U8, _I64 = (torch.float32,), (torch.int32, torch.uint32), (torch.uint8,), (torch.int64, torch.uint64)


def _p(t, dtypes=None):
    """Device pointer of a contiguous CUDA tensor (None -> NULL).  `dtypes`: the element types the C signature
    accepts for this argument (a tensor of another type would be reinterpreted silently by the library)."""
    if t is None:
        return C.c_void_p(0)
    if not t.is_cuda:
        raise TypeError("xpr: expected a CUDA tensor (the library takes device pointers; no CPU fallback)")
    if not t.is_contiguous():
        raise ValueError("xpr: tensor must be contiguous")
    if dtypes is not None and t.dtype not in dtypes:
        raise TypeError(f"xpr: expected a tensor of {' / '.join(str(d) for d in dtypes)}, got {t.dtype}")
    return C.c_void_p(t.data_ptr())


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _check(status: int, where: str):
    if status != XPR_OK:
        raise XprError(status, where)


def xpr_version() -> int:
    return int(lib().xpr_version())


def xpr_project(means, scales, quats, opacities, sh, cam: XprCamera, cfg: XprConfig, mean2d, conic_opac, rgb, depth,
                lnv, tile_rect, tile_count, flags, shade_rec=None, stream=None):
    N = int(means.shape[0])
    _check(lib().xpr_project(C.c_int64(N), _p(means, _F32), _p(scales, _F32), _p(quats, _F32), _p(opacities, _F32), _p(sh, _F32), C.byref(cam),
                             C.byref(cfg), _p(mean2d, _F32), _p(conic_opac, _F32), _p(rgb, _F32), _p(depth, _F32), _p(lnv, _F32), _p(tile_rect, _I32),
                             _p(tile_count, _I32), _p(flags, _U8), _p(shade_rec, _F32), _stream(stream)), "xpr_project")


def xpr_shade_record(mean2d, conic_opac, rgb, lnv, depth, tile_count, shade_rec, stream=None):
    N = int(mean2d.shape[0])
    _check(lib().xpr_shade_record(C.c_int64(N), _p(mean2d, _F32), _p(conic_opac, _F32), _p(rgb, _F32), _p(lnv, _F32),
                                  _p(depth, _F32), _p(tile_count, _I32), _p(shade_rec, _F32), _stream(stream)),
           "xpr_shade_record")


def xpr_bin_sort_workspace(N: int, pair_capacity: int, n_tiles: int) -> int:
    out = C.c_size_t(0)
    _check(lib().xpr_bin_sort_workspace(C.c_int64(N), C.c_int64(pair_capacity), C.c_int32(n_tiles), C.byref(out)),
           "xpr_bin_sort_workspace")
    return int(out.value)


def xpr_bin_sort(depth, tile_rect, tile_count, cam: XprCamera, cfg: XprConfig, pair_capacity: int, keys_sorted,
                 vals_sorted, tile_ranges, workspace, stream=None, raise_on_capacity: bool = True, sync: bool = True,
                 cull_data=None, lin_rec=None):
    """Returns (status, I).  On XPR_ERR_CAPACITY I is the required capacity.
    cull_data = (mean2d, conic_opac, lnv): call xpr_bin_sort_cull (tile_cull applied when cfg.tile_cull != 0).
    lin_rec: call xpr_bin_sort_lin (LinPrim pairs; Eq. 2 bound when cfg.tile_cull != 0).
    sync=False: num_pairs_host = NULL -- nothing waits for the host, I is returned as None and stays in the
    first 8 bytes of `workspace` (xpr.h); the caller checks it against pair_capacity later."""
    N = int(tile_count.shape[0])
    n_pairs = C.c_int64(0)
    tail = (C.byref(cam), C.byref(cfg), C.c_int64(pair_capacity), _p(keys_sorted, _I64), _p(vals_sorted, _I32), _p(tile_ranges, _I32),
            C.byref(n_pairs) if sync else None, _p(workspace, _U8), C.c_size_t(workspace.numel() * workspace.element_size()),
            _stream(stream))
    if lin_rec is not None:
        st = lib().xpr_bin_sort_lin(C.c_int64(N), _p(depth, _F32), _p(tile_rect, _I32), _p(tile_count, _I32), _p(lin_rec, _F32), *tail)
    elif cull_data is None:
        st = lib().xpr_bin_sort(C.c_int64(N), _p(depth, _F32), _p(tile_rect, _I32), _p(tile_count, _I32), *tail)
    else:
        st = lib().xpr_bin_sort_cull(C.c_int64(N), _p(depth, _F32), _p(tile_rect, _I32), _p(tile_count, _I32), _p(cull_data[0], _F32),
                                     _p(cull_data[1], _F32), _p(cull_data[2], _F32), *tail)
    if not sync:
        _check(st, "xpr_bin_sort")
        return st, None
    if st == XPR_ERR_CAPACITY and not raise_on_capacity:
        return st, int(n_pairs.value)
    _check(st, "xpr_bin_sort")
    return st, int(n_pairs.value)


def xpr_bin_sort_static(depth, tile_rect, tile_count, cam: XprCamera, cfg: XprConfig, pair_capacity: int, keys_sorted,
                        vals_sorted, tile_ranges, cull_data=None, stream=None, sync: bool = True):
    """xpr_bin_sort[_cull] on the library's static scratch (no workspace, no allocation; xpr.h).  Returns (status, I);
    raises XprError (XPR_ERR_SCRATCH_LIMIT) when the sizes need more than XPR_STATIC_SCRATCH_BYTES."""
    N = int(tile_count.shape[0])
    n_pairs = C.c_int64(0)
    cd = cull_data if cull_data is not None else (None, None, None)
    st = lib().xpr_bin_sort_static(C.c_int64(N), _p(depth, _F32), _p(tile_rect, _I32), _p(tile_count, _I32),
                                   _p(cd[0], _F32), _p(cd[1], _F32), _p(cd[2], _F32), C.byref(cam), C.byref(cfg),
                                   C.c_int64(pair_capacity), _p(keys_sorted, _I64), _p(vals_sorted, _I32),
                                   _p(tile_ranges, _I32), C.byref(n_pairs) if sync else None, _stream(stream))
    _check(st, "xpr_bin_sort_static")
    return st, (int(n_pairs.value) if sync else None)


def xpr_rasterize_fwd(cam: XprCamera, cfg: XprConfig, shade_rec, vals_sorted, tile_ranges, image, final_T, n_contrib,
                      stream=None):
    N = int(shade_rec.shape[0])
    _check(lib().xpr_rasterize_fwd(C.byref(cam), C.byref(cfg), C.c_int64(N), _p(shade_rec, _F32), _p(vals_sorted, _I32),
                                   _p(tile_ranges, _I32), _p(image, _F32), _p(final_T, _F32), _p(n_contrib, _I32),
                                   _stream(stream)), "xpr_rasterize_fwd")


def xpr_rasterize_stats(cam: XprCamera, cfg: XprConfig, shade_rec, vals_sorted, tile_ranges, stats, stream=None):
    N = int(shade_rec.shape[0])
    _check(lib().xpr_rasterize_stats(C.byref(cam), C.byref(cfg), C.c_int64(N), _p(shade_rec, _F32),
                                     _p(vals_sorted, _I32), _p(tile_ranges, _I32), _p(stats, _I64), _stream(stream)),
           "xpr_rasterize_stats")


def xpr_rasterize_bwd(cam: XprCamera, cfg: XprConfig, shade_rec, vals_sorted, tile_ranges, final_T, n_contrib,
                      dL_dimage, g_mean2d, g_conic, g_opac, g_rgb, zero_init: bool = True, stream=None):
    N = int(shade_rec.shape[0])
    _check(lib().xpr_rasterize_bwd(C.byref(cam), C.byref(cfg), C.c_int64(N), _p(shade_rec, _F32), _p(vals_sorted, _I32),
                                   _p(tile_ranges, _I32), _p(final_T, _F32), _p(n_contrib, _I32), _p(dL_dimage, _F32),
                                   _p(g_mean2d, _F32), _p(g_conic, _F32), _p(g_opac, _F32), _p(g_rgb, _F32),
                                   C.c_int32(1 if zero_init else 0), _stream(stream)), "xpr_rasterize_bwd")


def xpr_rasterize_bwd_loss(cam: XprCamera, cfg: XprConfig, shade_rec, vals_sorted, tile_ranges, image, final_T, n_contrib,
                           kind: str, target, g_mean2d, g_conic, g_opac, g_rgb, zero_init: bool = True, stream=None):
    """xpr_loss_grad + xpr_rasterize_bwd in one launch: kind "l1" (sum |I - target|) or "l2" (sum (I - target)^2)."""
    N = int(shade_rec.shape[0])
    _check(lib().xpr_rasterize_bwd_loss(C.byref(cam), C.byref(cfg), C.c_int64(N), _p(shade_rec, _F32), _p(vals_sorted, _I32),
                                        _p(tile_ranges, _I32), _p(image, _F32), _p(final_T, _F32), _p(n_contrib, _I32),
                                        C.c_int32({"l1": 0, "l2": 1}[kind]), _p(target, _F32), _p(g_mean2d, _F32),
                                        _p(g_conic, _F32), _p(g_opac, _F32), _p(g_rgb, _F32),
                                        C.c_int32(1 if zero_init else 0), _stream(stream)), "xpr_rasterize_bwd_loss")


def xpr_project_bwd_fill(cfg: XprConfig, g_means, g_scales, g_quats, g_opacities, g_sh, stream=None):
    N = int(g_means.shape[0])
    _check(lib().xpr_project_bwd_fill(C.c_int64(N), C.byref(cfg), _p(g_means, _F32), _p(g_scales, _F32), _p(g_quats, _F32),
                                      _p(g_opacities, _F32), _p(g_sh, _F32), _stream(stream)), "xpr_project_bwd_fill")


def xpr_project_bwd(means, scales, quats, opacities, sh, cam: XprCamera, cfg: XprConfig, tile_count, flags, g_mean2d,
                    g_conic, g_opac, g_rgb, g_means, g_scales, g_quats, g_opacities, g_sh, stream=None, filled: bool = False):
    """filled=True: xpr_project_bwd_filled (the outputs were zero-filled by xpr_project_bwd_fill, ordered by the caller)."""
    N = int(means.shape[0])
    fn = lib().xpr_project_bwd_filled if filled else lib().xpr_project_bwd
    _check(fn(C.c_int64(N), _p(means, _F32), _p(scales, _F32), _p(quats, _F32), _p(opacities, _F32), _p(sh, _F32), C.byref(cam),
                                 C.byref(cfg), _p(tile_count, _I32), _p(flags, _U8), _p(g_mean2d, _F32), _p(g_conic, _F32), _p(g_opac, _F32),
                                 _p(g_rgb, _F32), _p(g_means, _F32), _p(g_scales, _F32), _p(g_quats, _F32), _p(g_opacities, _F32), _p(g_sh, _F32),
                                 _stream(stream)), "xpr_project_bwd")


# ---- XPR-3DGUT ray evaluation (xpr.h) ----------------------------------------------------------

def xpr_pixel_info(cam: XprCamera, pixel_rays, stream=None):
    _check(lib().xpr_pixel_info(C.byref(cam), _p(pixel_rays, _F32), _stream(stream)), "xpr_pixel_info")


def xpr_project_ray(means, scales, quats, cam: XprCamera, tile_count, ray_rec, stream=None):
    N = int(means.shape[0])
    _check(lib().xpr_project_ray(C.c_int64(N), _p(means, _F32), _p(scales, _F32), _p(quats, _F32), C.byref(cam), _p(tile_count, _I32),
                                 _p(ray_rec, _F32), _stream(stream)), "xpr_project_ray")


def xpr_rasterize_ray_fwd(cam: XprCamera, cfg: XprConfig, ray_rec, conic_opac, rgb, lnv, pixel_rays, vals_sorted,
                          tile_ranges, image, final_T, n_contrib, stream=None):
    N = int(ray_rec.shape[0])
    _check(lib().xpr_rasterize_ray_fwd(C.byref(cam), C.byref(cfg), C.c_int64(N), _p(ray_rec, _F32), _p(conic_opac, _F32), _p(rgb, _F32),
                                       _p(lnv, _F32), _p(pixel_rays, _F32), _p(vals_sorted, _I32), _p(tile_ranges, _I32), _p(image, _F32),
                                       _p(final_T, _F32), _p(n_contrib, _I32), _stream(stream)), "xpr_rasterize_ray_fwd")


def xpr_rasterize_ray_stats(cam: XprCamera, cfg: XprConfig, ray_rec, conic_opac, rgb, lnv, pixel_rays, vals_sorted,
                            tile_ranges, stats, stream=None):
    N = int(ray_rec.shape[0])
    _check(lib().xpr_rasterize_ray_stats(C.byref(cam), C.byref(cfg), C.c_int64(N), _p(ray_rec, _F32), _p(conic_opac, _F32),
                                         _p(rgb, _F32), _p(lnv, _F32), _p(pixel_rays, _F32), _p(vals_sorted, _I32), _p(tile_ranges, _I32),
                                         _p(stats, _I64), _stream(stream)), "xpr_rasterize_ray_stats")


def xpr_rasterize_ray_bwd(cam: XprCamera, cfg: XprConfig, ray_rec, conic_opac, rgb, lnv, pixel_rays, vals_sorted,
                          tile_ranges, final_T, n_contrib, dL_dimage, g_ray_acc, g_opac, g_rgb, zero_init: bool = True,
                          stream=None):
    N = int(ray_rec.shape[0])
    _check(lib().xpr_rasterize_ray_bwd(C.byref(cam), C.byref(cfg), C.c_int64(N), _p(ray_rec, _F32), _p(conic_opac, _F32), _p(rgb, _F32),
                                       _p(lnv, _F32), _p(pixel_rays, _F32), _p(vals_sorted, _I32), _p(tile_ranges, _I32), _p(final_T, _F32),
                                       _p(n_contrib, _I32), _p(dL_dimage, _F32), _p(g_ray_acc, _F32), _p(g_opac, _F32), _p(g_rgb, _F32),
                                       C.c_int32(1 if zero_init else 0), _stream(stream)), "xpr_rasterize_ray_bwd")


def xpr_rasterize_ray_feat_fwd(cam: XprCamera, cfg: XprConfig, ray_rec, conic_opac, rgb, lnv, depth, pixel_rays, vals_sorted,
                               tile_ranges, image, final_T, n_contrib, depth_img, alpha_img, stream=None):
    N = int(ray_rec.shape[0])
    _check(lib().xpr_rasterize_ray_feat_fwd(C.byref(cam), C.byref(cfg), C.c_int64(N), _p(ray_rec, _F32), _p(conic_opac, _F32),
                                            _p(rgb, _F32), _p(lnv, _F32), _p(depth, _F32), _p(pixel_rays, _F32),
                                            _p(vals_sorted, _I32), _p(tile_ranges, _I32), _p(image, _F32), _p(final_T, _F32),
                                            _p(n_contrib, _I32), _p(depth_img, _F32), _p(alpha_img, _F32), _stream(stream)),
           "xpr_rasterize_ray_feat_fwd")


def xpr_rasterize_ray_feat_bwd(cam: XprCamera, cfg: XprConfig, ray_rec, conic_opac, rgb, lnv, depth, pixel_rays, vals_sorted,
                               tile_ranges, final_T, n_contrib, dL_dimage, dL_ddepth, dL_dalpha, g_ray_acc, g_opac, g_rgb,
                               g_depth, zero_init: bool = True, stream=None):
    N = int(ray_rec.shape[0])
    _check(lib().xpr_rasterize_ray_feat_bwd(C.byref(cam), C.byref(cfg), C.c_int64(N), _p(ray_rec, _F32), _p(conic_opac, _F32),
                                            _p(rgb, _F32), _p(lnv, _F32), _p(depth, _F32), _p(pixel_rays, _F32),
                                            _p(vals_sorted, _I32), _p(tile_ranges, _I32), _p(final_T, _F32), _p(n_contrib, _I32),
                                            _p(dL_dimage, _F32), _p(dL_ddepth, _F32), _p(dL_dalpha, _F32), _p(g_ray_acc, _F32),
                                            _p(g_opac, _F32), _p(g_rgb, _F32), _p(g_depth, _F32),
                                            C.c_int32(1 if zero_init else 0), _stream(stream)), "xpr_rasterize_ray_feat_bwd")


def xpr_ray_bwd(means, scales, quats, cam: XprCamera, tile_count, g_ray_acc, g_means, g_scales, g_quats, stream=None):
    N = int(means.shape[0])
    _check(lib().xpr_ray_bwd(C.c_int64(N), _p(means, _F32), _p(scales, _F32), _p(quats, _F32), C.byref(cam), _p(tile_count, _I32),
                             _p(g_ray_acc, _F32), _p(g_means, _F32), _p(g_scales, _F32), _p(g_quats, _F32), _stream(stream)), "xpr_ray_bwd")


# ---- Rendered depth and accumulated opacity (xpr.h) --------------------------------------------

def xpr_rasterize_feat_fwd(cam: XprCamera, cfg: XprConfig, shade_rec, vals_sorted, tile_ranges, image, final_T,
                           n_contrib, depth_img, alpha_img, stream=None):
    N = int(shade_rec.shape[0])
    _check(lib().xpr_rasterize_feat_fwd(C.byref(cam), C.byref(cfg), C.c_int64(N), _p(shade_rec, _F32),
                                        _p(vals_sorted, _I32), _p(tile_ranges, _I32), _p(image, _F32),
                                        _p(final_T, _F32), _p(n_contrib, _I32), _p(depth_img, _F32),
                                        _p(alpha_img, _F32), _stream(stream)), "xpr_rasterize_feat_fwd")


def xpr_rasterize_feat_bwd(cam: XprCamera, cfg: XprConfig, shade_rec, vals_sorted, tile_ranges, final_T, n_contrib,
                           dL_dimage, dL_ddepth, dL_dalpha, g_mean2d, g_conic, g_opac, g_rgb, g_depth,
                           zero_init: bool = True, stream=None):
    N = int(shade_rec.shape[0])
    _check(lib().xpr_rasterize_feat_bwd(C.byref(cam), C.byref(cfg), C.c_int64(N), _p(shade_rec, _F32),
                                        _p(vals_sorted, _I32), _p(tile_ranges, _I32), _p(final_T, _F32),
                                        _p(n_contrib, _I32), _p(dL_dimage, _F32), _p(dL_ddepth, _F32),
                                        _p(dL_dalpha, _F32), _p(g_mean2d, _F32), _p(g_conic, _F32), _p(g_opac, _F32),
                                        _p(g_rgb, _F32), _p(g_depth, _F32), C.c_int32(1 if zero_init else 0),
                                        _stream(stream)), "xpr_rasterize_feat_bwd")


def xpr_depth_bwd(cam: XprCamera, tile_count, g_depth, g_means, stream=None):
    N = int(tile_count.shape[0])
    _check(lib().xpr_depth_bwd(C.c_int64(N), C.byref(cam), _p(tile_count, _I32), _p(g_depth, _F32), _p(g_means, _F32), _stream(stream)),
           "xpr_depth_bwd")


def xpr_rasterize_featn_fwd(cam: XprCamera, cfg: XprConfig, mean2d, conic_opac, lnv, feat, vals_sorted, tile_ranges,
                            n_contrib, feat_img, stream=None):
    N, Cn = int(feat.shape[0]), int(feat.shape[1])
    _check(lib().xpr_rasterize_featn_fwd(C.byref(cam), C.byref(cfg), C.c_int64(N), _p(mean2d, _F32), _p(conic_opac, _F32), _p(lnv, _F32),
                                         _p(feat, _F32), C.c_int32(Cn), _p(vals_sorted, _I32), _p(tile_ranges, _I32), _p(n_contrib, _I32),
                                         _p(feat_img, _F32), _stream(stream)), "xpr_rasterize_featn_fwd")


def xpr_rasterize_featn_bwd(cam: XprCamera, cfg: XprConfig, mean2d, conic_opac, lnv, feat, vals_sorted, tile_ranges,
                            final_T, n_contrib, dL_dfeat, g_mean2d, g_conic, g_opac, g_feat, zero_init: int = 2,
                            stream=None):
    N, Cn = int(feat.shape[0]), int(feat.shape[1])
    _check(lib().xpr_rasterize_featn_bwd(C.byref(cam), C.byref(cfg), C.c_int64(N), _p(mean2d, _F32), _p(conic_opac, _F32), _p(lnv, _F32),
                                         _p(feat, _F32), C.c_int32(Cn), _p(vals_sorted, _I32), _p(tile_ranges, _I32), _p(final_T, _F32),
                                         _p(n_contrib, _I32), _p(dL_dfeat, _F32), _p(g_mean2d, _F32), _p(g_conic, _F32), _p(g_opac, _F32),
                                         _p(g_feat, _F32), C.c_int32(int(zero_init)), _stream(stream)),
           "xpr_rasterize_featn_bwd")


def xpr_lin_project(means, scales, quats, opacities, sh, cam: XprCamera, cfg: XprConfig, lin_rec, depth, tile_rect,
                    tile_count, stream=None):
    N = int(means.shape[0])
    _check(lib().xpr_lin_project(C.c_int64(N), _p(means, _F32), _p(scales, _F32), _p(quats, _F32), _p(opacities, _F32),
                                 _p(sh, _F32), C.byref(cam), C.byref(cfg), _p(lin_rec, _F32), _p(depth, _F32),
                                 _p(tile_rect, _I32), _p(tile_count, _I32), _stream(stream)), "xpr_lin_project")


def xpr_lin_rasterize_fwd(cam: XprCamera, cfg: XprConfig, lin_rec, vals_sorted, tile_ranges, image, final_T, n_contrib,
                          stream=None):
    N = int(lin_rec.shape[0])
    _check(lib().xpr_lin_rasterize_fwd(C.byref(cam), C.byref(cfg), C.c_int64(N), _p(lin_rec, _F32), _p(vals_sorted, _I32),
                                       _p(tile_ranges, _I32), _p(image, _F32), _p(final_T, _F32), _p(n_contrib, _I32),
                                       _stream(stream)), "xpr_lin_rasterize_fwd")


def xpr_lin_rasterize_stats(cam: XprCamera, cfg: XprConfig, lin_rec, vals_sorted, tile_ranges, stats, stream=None):
    N = int(lin_rec.shape[0])
    _check(lib().xpr_lin_rasterize_stats(C.byref(cam), C.byref(cfg), C.c_int64(N), _p(lin_rec, _F32),
                                         _p(vals_sorted, _I32), _p(tile_ranges, _I32), _p(stats, _I64), _stream(stream)),
           "xpr_lin_rasterize_stats")


def xpr_lin_rasterize_bwd(cam: XprCamera, cfg: XprConfig, lin_rec, vals_sorted, tile_ranges, final_T, n_contrib,
                          dL_dimage, g_lin_rec, stream=None):
    N = int(lin_rec.shape[0])
    _check(lib().xpr_lin_rasterize_bwd(C.byref(cam), C.byref(cfg), C.c_int64(N), _p(lin_rec, _F32), _p(vals_sorted, _I32),
                                       _p(tile_ranges, _I32), _p(final_T, _F32), _p(n_contrib, _I32), _p(dL_dimage, _F32),
                                       _p(g_lin_rec, _F32), _stream(stream)), "xpr_lin_rasterize_bwd")


def xpr_lin_project_bwd(means, scales, quats, opacities, sh, cam: XprCamera, cfg: XprConfig, tile_count, lin_rec,
                        g_lin_rec, g_means, g_scales, g_quats, g_opacities, g_sh, stream=None):
    N = int(means.shape[0])
    _check(lib().xpr_lin_project_bwd(C.c_int64(N), _p(means, _F32), _p(scales, _F32), _p(quats, _F32), _p(opacities, _F32),
                                     _p(sh, _F32), C.byref(cam), C.byref(cfg), _p(tile_count, _I32), _p(lin_rec, _F32),
                                     _p(g_lin_rec, _F32), _p(g_means, _F32), _p(g_scales, _F32), _p(g_quats, _F32),
                                     _p(g_opacities, _F32), _p(g_sh, _F32), _stream(stream)), "xpr_lin_project_bwd")


def xpr_loss_grad(kind: str, image, target, dL_dimage, stream=None):
    """kind: "l1" (sum of absolute differences) or "l2" (sum of squares); dL/dimage in one pass (xpr.h)."""
    k = {"l1": 0, "l2": 1}[kind]
    _check(lib().xpr_loss_grad(C.c_int32(k), C.c_int64(image.numel()), _p(image, _F32), _p(target, _F32), _p(dL_dimage, _F32),
                               _stream(stream)), "xpr_loss_grad")
