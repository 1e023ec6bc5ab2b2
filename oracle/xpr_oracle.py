"""ctypes binding of the CPU oracle (TEST INFRASTRUCTURE, not the product; see xpr_oracle.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from paper_2606_11529_b200 except (optionally, by the
caller) the seeded scene containers, which carry no arithmetic of the method.
"""
from __future__ import annotations

import ctypes as C
import os
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
if _HERE not in sys.path:
    sys.path.insert(0, _HERE)
import build as _build  # noqa: E402  (oracle/build.py)


class XoCamera(C.Structure):
    _fields_ = [("model", C.c_int32), ("width", C.c_int32), ("height", C.c_int32),
                ("fx", C.c_double), ("fy", C.c_double), ("cx", C.c_double), ("cy", C.c_double),
                ("k", C.c_double * 4), ("w2c", C.c_double * 12)]


class XoConfig(C.Structure):
    _fields_ = [("projection", C.c_int32), ("sh_degree", C.c_int32), ("tile", C.c_int32), ("antialias", C.c_int32),
                ("alpha_thresh", C.c_double), ("alpha_max", C.c_double), ("t_min", C.c_double),
                ("z_near", C.c_double), ("lowpass", C.c_double),
                ("ut_alpha", C.c_double), ("ut_beta", C.c_double), ("ut_kappa", C.c_double),
                ("bg", C.c_double * 3), ("fragile_rel", C.c_double), ("tile_cull", C.c_int32)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.xpr_oracle_bin_sort.restype = C.c_int64
        _lib.xpr_oracle_emit.restype = C.c_int64
        _lib.xpr_oracle_emit_cull.restype = C.c_int64
        _lib.xpr_oracle_bin_sort_cull.restype = C.c_int64
        _lib.xpr_oracle_num_threads.restype = C.c_int32
    return _lib


def num_threads() -> int:
    return int(lib().xpr_oracle_num_threads())


def make_camera(cam) -> XoCamera:
    """cam: any object with model,width,height,fx,fy,cx,cy,k,w2c (e.g. scenes.Camera)."""
    c = XoCamera()
    c.model, c.width, c.height = int(cam.model), int(cam.width), int(cam.height)
    c.fx, c.fy, c.cx, c.cy = float(cam.fx), float(cam.fy), float(cam.cx), float(cam.cy)
    for i in range(4):
        c.k[i] = float(cam.k[i])
    w = np.asarray(cam.w2c, np.float64).reshape(12)
    for i in range(12):
        c.w2c[i] = float(w[i])
    return c


def make_config(d: dict, fragile_rel: float = 2e-5) -> XoConfig:
    c = XoConfig()
    c.projection, c.sh_degree, c.tile, c.antialias = int(d["projection"]), int(d["sh_degree"]), int(d["tile"]), int(d["antialias"])
    c.alpha_thresh, c.alpha_max, c.t_min = float(d["alpha_thresh"]), float(d["alpha_max"]), float(d["t_min"])
    c.z_near, c.lowpass = float(d["z_near"]), float(d["lowpass"])
    c.ut_alpha, c.ut_beta, c.ut_kappa = float(d["ut_alpha"]), float(d["ut_beta"]), float(d["ut_kappa"])
    for i in range(3):
        c.bg[i] = float(d["bg"][i])
    c.fragile_rel = float(fragile_rel)
    c.tile_cull = int(d.get("tile_cull", 0))
    return c


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _sfx(dtype):
    return {np.dtype(np.float32): "f32", np.dtype(np.float64): "f64"}[np.dtype(dtype)]


def tiles(cam, cfg):
    ts = int(cfg.tile)
    return (int(cam.width) + ts - 1) // ts, (int(cam.height) + ts - 1) // ts


def project(means, scales, quats, opacities, sh, cam: XoCamera, cfg: XoConfig, dtype=np.float32) -> dict:
    dt = np.dtype(dtype)
    N = int(means.shape[0])
    a = [np.ascontiguousarray(x, dt) for x in (means, scales, quats, opacities, sh)]
    out = dict(mean2d=np.empty((N, 2), dt), conic=np.empty((N, 3), dt), opac_eff=np.empty(N, dt),
               rgb=np.empty((N, 3), dt), depth=np.empty(N, dt), lnv=np.empty(N, dt),
               tile_rect=np.empty((N, 4), np.int32), tile_count=np.empty(N, np.uint32), flags=np.empty(N, np.uint8))
    fn = getattr(lib(), "xpr_oracle_project_" + _sfx(dt))
    fn(C.c_int64(N), *[_p(x) for x in a], C.byref(cam), C.byref(cfg),
       *[_p(out[k]) for k in ("mean2d", "conic", "opac_eff", "rgb", "depth", "lnv", "tile_rect", "tile_count", "flags")])
    return out


def _cull_args(proj: dict):
    """tile_cull data p_tcd: mean2d, conic, lnv -- always fp32, like depth (the decision is
    taken on the fp32 projection outputs)."""
    return (np.ascontiguousarray(proj["mean2d"], np.float32), np.ascontiguousarray(proj["conic"], np.float32),
            np.ascontiguousarray(proj["lnv"], np.float32))


def tile_keep(mean2d, conic, lnv, tile_xy, ts: int, dtype=np.float32):
    """keep flags of (primitive, tile) pairs: arrays [n,2], [n,3], [n], int32 [n,2]."""
    sfx = _sfx(dtype)
    m, c, l = (np.ascontiguousarray(a, dtype) for a in (mean2d, conic, lnv))
    t = np.ascontiguousarray(tile_xy, np.int32)
    keep = np.zeros(len(l), np.uint8)
    getattr(lib(), "xpr_oracle_tile_keep_" + sfx)(C.c_int64(len(l)), _p(m), _p(c), _p(l), _p(t), C.c_int32(ts), _p(keep))
    return keep.astype(bool)


def emit(proj: dict, cam: XoCamera, cfg: XoConfig):
    tx, _ = tiles(cam, cfg)
    N = int(proj["tile_count"].shape[0])
    depth = np.ascontiguousarray(proj["depth"], np.float32)
    I = int(proj["tile_count"].astype(np.int64).sum())
    keys = np.empty(I, np.uint64)
    vals = np.empty(I, np.uint32)
    if cfg.tile_cull:
        m, c, l = _cull_args(proj)
        n = lib().xpr_oracle_emit_cull(C.c_int64(N), _p(depth), _p(proj["tile_rect"]), _p(proj["tile_count"]), _p(m),
                                       _p(c), _p(l), C.c_int32(tx), C.c_int32(cfg.tile), C.c_int64(I), _p(keys), _p(vals))
        assert n <= I
        return keys[:n], vals[:n]
    n = lib().xpr_oracle_emit(C.c_int64(N), _p(depth), _p(proj["tile_rect"]), _p(proj["tile_count"]), C.c_int32(tx),
                              C.c_int64(I), _p(keys), _p(vals))
    assert n == I
    return keys, vals


def bin_sort(proj: dict, cam: XoCamera, cfg: XoConfig) -> dict:
    tx, ty = tiles(cam, cfg)
    N = int(proj["tile_count"].shape[0])
    depth = np.ascontiguousarray(proj["depth"], np.float32)
    I = int(proj["tile_count"].astype(np.int64).sum())
    keys = np.empty(I, np.uint64)
    vals = np.empty(I, np.uint32)
    ranges = np.zeros((tx * ty, 2), np.uint32)
    if cfg.tile_cull:
        m, c, l = _cull_args(proj)
        n = lib().xpr_oracle_bin_sort_cull(C.c_int64(N), _p(depth), _p(proj["tile_rect"]), _p(proj["tile_count"]),
                                           _p(m), _p(c), _p(l), C.c_int32(tx), C.c_int32(ty), C.c_int32(cfg.tile),
                                           C.c_int64(I), _p(keys), _p(vals), _p(ranges))
        assert n <= I, (n, I)
        return dict(keys=keys[:n].copy(), vals=vals[:n].copy(), ranges=ranges, num_pairs=int(n), num_candidates=I)
    n = lib().xpr_oracle_bin_sort(C.c_int64(N), _p(depth), _p(proj["tile_rect"]), _p(proj["tile_count"]),
                                  C.c_int32(tx), C.c_int32(ty), C.c_int64(I), _p(keys), _p(vals), _p(ranges))
    assert n == I, (n, I)
    return dict(keys=keys, vals=vals, ranges=ranges, num_pairs=I, num_candidates=I)


def rasterize_fwd(proj: dict, binned: dict, cam: XoCamera, cfg: XoConfig, dtype=np.float32) -> dict:
    dt = np.dtype(dtype)
    H, W = int(cam.height), int(cam.width)
    N = int(proj["tile_count"].shape[0])
    a = [np.ascontiguousarray(proj[k], dt) for k in ("mean2d", "conic", "opac_eff", "rgb", "lnv")]
    out = dict(image=np.empty((H, W, 3), dt), final_T=np.empty((H, W), dt), n_contrib=np.empty((H, W), np.uint32),
               fragile=np.empty((H, W), np.uint8))
    counters = np.zeros(2, np.int64)
    fn = getattr(lib(), "xpr_oracle_rasterize_fwd_" + _sfx(dt))
    fn(C.byref(cam), C.byref(cfg), C.c_int64(N), *[_p(x) for x in a], _p(binned["vals"]), _p(binned["ranges"]),
       _p(out["image"]), _p(out["final_T"]), _p(out["n_contrib"]), _p(out["fragile"]), _p(counters))
    out["pp_visit"], out["pp_pass"] = int(counters[0]), int(counters[1])
    return out


def rasterize_fwd_strict(proj: dict, cam: XoCamera, cfg: XoConfig, dtype=np.float32) -> dict:
    dt = np.dtype(dtype)
    H, W = int(cam.height), int(cam.width)
    N = int(proj["tile_count"].shape[0])
    a = [np.ascontiguousarray(proj[k], dt) for k in ("mean2d", "conic", "opac_eff", "rgb", "lnv", "depth")]
    out = dict(image=np.empty((H, W, 3), dt), final_T=np.empty((H, W), dt), n_contrib=np.empty((H, W), np.uint32))
    fn = getattr(lib(), "xpr_oracle_rasterize_fwd_strict_" + _sfx(dt))
    fn(C.byref(cam), C.byref(cfg), C.c_int64(N), *[_p(x) for x in a], _p(proj["tile_rect"]), _p(proj["tile_count"]),
       _p(out["image"]), _p(out["final_T"]), _p(out["n_contrib"]))
    return out


def rasterize_bwd(proj: dict, binned: dict, fwd: dict, dL_dimage, cam: XoCamera, cfg: XoConfig, dtype=np.float32,
                  mass: bool = False, acc32: bool = False) -> dict:
    """acc32: every sum kept in fp32 (what a CPU fp32 implementation returns; only to put the GPU's summation error
    beside it)."""
    dt = np.dtype(dtype)
    N = int(proj["tile_count"].shape[0])
    a = [np.ascontiguousarray(proj[k], dt) for k in ("mean2d", "conic", "opac_eff", "rgb", "lnv")]
    dL = np.ascontiguousarray(dL_dimage, dt)
    out = dict(g_mean2d=np.empty((N, 2), np.float64), g_conic=np.empty((N, 3), np.float64),
               g_opac_eff=np.empty(N, np.float64), g_rgb=np.empty((N, 3), np.float64))
    name = "xpr_oracle_rasterize_bwd_mass_" if mass else "xpr_oracle_rasterize_bwd_acc32_" if acc32 else "xpr_oracle_rasterize_bwd_"
    fn = getattr(lib(), name + _sfx(dt))
    fn(C.byref(cam), C.byref(cfg), C.c_int64(N), *[_p(x) for x in a], _p(binned["vals"]), _p(binned["ranges"]),
       _p(np.ascontiguousarray(fwd["n_contrib"], np.uint32)), _p(dL),
       _p(out["g_mean2d"]), _p(out["g_conic"]), _p(out["g_opac_eff"]), _p(out["g_rgb"]))
    return out


def project_bwd(means, scales, quats, opacities, sh, cam: XoCamera, cfg: XoConfig, grads: dict, dtype=np.float32) -> dict:
    dt = np.dtype(dtype)
    N = int(means.shape[0])
    K = (int(cfg.sh_degree) + 1) ** 2
    a = [np.ascontiguousarray(x, dt) for x in (means, scales, quats, opacities, sh)]
    g = [np.ascontiguousarray(grads[k], np.float64) for k in ("g_mean2d", "g_conic", "g_opac_eff", "g_rgb")]
    out = dict(g_means=np.empty((N, 3), np.float64), g_scales=np.empty((N, 3), np.float64),
               g_quats=np.empty((N, 4), np.float64), g_opacities=np.empty(N, np.float64),
               g_sh=np.empty((N, K, 3), np.float64))
    fn = getattr(lib(), "xpr_oracle_project_bwd_" + _sfx(dt))
    fn(C.c_int64(N), *[_p(x) for x in a], C.byref(cam), C.byref(cfg), *[_p(x) for x in g],
       *[_p(out[k]) for k in ("g_means", "g_scales", "g_quats", "g_opacities", "g_sh")])
    return out


def sh_basis(d, dtype=np.float64):
    dt = np.dtype(dtype)
    d = np.ascontiguousarray(d, dt)
    out = np.empty(16, dt)
    getattr(lib(), "xpr_oracle_sh_basis_" + _sfx(dt))(_p(d), _p(out))
    return out


def camera_project(cam: XoCamera, p, dtype=np.float64):
    dt = np.dtype(dtype)
    p = np.ascontiguousarray(p, dt)
    out = np.empty(2, dt)
    getattr(lib(), "xpr_oracle_camera_project_" + _sfx(dt))(C.byref(cam), _p(p), _p(out))
    return out


def render(scene_arrays: dict, cam: XoCamera, cfg: XoConfig, dtype=np.float32) -> dict:
    """Full forward: project -> bin_sort -> rasterize_fwd. scene_arrays: means,scales,quats,opacities,sh."""
    s = scene_arrays
    proj = project(s["means"], s["scales"], s["quats"], s["opacities"], s["sh"], cam, cfg, dtype)
    binned = bin_sort(proj, cam, cfg)
    fwd = rasterize_fwd(proj, binned, cam, cfg, dtype)
    return dict(proj=proj, binned=binned, fwd=fwd)


def backward(scene_arrays: dict, r: dict, dL_dimage, cam: XoCamera, cfg: XoConfig, dtype=np.float32) -> dict:
    """Full backward given render() output and dL/dimage; returns parameter gradients (fp64)."""
    s = scene_arrays
    g2 = rasterize_bwd(r["proj"], r["binned"], r["fwd"], dL_dimage, cam, cfg, dtype)
    g3 = project_bwd(s["means"], s["scales"], s["quats"], s["opacities"], s["sh"], cam, cfg, g2, dtype)
    g3.update(g2)
    return g3


# ---- batch of views (Table 2): the definition is a loop over the views ------------

def render_views(scene_arrays: dict, cams: list, cfg: XoConfig, dtype=np.float32) -> list:
    """One render() per camera: a batch of views is V independent renders of the same primitives."""
    return [render(scene_arrays, cam, cfg, dtype) for cam in cams]


def backward_views(scene_arrays: dict, rs: list, dLs: list, cams: list, cfg: XoConfig, dtype=np.float32) -> dict:
    """Parameter gradients of L = sum over the views of L_v: the sum of the single-view gradients (fp64)."""
    out = None
    for r, dL, cam in zip(rs, dLs, cams):
        g = backward(scene_arrays, r, dL, cam, cfg, dtype)
        g = {k: g[k] for k in ("g_means", "g_scales", "g_quats", "g_opacities", "g_sh")}
        out = g if out is None else {k: out[k] + g[k] for k in out}
    return out


# ---- XPR-3DGUT ray evaluation (xpr_oracle_ray.inc) -------------------------------------------

def pixel_info(cam: XoCamera, dtype=np.float32):
    dt = np.dtype(dtype)
    if int(cam.model) not in (0, 1):
        raise ValueError("ray evaluation is defined for the pinhole and fisheye models only")
    rays = np.empty((int(cam.height), int(cam.width), 3), dt)
    getattr(lib(), "xpr_oracle_pixel_info_" + _sfx(dt))(C.byref(cam), _p(rays))
    return rays


def pixel_ray(cam: XoCamera, u: float, v: float, dtype=np.float64):
    dt = np.dtype(dtype)
    d = np.empty(3, dt)
    getattr(lib(), "xpr_oracle_pixel_ray_" + _sfx(dt))(C.byref(cam), C.c_double(u), C.c_double(v), _p(d))
    return d


def project_ray(means, scales, quats, tile_count, cam: XoCamera, dtype=np.float32):
    dt = np.dtype(dtype)
    N = int(means.shape[0])
    a = [np.ascontiguousarray(x, dt) for x in (means, scales, quats)]
    rec = np.empty((N, 12), dt)
    getattr(lib(), "xpr_oracle_project_ray_" + _sfx(dt))(C.c_int64(N), *[_p(x) for x in a], C.byref(cam),
                                                         _p(np.ascontiguousarray(tile_count, np.uint32)), _p(rec))
    return rec


def ray_power(rec12, d3, dtype=np.float64):
    dt = np.dtype(dtype)
    out = np.empty(3, dt)
    getattr(lib(), "xpr_oracle_ray_power_" + _sfx(dt))(_p(np.ascontiguousarray(rec12, dt)), _p(np.ascontiguousarray(d3, dt)), _p(out))
    return out


def rasterize_ray_fwd(proj: dict, binned: dict, cam: XoCamera, cfg: XoConfig, dtype=np.float32) -> dict:
    """proj additionally holds ray_rec [N,12] and pixel_rays [H,W,3]."""
    dt = np.dtype(dtype)
    H, W = int(cam.height), int(cam.width)
    N = int(proj["tile_count"].shape[0])
    a = [np.ascontiguousarray(proj[k], dt) for k in ("ray_rec", "opac_eff", "rgb", "lnv", "pixel_rays")]
    out = dict(image=np.empty((H, W, 3), dt), final_T=np.empty((H, W), dt), n_contrib=np.empty((H, W), np.uint32),
               fragile=np.empty((H, W), np.uint8))
    counters = np.zeros(2, np.int64)
    fn = getattr(lib(), "xpr_oracle_rasterize_ray_fwd_" + _sfx(dt))
    fn(C.byref(cam), C.byref(cfg), C.c_int64(N), *[_p(x) for x in a], _p(binned["vals"]), _p(binned["ranges"]),
       _p(out["image"]), _p(out["final_T"]), _p(out["n_contrib"]), _p(out["fragile"]), _p(counters))
    out["pp_visit"], out["pp_pass"] = int(counters[0]), int(counters[1])
    return out


def rasterize_ray_bwd(proj: dict, binned: dict, fwd: dict, dL_dimage, cam: XoCamera, cfg: XoConfig, dtype=np.float32,
                      mass: bool = False) -> dict:
    dt = np.dtype(dtype)
    N = int(proj["tile_count"].shape[0])
    a = [np.ascontiguousarray(proj[k], dt) for k in ("ray_rec", "opac_eff", "rgb", "lnv", "pixel_rays")]
    dL = np.ascontiguousarray(dL_dimage, dt)
    out = dict(g_ray_rec=np.empty((N, 12), np.float64), g_opac_eff=np.empty(N, np.float64),
               g_rgb=np.empty((N, 3), np.float64))
    fn = getattr(lib(), ("xpr_oracle_rasterize_ray_bwd_mass_" if mass else "xpr_oracle_rasterize_ray_bwd_") + _sfx(dt))
    fn(C.byref(cam), C.byref(cfg), C.c_int64(N), *[_p(x) for x in a], _p(binned["vals"]), _p(binned["ranges"]),
       _p(np.ascontiguousarray(fwd["n_contrib"], np.uint32)), _p(dL),
       _p(out["g_ray_rec"]), _p(out["g_opac_eff"]), _p(out["g_rgb"]))
    return out


def ray_bwd(means, scales, quats, tile_count, g_ray_rec, cam: XoCamera, dtype=np.float32) -> dict:
    dt = np.dtype(dtype)
    N = int(means.shape[0])
    a = [np.ascontiguousarray(x, dt) for x in (means, scales, quats)]
    out = dict(g_means=np.empty((N, 3), np.float64), g_scales=np.empty((N, 3), np.float64),
               g_quats=np.empty((N, 4), np.float64))
    getattr(lib(), "xpr_oracle_ray_bwd_" + _sfx(dt))(
        C.c_int64(N), *[_p(x) for x in a], C.byref(cam), _p(np.ascontiguousarray(tile_count, np.uint32)),
        _p(np.ascontiguousarray(g_ray_rec, np.float64)), *[_p(out[k]) for k in ("g_means", "g_scales", "g_quats")])
    return out


def rasterize_ray_bwd_acc(proj: dict, binned: dict, fwd: dict, dL_dimage, cam: XoCamera, cfg: XoConfig, dtype=np.float32,
                          mass: bool = False) -> dict:
    """rasterize_ray_bwd with the record gradient in the accumulator form the GPU sums (g_ray_acc [N,16]: S_c 6, D 6,
    sum dL/do_c 3, unused 1; xpr_oracle_ray.inc)."""
    dt = np.dtype(dtype)
    N = int(proj["tile_count"].shape[0])
    a = [np.ascontiguousarray(proj[k], dt) for k in ("ray_rec", "opac_eff", "rgb", "lnv", "pixel_rays")]
    dL = np.ascontiguousarray(dL_dimage, dt)
    out = dict(g_ray_acc=np.empty((N, 16), np.float64), g_opac_eff=np.empty(N, np.float64),
               g_rgb=np.empty((N, 3), np.float64))
    fn = getattr(lib(), "xpr_oracle_rasterize_ray_bwd_acc_" + _sfx(dt))
    fn(C.byref(cam), C.byref(cfg), C.c_int64(N), *[_p(x) for x in a], _p(binned["vals"]), _p(binned["ranges"]),
       _p(np.ascontiguousarray(fwd["n_contrib"], np.uint32)), _p(dL), C.c_int32(1 if mass else 0),
       _p(out["g_ray_acc"]), _p(out["g_opac_eff"]), _p(out["g_rgb"]))
    return out


def ray_bwd_acc(means, scales, quats, tile_count, g_ray_acc, cam: XoCamera, dtype=np.float32) -> dict:
    """Chain rule from the accumulators of rasterize_ray_bwd_acc to (mu, s, q)."""
    dt = np.dtype(dtype)
    N = int(means.shape[0])
    a = [np.ascontiguousarray(x, dt) for x in (means, scales, quats)]
    out = dict(g_means=np.empty((N, 3), np.float64), g_scales=np.empty((N, 3), np.float64),
               g_quats=np.empty((N, 4), np.float64))
    getattr(lib(), "xpr_oracle_ray_bwd_acc_" + _sfx(dt))(
        C.c_int64(N), *[_p(x) for x in a], C.byref(cam), _p(np.ascontiguousarray(tile_count, np.uint32)),
        _p(np.ascontiguousarray(g_ray_acc, np.float64)), *[_p(out[k]) for k in ("g_means", "g_scales", "g_quats")])
    return out


def render_ray(scene_arrays: dict, cam: XoCamera, cfg: XoConfig, dtype=np.float32) -> dict:
    """XPR-3DGUT forward (PAPER A.1.2): project (2D footprint for tiling / culling) -> shader record -> bin_sort ->
    pixel_info -> compositing with the ray evaluation."""
    s = scene_arrays
    proj = project(s["means"], s["scales"], s["quats"], s["opacities"], s["sh"], cam, cfg, dtype)
    proj["ray_rec"] = project_ray(s["means"], s["scales"], s["quats"], proj["tile_count"], cam, dtype)
    proj["pixel_rays"] = pixel_info(cam, dtype)
    binned = bin_sort(proj, cam, cfg)
    fwd = rasterize_ray_fwd(proj, binned, cam, cfg, dtype)
    return dict(proj=proj, binned=binned, fwd=fwd)


def backward_ray(scene_arrays: dict, r: dict, dL_dimage, cam: XoCamera, cfg: XoConfig, dtype=np.float32) -> dict:
    """Backward of render_ray: the 2D footprint only tiles (no gradient through mean2d / conic); the opacity
    factor (C19) and the colour go through project_bwd, the record through ray_bwd."""
    s = scene_arrays
    g2 = rasterize_ray_bwd(r["proj"], r["binned"], r["fwd"], dL_dimage, cam, cfg, dtype)
    N = int(s["means"].shape[0])
    gz = dict(g_mean2d=np.zeros((N, 2)), g_conic=np.zeros((N, 3)), g_opac_eff=g2["g_opac_eff"], g_rgb=g2["g_rgb"])
    g3 = project_bwd(s["means"], s["scales"], s["quats"], s["opacities"], s["sh"], cam, cfg, gz, dtype)
    gr = ray_bwd(s["means"], s["scales"], s["quats"], r["proj"]["tile_count"], g2["g_ray_rec"], cam, dtype)
    for k in ("g_means", "g_scales", "g_quats"):
        g3[k] = g3[k] + gr[k]
    g3.update(g2)
    g3["ray_part"] = gr
    return g3


# ---- Rendered depth and accumulated opacity (xpr_oracle_feat.inc, reading C31) ---------------

def rasterize_fwd_da(proj: dict, binned: dict, cam: XoCamera, cfg: XoConfig, dtype=np.float32) -> dict:
    """depth image D = sum_k z_k alpha_k T_k and accumulated opacity A = sum_k alpha_k T_k, [H,W] each."""
    dt = np.dtype(dtype)
    H, W = int(cam.height), int(cam.width)
    N = int(proj["tile_count"].shape[0])
    a = [np.ascontiguousarray(proj[k], dt) for k in ("mean2d", "conic", "opac_eff", "rgb", "lnv", "depth")]
    out = dict(depth_img=np.empty((H, W), dt), alpha_img=np.empty((H, W), dt))
    fn = getattr(lib(), "xpr_oracle_rasterize_fwd_da_" + _sfx(dt))
    fn(C.byref(cam), C.byref(cfg), C.c_int64(N), *[_p(x) for x in a], _p(binned["vals"]), _p(binned["ranges"]),
       _p(out["depth_img"]), _p(out["alpha_img"]))
    return out


def rasterize_bwd_da(proj: dict, binned: dict, fwd: dict, dL_dimage, dL_ddepth, dL_dalpha, cam: XoCamera,
                     cfg: XoConfig, dtype=np.float32, mass: bool = False) -> dict:
    dt = np.dtype(dtype)
    N = int(proj["tile_count"].shape[0])
    a = [np.ascontiguousarray(proj[k], dt) for k in ("mean2d", "conic", "opac_eff", "rgb", "lnv", "depth")]
    d = [np.ascontiguousarray(x, dt) for x in (dL_dimage, dL_ddepth, dL_dalpha)]
    out = dict(g_mean2d=np.empty((N, 2), np.float64), g_conic=np.empty((N, 3), np.float64),
               g_opac_eff=np.empty(N, np.float64), g_rgb=np.empty((N, 3), np.float64), g_depth=np.empty(N, np.float64))
    fn = getattr(lib(), ("xpr_oracle_rasterize_bwd_da_mass_" if mass else "xpr_oracle_rasterize_bwd_da_") + _sfx(dt))
    fn(C.byref(cam), C.byref(cfg), C.c_int64(N), *[_p(x) for x in a], _p(binned["vals"]), _p(binned["ranges"]),
       _p(np.ascontiguousarray(fwd["n_contrib"], np.uint32)), *[_p(x) for x in d],
       *[_p(out[k]) for k in ("g_mean2d", "g_conic", "g_opac_eff", "g_rgb", "g_depth")])
    return out


def rasterize_fwd_featn(proj: dict, binned: dict, feat, cam: XoCamera, cfg: XoConfig, dtype=np.float32):
    """N-channel feature image [H,W,C] = sum_k feat[g_k,:] alpha_k T_k (no background); feat [N,C]."""
    dt = np.dtype(dtype)
    H, W = int(cam.height), int(cam.width)
    N = int(proj["tile_count"].shape[0])
    f = np.ascontiguousarray(feat, dt).reshape(N, -1)
    Cn = int(f.shape[1])
    a = [np.ascontiguousarray(proj[k], dt) for k in ("mean2d", "conic", "opac_eff", "rgb", "lnv")]
    out = np.empty((H, W, Cn), dt)
    fn = getattr(lib(), "xpr_oracle_rasterize_fwd_featn_" + _sfx(dt))
    fn(C.byref(cam), C.byref(cfg), C.c_int64(N), *[_p(x) for x in a], _p(f), C.c_int32(Cn), _p(binned["vals"]),
       _p(binned["ranges"]), _p(out))
    return out


def rasterize_bwd_featn(proj: dict, binned: dict, fwd: dict, feat, dL_dfeat, cam: XoCamera, cfg: XoConfig,
                        dtype=np.float32) -> dict:
    """The feature part of the compositing gradients (fp64) for dL/dfeat_img [H,W,C] alone, plus g_feat [N,C]."""
    dt = np.dtype(dtype)
    N = int(proj["tile_count"].shape[0])
    f = np.ascontiguousarray(feat, dt).reshape(N, -1)
    Cn = int(f.shape[1])
    a = [np.ascontiguousarray(proj[k], dt) for k in ("mean2d", "conic", "opac_eff", "rgb", "lnv")]
    d = np.ascontiguousarray(dL_dfeat, dt)
    out = dict(g_mean2d=np.empty((N, 2), np.float64), g_conic=np.empty((N, 3), np.float64),
               g_opac_eff=np.empty(N, np.float64), g_feat=np.empty((N, Cn), np.float64))
    fn = getattr(lib(), "xpr_oracle_rasterize_bwd_featn_" + _sfx(dt))
    fn(C.byref(cam), C.byref(cfg), C.c_int64(N), *[_p(x) for x in a], _p(f), C.c_int32(Cn), _p(binned["vals"]),
       _p(binned["ranges"]), _p(np.ascontiguousarray(fwd["n_contrib"], np.uint32)), _p(d),
       *[_p(out[k]) for k in ("g_mean2d", "g_conic", "g_opac_eff", "g_feat")])
    return out


def depth_bwd(tile_count, g_depth, cam: XoCamera):
    N = int(tile_count.shape[0])
    g = np.ascontiguousarray(g_depth, np.float64)
    out = np.empty((N, 3), np.float64)
    lib().xpr_oracle_depth_bwd(C.c_int64(N), C.byref(cam), _p(np.ascontiguousarray(tile_count, np.uint32)), _p(g), _p(out))
    return out


def render_da(scene_arrays: dict, cam: XoCamera, cfg: XoConfig, dtype=np.float32) -> dict:
    """render() plus the depth image and the accumulated opacity (fwd["depth_img"], fwd["alpha_img"])."""
    r = render(scene_arrays, cam, cfg, dtype)
    r["fwd"].update(rasterize_fwd_da(r["proj"], r["binned"], cam, cfg, dtype))
    return r


def backward_da(scene_arrays: dict, r: dict, dL_dimage, dL_ddepth, dL_dalpha, cam: XoCamera, cfg: XoConfig,
                dtype=np.float32) -> dict:
    """Backward of render_da: parameter gradients (fp64) of a loss with dL/dimage, dL/dD, dL/dA."""
    s = scene_arrays
    g2 = rasterize_bwd_da(r["proj"], r["binned"], r["fwd"], dL_dimage, dL_ddepth, dL_dalpha, cam, cfg, dtype)
    g3 = project_bwd(s["means"], s["scales"], s["quats"], s["opacities"], s["sh"], cam, cfg, g2, dtype)
    g3["g_means"] = g3["g_means"] + depth_bwd(r["proj"]["tile_count"], g2["g_depth"], cam)
    g3.update(g2)
    return g3


# ---- XPR-LinPrim (xpr_oracle_lin.inc; PAPER A.1.3 L506-697) ----------------------------------------

def lin_project(means, scales, quats, opacities, sh, cam: XoCamera, cfg: XoConfig, dtype=np.float32) -> dict:
    """lin_rec [N,20] = (mu2D 2, sigma, depth | (kx, ky, h) of the four slab pairs | rgb, 0); depth = |p|."""
    dt = np.dtype(dtype)
    N = int(means.shape[0])
    a = [np.ascontiguousarray(x, dt) for x in (means, scales, quats, opacities, sh)]
    out = dict(lin_rec=np.empty((N, 20), dt), depth=np.empty(N, dt), tile_rect=np.empty((N, 4), np.int32),
               tile_count=np.empty(N, np.uint32))
    getattr(lib(), "xpr_oracle_lin_project_" + _sfx(dt))(
        C.c_int64(N), *[_p(x) for x in a], C.byref(cam), C.byref(cfg), _p(out["lin_rec"]), _p(out["depth"]),
        _p(out["tile_rect"]), _p(out["tile_count"]))
    return out


def lin_chord(rec20, pix_xy, dtype=np.float64):
    """sigma * (tau_exit - tau_enter) of one primitive at pixel-centre positions pix_xy [n,2] (0 where the ray misses)."""
    dt = np.dtype(dtype)
    r = np.ascontiguousarray(rec20, dt)
    p = np.ascontiguousarray(pix_xy, dt).reshape(-1, 2)
    out = np.empty(len(p), dt)
    getattr(lib(), "xpr_oracle_lin_chord_" + _sfx(dt))(_p(r), C.c_int64(len(p)), _p(p), _p(out))
    return out


def lin_tile_keep(rec20, tile_xy, cfg: XoConfig, dtype=np.float32):
    dt = np.dtype(dtype)
    r = np.ascontiguousarray(rec20, dt)
    t = np.ascontiguousarray(tile_xy, np.int32).reshape(-1, 2)
    keep = np.zeros(len(t), np.uint8)
    getattr(lib(), "xpr_oracle_lin_tile_keep_" + _sfx(dt))(_p(r), C.c_int64(len(t)), _p(t), C.c_int32(cfg.tile), C.byref(cfg), _p(keep))
    return keep.astype(bool)


def lin_bin_sort(proj: dict, cam: XoCamera, cfg: XoConfig) -> dict:
    lib().xpr_oracle_lin_bin_sort.restype = C.c_int64
    tx, ty = tiles(cam, cfg)
    N = int(proj["tile_count"].shape[0])
    depth = np.ascontiguousarray(proj["depth"], np.float32)
    rec = np.ascontiguousarray(proj["lin_rec"], np.float32)
    I = int(proj["tile_count"].astype(np.int64).sum())
    keys, vals = np.empty(I, np.uint64), np.empty(I, np.uint32)
    ranges = np.zeros((tx * ty, 2), np.uint32)
    n = lib().xpr_oracle_lin_bin_sort(C.c_int64(N), _p(depth), _p(proj["tile_rect"]), _p(proj["tile_count"]), _p(rec),
                                      C.byref(cfg), C.c_int32(tx), C.c_int32(ty), C.c_int32(int(cfg.tile_cull)),
                                      C.c_int64(I), _p(keys), _p(vals), _p(ranges))
    assert n <= I
    return dict(keys=keys[:n].copy(), vals=vals[:n].copy(), ranges=ranges, num_pairs=int(n), num_candidates=I)


def lin_rasterize_fwd(proj: dict, binned: dict, cam: XoCamera, cfg: XoConfig, dtype=np.float32) -> dict:
    dt = np.dtype(dtype)
    H, W = int(cam.height), int(cam.width)
    N = int(proj["tile_count"].shape[0])
    rec = np.ascontiguousarray(proj["lin_rec"], dt)
    out = dict(image=np.empty((H, W, 3), dt), final_T=np.empty((H, W), dt), n_contrib=np.empty((H, W), np.uint32),
               fragile=np.empty((H, W), np.uint8))
    counters = np.zeros(2, np.int64)
    getattr(lib(), "xpr_oracle_lin_rasterize_fwd_" + _sfx(dt))(
        C.byref(cam), C.byref(cfg), C.c_int64(N), _p(rec), _p(binned["vals"]), _p(binned["ranges"]), _p(out["image"]),
        _p(out["final_T"]), _p(out["n_contrib"]), _p(out["fragile"]), _p(counters))
    out["pp_visit"], out["pp_pass"] = int(counters[0]), int(counters[1])
    return out


def render_lin(scene_arrays: dict, cam: XoCamera, cfg: XoConfig, dtype=np.float32) -> dict:
    """XPR-LinPrim forward: project -> bin_sort (Eq. 2 cull when cfg.tile_cull) -> compositing with Beer-Lambert alpha."""
    s = scene_arrays
    proj = lin_project(s["means"], s["scales"], s["quats"], s["opacities"], s["sh"], cam, cfg, dtype)
    binned = lin_bin_sort(proj, cam, cfg)
    fwd = lin_rasterize_fwd(proj, binned, cam, cfg, dtype)
    return dict(proj=proj, binned=binned, fwd=fwd)


def lin_rasterize_bwd(proj: dict, binned: dict, fwd: dict, dL_dimage, cam: XoCamera, cfg: XoConfig, dtype=np.float32,
                      mass: bool = False) -> np.ndarray:
    """dL/d(lin_rec) [N,20] (fp64) in the layout of the record; mass=True: sum of |addend| per element."""
    dt = np.dtype(dtype)
    N = int(proj["tile_count"].shape[0])
    rec = np.ascontiguousarray(proj["lin_rec"], dt)
    dL = np.ascontiguousarray(dL_dimage, dt)
    g = np.empty((N, 20), np.float64)
    getattr(lib(), "xpr_oracle_lin_rasterize_bwd_" + _sfx(dt))(
        C.byref(cam), C.byref(cfg), C.c_int64(N), _p(rec), _p(binned["vals"]), _p(binned["ranges"]),
        _p(np.ascontiguousarray(fwd["n_contrib"], np.uint32)), _p(dL), C.c_int32(1 if mass else 0), _p(g))
    return g


def lin_project_bwd(means, scales, quats, opacities, sh, cam: XoCamera, cfg: XoConfig, g_lin_rec, dtype=np.float32) -> dict:
    dt = np.dtype(dtype)
    N = int(means.shape[0])
    K = (int(cfg.sh_degree) + 1) ** 2
    a = [np.ascontiguousarray(x, dt) for x in (means, scales, quats, opacities, sh)]
    out = dict(g_means=np.empty((N, 3), np.float64), g_scales=np.empty((N, 3), np.float64),
               g_quats=np.empty((N, 4), np.float64), g_opacities=np.empty(N, np.float64),
               g_sh=np.empty((N, K, 3), np.float64))
    getattr(lib(), "xpr_oracle_lin_project_bwd_" + _sfx(dt))(
        C.c_int64(N), *[_p(x) for x in a], C.byref(cam), C.byref(cfg), _p(np.ascontiguousarray(g_lin_rec, np.float64)),
        *[_p(out[k]) for k in ("g_means", "g_scales", "g_quats", "g_opacities", "g_sh")])
    return out


def backward_lin(scene_arrays: dict, r: dict, dL_dimage, cam: XoCamera, cfg: XoConfig, dtype=np.float32) -> dict:
    """Full LinPrim backward given render_lin() output and dL/dimage; parameter gradients (fp64) + g_lin_rec."""
    s = scene_arrays
    g2 = lin_rasterize_bwd(r["proj"], r["binned"], r["fwd"], dL_dimage, cam, cfg, dtype)
    g3 = lin_project_bwd(s["means"], s["scales"], s["quats"], s["opacities"], s["sh"], cam, cfg, g2, dtype)
    g3["g_lin_rec"] = g2
    return g3


# ---- rendered depth / accumulated opacity with the ray evaluation (f3 x f2; reading C31) ---------------------------

def rasterize_ray_fwd_da(proj: dict, binned: dict, cam: XoCamera, cfg: XoConfig, dtype=np.float32) -> dict:
    dt = np.dtype(dtype)
    H, W = int(cam.height), int(cam.width)
    N = int(proj["tile_count"].shape[0])
    a = [np.ascontiguousarray(proj[k], dt) for k in ("ray_rec", "opac_eff", "rgb", "lnv", "depth", "pixel_rays")]
    out = dict(depth_img=np.empty((H, W), dt), alpha_img=np.empty((H, W), dt))
    getattr(lib(), "xpr_oracle_rasterize_ray_fwd_da_" + _sfx(dt))(
        C.byref(cam), C.byref(cfg), C.c_int64(N), *[_p(x) for x in a], _p(binned["vals"]), _p(binned["ranges"]),
        _p(out["depth_img"]), _p(out["alpha_img"]))
    return out


def rasterize_ray_bwd_da(proj: dict, binned: dict, fwd: dict, dL_dimage, dL_ddepth, dL_dalpha, cam: XoCamera,
                         cfg: XoConfig, dtype=np.float32, acc: bool = False, mass: bool = False) -> dict:
    """rasterize_ray_bwd for a loss that also depends on the depth image and the accumulated opacity; acc=True returns the
    record gradient in the accumulator form (g_ray_acc [N,16]) instead of g_ray_rec [N,12]."""
    dt = np.dtype(dtype)
    N = int(proj["tile_count"].shape[0])
    a = [np.ascontiguousarray(proj[k], dt) for k in ("ray_rec", "opac_eff", "rgb", "lnv", "depth", "pixel_rays")]
    g = [np.ascontiguousarray(x, dt) for x in (dL_dimage, dL_ddepth, dL_dalpha)]
    key = "g_ray_acc" if acc else "g_ray_rec"
    out = {key: np.empty((N, 16 if acc else 12), np.float64), "g_opac_eff": np.empty(N, np.float64),
           "g_rgb": np.empty((N, 3), np.float64), "g_depth": np.empty(N, np.float64)}
    getattr(lib(), "xpr_oracle_rasterize_ray_bwd_da_" + _sfx(dt))(
        C.byref(cam), C.byref(cfg), C.c_int64(N), *[_p(x) for x in a], _p(binned["vals"]), _p(binned["ranges"]),
        _p(np.ascontiguousarray(fwd["n_contrib"], np.uint32)), *[_p(x) for x in g],
        C.c_int32((1 if acc else 0) | (2 if mass else 0)), _p(out[key]), _p(out["g_opac_eff"]), _p(out["g_rgb"]),
        _p(out["g_depth"]))
    return out


def render_ray_da(scene_arrays: dict, cam: XoCamera, cfg: XoConfig, dtype=np.float32) -> dict:
    r = render_ray(scene_arrays, cam, cfg, dtype)
    r["fwd"].update(rasterize_ray_fwd_da(r["proj"], r["binned"], cam, cfg, dtype))
    return r


def backward_ray_da(scene_arrays: dict, r: dict, dL_dimage, dL_ddepth, dL_dalpha, cam: XoCamera, cfg: XoConfig,
                    dtype=np.float32) -> dict:
    """Backward of render_ray_da (backward_ray + the depth's own path z = (W mu + t)_z)."""
    s = scene_arrays
    g2 = rasterize_ray_bwd_da(r["proj"], r["binned"], r["fwd"], dL_dimage, dL_ddepth, dL_dalpha, cam, cfg, dtype)
    N = int(s["means"].shape[0])
    gz = dict(g_mean2d=np.zeros((N, 2)), g_conic=np.zeros((N, 3)), g_opac_eff=g2["g_opac_eff"], g_rgb=g2["g_rgb"])
    g3 = project_bwd(s["means"], s["scales"], s["quats"], s["opacities"], s["sh"], cam, cfg, gz, dtype)
    gr = ray_bwd(s["means"], s["scales"], s["quats"], r["proj"]["tile_count"], g2["g_ray_rec"], cam, dtype)
    for k in ("g_means", "g_scales", "g_quats"):
        g3[k] = g3[k] + gr[k]
    g3["g_means"] = g3["g_means"] + depth_bwd(r["proj"]["tile_count"], g2["g_depth"], cam)
    g3.update(g2)
    return g3
