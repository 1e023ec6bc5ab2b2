"""Seeded synthetic scenes, cameras and target images (BASELINE.json:configs).

This module is the ONLY code shared by the CUDA path and the CPU oracle.  It draws random
inputs and assembles camera matrices; it contains none of the method's arithmetic
(no projection, no SH evaluation, no binning, no compositing) and imports neither the
binding nor anything under ``oracle/``.

The paper measures on Mip-NeRF360 / Tanks&Temples / Blender scenes with trained models
(PAPER.md L207-209); none of that is available, so these synthetic scenes stand in for
them (object-scale ~ Blender, unbounded ~ 360/T&T).  Recipe:
numpy ``default_rng(seed)``, fp64 draws cast to fp32, draw order means -> log-scales ->
quats -> opacity logits -> SH DC -> SH rest; scene seed 1000+i, target seed 2000+i,
camera seed 3000+i for config i = 1..5.  "N(a, b)": b is a standard deviation.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

SH_C0 = 0.28209479177387814  # 1/(2 sqrt(pi)); only used to turn an RGB draw into a DC coefficient


@dataclasses.dataclass
class Camera:
    """Plain container; every float is already rounded to fp32 (stored as Python float)."""
    model: int            # 0 pinhole, 1 fisheye-equidistant
    width: int
    height: int
    fx: float
    fy: float
    cx: float
    cy: float
    k: tuple              # fisheye k1..k4
    w2c: np.ndarray       # [3,4] fp32 row-major [W|t], x_cam = W x_world + t


@dataclasses.dataclass
class Scene:
    name: str
    means: np.ndarray     # [N,3] fp32
    scales: np.ndarray    # [N,3] fp32, activated (positive)
    quats: np.ndarray     # [N,4] fp32 (w,x,y,z), normalised in fp64 before the cast
    opacities: np.ndarray # [N]   fp32 in (0,1)
    sh: np.ndarray        # [N,K,3] fp32
    sh_degree: int
    cameras: list         # list[Camera]
    projection: int       # 0 EWA, 1 UT
    antialias: int
    loss: str             # "l2" (sum of squares) or "l1" (sum of abs)
    target_seed: int

    @property
    def N(self) -> int:
        return int(self.means.shape[0])

    def target(self, view: int = 0) -> np.ndarray:
        """Seeded uniform[0,1] target image [H,W,3] fp32 (one stream per view)."""
        cam = self.cameras[view]
        rng = np.random.default_rng(self.target_seed + 100 * view)
        return rng.random((cam.height, cam.width, 3)).astype(np.float32)


def _f32(x) -> float:
    return float(np.float32(x))


def look_at(eye, target, up=(0.0, 1.0, 0.0)) -> np.ndarray:
    """[3,4] fp32 world-to-camera, +z forward, x right, y down (f,r,u rows)."""
    eye = np.asarray(eye, np.float64)
    f = np.asarray(target, np.float64) - eye
    f = f / np.linalg.norm(f)
    r = np.cross(np.asarray(up, np.float64), f)
    r = r / np.linalg.norm(r)
    u = np.cross(f, r)
    W = np.stack([r, u, f])
    t = -W @ eye
    return np.concatenate([W, t[:, None]], axis=1).astype(np.float32)


def make_camera(model, width, height, fx, fy, cx, cy, w2c, k=(0.0, 0.0, 0.0, 0.0)) -> Camera:
    return Camera(int(model), int(width), int(height), _f32(fx), _f32(fy), _f32(cx), _f32(cy),
                  tuple(_f32(v) for v in k), np.ascontiguousarray(w2c, np.float32))


def _unit_dirs(rng, n):
    v = rng.standard_normal((n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


def _sigmoid(x):
    return 1.0 / (1.0 + np.exp(-x))


def _common(rng, n, means, ls_mu, ls_sd, op_sd, K):
    """Draw order after means: log-scales -> quats -> opacity logits -> SH DC -> SH rest."""
    log_s = rng.normal(ls_mu, ls_sd, (n, 3))
    q = rng.standard_normal((n, 4))
    q = q / np.linalg.norm(q, axis=1, keepdims=True)
    logit = rng.normal(0.0, op_sd, n)
    return (means.astype(np.float32), np.exp(log_s).astype(np.float32), q.astype(np.float32),
            _sigmoid(logit).astype(np.float32))


def _sh16(rng, n):
    dc = rng.normal(0.0, 0.3, (n, 1, 3))
    rest = rng.normal(0.0, 0.05, (n, 15, 3))
    return np.concatenate([dc, rest], axis=1).astype(np.float32)


def _blob_shell_means(rng, n):
    n_blob = int(round(0.8 * n))
    blob = rng.normal(0.0, 2.0, (n_blob, 3))
    rad = rng.uniform(20.0, 50.0, (n - n_blob, 1))
    shell = rad * _unit_dirs(rng, n - n_blob)
    return np.concatenate([blob, shell], axis=0)


def _yaw(deg):
    a = math.radians(deg)
    return np.array([[math.cos(a), 0.0, math.sin(a)], [0.0, 1.0, 0.0], [-math.sin(a), 0.0, math.cos(a)]])


def make_scene(config: int, n_override: int | None = None, image_override: tuple | None = None) -> Scene:
    """config = 1..5 (BASELINE.json:configs[config-1]).

    ``n_override`` shrinks the Gaussian count and ``image_override=(W,H)`` the image (focal
    length scaled with W so the field of view is kept) for parity cases the oracle finishes in
    seconds; the distributions are unchanged.
    """
    i = config
    rng = np.random.default_rng(1000 + i)
    crng = np.random.default_rng(3000 + i)
    if i == 1:
        n = n_override or 1000
        means = rng.uniform(-1.0, 1.0, (n, 3))
        m, s, q, o = _common(rng, n, means, -3.0, 0.5, 1.0, 1)
        rgb = rng.uniform(0.0, 1.0, (n, 1, 3))
        sh = ((rgb - 0.5) / SH_C0).astype(np.float32)
        W, H = image_override or (64, 64)
        f = 80.0 * W / 64.0
        w2c = np.array([[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 4]], np.float32)
        cams = [make_camera(0, W, H, f, f, W / 2.0, H / 2.0, w2c)]
        return Scene("config1-tiny", m, s, q, o, sh, 0, cams, 0, 0, "l2", 2000 + i)
    if i == 2:
        n = n_override or 100_000
        rad = rng.uniform(0.3, 1.0, (n, 1))
        means = rad * _unit_dirs(rng, n)
        m, s, q, o = _common(rng, n, means, -4.5, 0.6, 1.5, 16)
        sh = _sh16(rng, n)
        W, H = image_override or (800, 800)
        f = (W / 2.0) / math.tan(math.radians(20.0))
        eye = 4.0 * _unit_dirs(crng, 1)[0]
        cams = [make_camera(0, W, H, f, f, W / 2.0, H / 2.0, look_at(eye, (0, 0, 0)))]
        return Scene("config2-object", m, s, q, o, sh, 3, cams, 0, 0, "l1", 2000 + i)
    if i in (3, 4):
        # config 4 reuses the scene of config 3 (same scene seed) with a different camera model.
        rng = np.random.default_rng(1000 + 3)
        n = n_override or 1_000_000
        means = _blob_shell_means(rng, n)
        m, s, q, o = _common(rng, n, means, -4.0, 0.8, 1.5, 16)
        sh = _sh16(rng, n)
        W, H = image_override or (1920, 1080)
        f = 1100.0 * W / 1920.0
        poseA = np.array([[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 0]], np.float32)
        poseB = look_at((1.0, 0.5, -1.5), (0.0, 0.0, 0.5))
        if i == 3:
            cams = [make_camera(0, W, H, f, f, W / 2.0, H / 2.0, p) for p in (poseA, poseB)]
            return Scene("config3-unbounded", m, s, q, o, sh, 3, cams, 0, 0, "l1", 2000 + i)
        k = tuple(crng.uniform(-0.05, 0.05, 4))
        cams = [make_camera(1, W, H, f, f, W / 2.0, H / 2.0, p, k) for p in (poseA, poseB)]
        return Scene("config4-3dgut-fisheye", m, s, q, o, sh, 3, cams, 1, 1, "l1", 2000 + i)
    if i == 5:
        n = n_override or 3_000_000
        means = _blob_shell_means(rng, n)
        m, s, q, o = _common(rng, n, means, -3.0, 0.8, 1.5, 16)
        sh = _sh16(rng, n)
        W, H = image_override or (1920, 1080)
        f = 1100.0 * W / 1920.0
        cams = []
        eyes = crng.normal(0.0, 0.5, (4, 3))
        for v, deg in enumerate((0.0, 90.0, 180.0, 270.0)):
            Wm = _yaw(deg).T  # camera looks along the yawed +z axis
            t = -Wm @ eyes[v]
            w2c = np.concatenate([Wm, t[:, None]], axis=1).astype(np.float32)
            cams.append(make_camera(0, W, H, f, f, W / 2.0, H / 2.0, w2c))
        return Scene("config5-stress", m, s, q, o, sh, 3, cams, 0, 0, "l1", 2000 + i)
    raise ValueError(f"unknown config {config}")


def default_render_config(scene: Scene) -> dict:
    """Renderer constants; fp32-rounded values as Python floats."""
    return dict(projection=scene.projection, sh_degree=scene.sh_degree, tile=16, antialias=scene.antialias,
                alpha_thresh=_f32(1.0 / 255.0), alpha_max=_f32(0.99), t_min=_f32(1e-4), z_near=_f32(0.2),
                lowpass=_f32(0.3), ut_alpha=1.0, ut_beta=2.0, ut_kappa=0.0, bg=(0.0, 0.0, 0.0), tile_cull=0, ray_eval=0, tile_order=-1)


def loss_and_grad(kind: str, image: np.ndarray, target: np.ndarray):
    """Loss value (fp64) and dL/dimage (fp32). Sums, not means. Lives outside the library."""
    diff = image.astype(np.float64) - target.astype(np.float64)
    if kind == "l2":
        return float((diff * diff).sum()), (2.0 * diff).astype(np.float32)
    if kind == "l1":
        return float(np.abs(diff).sum()), np.sign(diff).astype(np.float32)
    raise ValueError(kind)
