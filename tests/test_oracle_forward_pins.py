"""Pins of the ORACLE's forward path against what the paper and the mathematics fix.

None of these re-type the oracle's own formulas in the oracle's own form: they use closed forms
(P1), library routines (numpy inverse, scipy spherical harmonics, numerical Jacobians), invariants
(P2, P4, P5), brute force (P3) and special cases (P7-P9).  Citations: PAPER.md L<line>.
"""
import math
import types

import numpy as np
import pytest

import xpr_oracle as xo
from paper_2606_11529_b200 import scenes

C0 = 0.28209479177387814
AT = 1.0 / 255.0


def cam_obj(model=0, W=64, H=64, fx=80.0, fy=80.0, cx=None, cy=None, w2c=None, k=(0, 0, 0, 0)):
    if w2c is None:
        w2c = np.array([[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 0]], np.float64)
    return types.SimpleNamespace(model=model, width=W, height=H, fx=fx, fy=fy, cx=W / 2 if cx is None else cx,
                                 cy=H / 2 if cy is None else cy, k=k, w2c=np.asarray(w2c, np.float64))


def cfg_dict(**kw):
    d = dict(projection=0, sh_degree=0, tile=16, antialias=0, alpha_thresh=AT, alpha_max=0.99, t_min=1e-4,
             z_near=0.2, lowpass=0.3, ut_alpha=1.0, ut_beta=2.0, ut_kappa=0.0, bg=(0.0, 0.0, 0.0))
    d.update(kw)
    return d


def one_gaussian(mu, s, q=(1, 0, 0, 0), o=0.8, rgb=(0.2, 0.5, 0.9)):
    sh = ((np.asarray(rgb, np.float64) - 0.5) / C0).reshape(1, 1, 3)
    return dict(means=np.asarray(mu, np.float64).reshape(1, 3), scales=np.asarray(s, np.float64).reshape(1, 3),
                quats=np.asarray(q, np.float64).reshape(1, 4), opacities=np.asarray([o], np.float64), sh=sh)


def rot_from_quat_lib(q):
    """Independent rotation: scipy (x,y,z,w order)."""
    from scipy.spatial.transform import Rotation
    w, x, y, z = q
    return Rotation.from_quat([x, y, z, w]).as_matrix()


# ------------------------------------------------------------------------------------------------
# P1: single Gaussian closed form (PAPER L78 G(x), L435 conic = inverse projected covariance,
#     alpha = o G_2D(px), alpha_thresh = 1/255)
# ------------------------------------------------------------------------------------------------
def test_p1_isotropic_on_axis_closed_form():
    f, z0, s, o = 80.0, 4.0, 0.25, 0.8
    rgb = np.array([0.2, 0.5, 0.9])
    cam = xo.make_camera(cam_obj(fx=f, fy=f))
    cfg = xo.make_config(cfg_dict())
    g = one_gaussian((0, 0, z0), (s, s, s), o=o, rgb=rgb)
    r = xo.render(g, cam, cfg, np.float64)
    var = (f * s / z0) ** 2 + 0.3
    p = r["proj"]
    assert p["tile_count"][0] > 0
    np.testing.assert_allclose(p["mean2d"][0], [32.0, 32.0], atol=1e-12)
    np.testing.assert_allclose(p["conic"][0], [1 / var, 0.0, 1 / var], rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(p["depth"][0], z0)
    np.testing.assert_allclose(p["rgb"][0], rgb, rtol=1e-12)
    # rectangle = tile box of radius sigma' sqrt(2 ln(255 o))
    rad = math.sqrt(var) * math.sqrt(2 * math.log(255 * o))
    exp_rect = [math.floor((32 - rad) / 16), math.floor((32 - rad) / 16), math.ceil((32 + rad) / 16), math.ceil((32 + rad) / 16)]
    assert list(p["tile_rect"][0]) == [max(0, exp_rect[0]), max(0, exp_rect[1]), min(4, exp_rect[2]), min(4, exp_rect[3])]
    # image: rgb * min(0.99, o exp(-r^2 / 2 var)) where alpha >= 1/255, else 0
    ys, xs = np.mgrid[0:64, 0:64]
    r2 = (xs + 0.5 - 32.0) ** 2 + (ys + 0.5 - 32.0) ** 2
    alpha = np.minimum(0.99, o * np.exp(-0.5 * r2 / var))
    alpha = np.where(o * np.exp(-0.5 * r2 / var) >= AT, alpha, 0.0)
    np.testing.assert_allclose(r["fwd"]["image"], alpha[..., None] * rgb, rtol=1e-11, atol=1e-14)
    np.testing.assert_allclose(r["fwd"]["final_T"], 1 - alpha, rtol=1e-12)
    assert ((r["fwd"]["n_contrib"] > 0) == (alpha > 0)).all()


def test_p1_alpha_clamp_099():
    # o G > 0.99 at the centre -> alpha = 0.99 exactly (C11, BASELINE.json:north_star)
    cam = xo.make_camera(cam_obj())
    cfg = xo.make_config(cfg_dict())
    g = one_gaussian((0.0125, 0.0125, 4.0), (0.5, 0.5, 0.5), o=0.9999, rgb=(1.0, 1.0, 1.0))  # mean2d = (32.25, 32.25)
    r = xo.render(g, cam, cfg, np.float64)
    np.testing.assert_allclose(r["fwd"]["image"][32, 32], 0.99, rtol=1e-12)
    np.testing.assert_allclose(r["fwd"]["final_T"][32, 32], 0.01, rtol=1e-10)


def test_p1_anisotropic_rotated_against_library_inverse():
    # Sigma = R S S^T R^T (L78); on the optical axis J = diag(f/z) so cov2D = (f/z)^2 Sigma[:2,:2] + 0.3 I
    f, z0 = 100.0, 5.0
    q = np.array([0.9, 0.1, -0.3, 0.2]); q /= np.linalg.norm(q)
    s = np.array([0.3, 0.1, 0.05])
    R = rot_from_quat_lib(q)
    Sigma = R @ np.diag(s ** 2) @ R.T
    cov = (f / z0) ** 2 * Sigma[:2, :2] + 0.3 * np.eye(2)
    K = np.linalg.inv(cov)
    cam = xo.make_camera(cam_obj(W=128, H=96, fx=f, fy=f))
    cfg = xo.make_config(cfg_dict())
    p = xo.project(**one_gaussian((0, 0, z0), s, q), cam=cam, cfg=cfg, dtype=np.float64)
    np.testing.assert_allclose(p["conic"][0], [K[0, 0], K[0, 1], K[1, 1]], rtol=1e-11)
    # extents: exact axis-aligned box of {alpha >= 1/255} (C7): half-widths sqrt(2 lnv cov_ii)
    lnv = math.log(0.8 * 255)
    np.testing.assert_allclose(p["lnv"][0], lnv, rtol=1e-14)
    ex, ey = math.sqrt(2 * lnv * cov[0, 0]), math.sqrt(2 * lnv * cov[1, 1])
    rect = p["tile_rect"][0]
    assert rect[0] == max(0, math.floor((64 - ex) / 16)) and rect[2] == min(8, math.ceil((64 + ex) / 16))
    assert rect[1] == max(0, math.floor((48 - ey) / 16)) and rect[3] == min(6, math.ceil((48 + ey) / 16))


def test_p1_off_axis_ewa_against_numerical_jacobian():
    # EWA (L106, L435, [59]): cov2D = J W Sigma W^T J^T with J the Jacobian of the pinhole map at the mean.
    f = 120.0
    w2c = scenes.look_at((0.3, -0.2, -3.0), (0.1, 0.0, 0.5)).astype(np.float64)
    W, t = w2c[:, :3], w2c[:, 3]
    co = cam_obj(W=160, H=128, fx=f, fy=1.1 * f, cx=75.0, cy=70.0, w2c=w2c)
    mu = np.array([0.4, 0.25, 0.8]); s = np.array([0.2, 0.07, 0.12])
    q = np.array([0.3, 0.5, -0.4, 0.7]); q /= np.linalg.norm(q)
    pin = lambda p: np.array([co.fx * p[0] / p[2] + co.cx, co.fy * p[1] / p[2] + co.cy])
    pc = W @ mu + t
    h = 1e-6
    J = np.stack([(pin(pc + h * e) - pin(pc - h * e)) / (2 * h) for e in np.eye(3)], axis=1)
    R = rot_from_quat_lib(q)
    cov = J @ W @ R @ np.diag(s ** 2) @ R.T @ W.T @ J.T + 0.3 * np.eye(2)
    K = np.linalg.inv(cov)
    p = xo.project(**one_gaussian(mu, s, q), cam=xo.make_camera(co), cfg=xo.make_config(cfg_dict()), dtype=np.float64)
    assert p["tile_count"][0] > 0 and not (p["flags"][0] & 6)
    np.testing.assert_allclose(p["mean2d"][0], pin(pc), rtol=1e-12)
    np.testing.assert_allclose(p["depth"][0], pc[2], rtol=1e-12)
    np.testing.assert_allclose(p["conic"][0], [K[0, 0], K[0, 1], K[1, 1]], rtol=1e-7)


def test_visibility_rules():
    # L262: (det>0) & (o >= alpha_thresh) & (r>0) & (tc>0) & (z > z_near); L80 "outside the view ... flagged"
    cam = xo.make_camera(cam_obj())
    cfg = xo.make_config(cfg_dict())
    base = dict(s=(0.05, 0.05, 0.05))
    vis = lambda mu, o=0.5: int(xo.project(**one_gaussian(mu, o=o, **base), cam=cam, cfg=cfg, dtype=np.float64)["tile_count"][0])
    assert vis((0, 0, 4)) > 0
    assert vis((0, 0, 0.1)) == 0          # behind z_near
    assert vis((0, 0, -4)) == 0           # behind the camera
    assert vis((10, 0, 4)) == 0           # off screen: empty rectangle
    assert vis((0, 0, 4), o=AT * 0.99) == 0   # negligible opacity
    assert vis((0, 0, 4), o=AT * 1.01) > 0
    # NaN input -> culled (C26)
    assert vis((float("nan"), 0, 4)) == 0


# ------------------------------------------------------------------------------------------------
# P2: transmittance product / opacity sum
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype,tol", [(np.float64, 1e-12), (np.float32, 2e-5)])
def test_p2_transmittance_invariants(dtype, tol):
    sc = scenes.make_scene(1)
    arr = dict(means=sc.means, scales=sc.scales, quats=sc.quats, opacities=sc.opacities,
               sh=np.full_like(sc.sh, 0.5 / C0))       # rgb == 1 for every primitive
    cam = xo.make_camera(sc.cameras[0]); cfg = xo.make_config(scenes.default_render_config(sc))
    r = xo.render(arr, cam, cfg, dtype)
    img, T = r["fwd"]["image"].astype(np.float64), r["fwd"]["final_T"].astype(np.float64)
    # sum_k alpha_k T_k + T_final = 1  ->  image = 1 - final_T with rgb = 1, bg = 0
    np.testing.assert_allclose(img, (1 - T)[..., None] * np.ones(3), atol=tol)
    assert (T <= 1).all() and (T >= 1e-4 * (1 - 1e-6)).all()     # never blends past the exit threshold (C12)
    # background: C += T bg (C13)
    cfg2 = xo.make_config(dict(scenes.default_render_config(sc), bg=(0.25, 0.5, 1.0)))
    r2 = xo.render(arr, cam, cfg2, dtype)
    np.testing.assert_allclose(r2["fwd"]["image"].astype(np.float64), img + T[..., None] * np.array([0.25, 0.5, 1.0]), atol=tol)


def test_p2_final_T_is_product_of_one_minus_alpha():
    # Recompute alpha_k for one pixel directly from the projected records with numpy and the
    # definition T_i = prod_{j<i}(1 - alpha_j) (L86).
    sc = scenes.make_scene(1)
    arr = dict(means=sc.means, scales=sc.scales, quats=sc.quats, opacities=sc.opacities, sh=sc.sh)
    cam = xo.make_camera(sc.cameras[0]); cfg = xo.make_config(scenes.default_render_config(sc))
    r = xo.render(arr, cam, cfg, np.float64)
    p, b, fwd = r["proj"], r["binned"], r["fwd"]
    rng = np.random.default_rng(0)
    for _ in range(40):
        px, py = int(rng.integers(0, 64)), int(rng.integers(0, 64))
        t = (py // 16) * 4 + px // 16
        lst = b["vals"][b["ranges"][t, 0]:b["ranges"][t, 1]]
        T, C = 1.0, np.zeros(3)
        for g in lst:
            d = np.array([px + 0.5, py + 0.5]) - p["mean2d"][g]
            A, B, Cc = p["conic"][g]
            Km = np.array([[A, B], [B, Cc]])
            power = -0.5 * d @ Km @ d
            a = p["opac_eff"][g] * math.exp(power)
            if power > 0 or a < AT:
                continue
            a = min(0.99, a)
            if T * (1 - a) < 1e-4:
                break
            C += p["rgb"][g] * a * T
            T *= (1 - a)
        np.testing.assert_allclose(fwd["final_T"][py, px], T, rtol=1e-9)
        np.testing.assert_allclose(fwd["image"][py, px], C, rtol=1e-9, atol=1e-12)


# ------------------------------------------------------------------------------------------------
# P3 + P5: brute-force binning, sort invariants
# ------------------------------------------------------------------------------------------------
def _project_scene(config, dtype=np.float32, **kw):
    sc = scenes.make_scene(config, **kw)
    cam = xo.make_camera(sc.cameras[0]); cfg = xo.make_config(scenes.default_render_config(sc))
    arr = dict(means=sc.means, scales=sc.scales, quats=sc.quats, opacities=sc.opacities, sh=sc.sh)
    return sc, arr, cam, cfg, xo.project(cam=cam, cfg=cfg, dtype=dtype, **arr)


@pytest.mark.parametrize("config,kw", [(1, {}), (2, dict(n_override=3000, image_override=(200, 136)))])
def test_p3_bruteforce_pairs_and_p5_sort_invariants(config, kw):
    sc, arr, cam, cfg, p = _project_scene(config, **kw)
    tx, ty = xo.tiles(cam, cfg)
    b = xo.bin_sort(p, cam, cfg)
    # brute force O(N T): tile t=(x,y) overlaps primitive i iff x_min <= x < x_max and y_min <= y < y_max (L147)
    pairs = []
    rect, tc = p["tile_rect"], p["tile_count"]
    for y in range(ty):
        for x in range(tx):
            hit = np.nonzero((tc > 0) & (rect[:, 0] <= x) & (x < rect[:, 2]) & (rect[:, 1] <= y) & (y < rect[:, 3]))[0]
            d = p["depth"][hit]
            order = np.lexsort((hit, d.view(np.uint32)))          # by depth bits, ties by index (C10)
            pairs.append((y * tx + x, hit[order]))
    exp_vals = np.concatenate([h for _, h in pairs]).astype(np.uint32)
    exp_tiles = np.concatenate([np.full(len(h), t) for t, h in pairs]).astype(np.uint64)
    exp_keys = (exp_tiles << np.uint64(32)) | p["depth"][exp_vals].view(np.uint32).astype(np.uint64)
    assert b["num_pairs"] == len(exp_vals) == int(tc.sum())
    np.testing.assert_array_equal(b["vals"], exp_vals)
    np.testing.assert_array_equal(b["keys"], exp_keys)
    # P5 invariants
    assert (np.diff(b["keys"].astype(np.uint64)) >= 0).all() if len(b["keys"]) > 1 else True
    starts = np.cumsum([0] + [len(h) for _, h in pairs])
    for t, (_, h) in enumerate(pairs):
        if len(h):
            assert tuple(b["ranges"][t]) == (starts[t], starts[t + 1])
        else:
            assert tuple(b["ranges"][t]) == (0, 0)
    # unsorted emission: row-major inside the rectangle (L149), multiset preserved by the sort
    keys_u, vals_u = xo.emit(p, cam, cfg)
    i = int(np.argmax(tc))
    off = int(tc[:i].astype(np.int64).sum())
    w = rect[i, 2] - rect[i, 0]
    for r_ in range(int(tc[i])):
        x, y = rect[i, 0] + r_ % w, rect[i, 1] + r_ // w
        assert int(keys_u[off + r_] >> np.uint64(32)) == y * tx + x and vals_u[off + r_] == i
    a = np.sort(np.stack([keys_u, vals_u.astype(np.uint64)], 1).view([("k", "u8"), ("v", "u8")]).ravel())
    c = np.sort(np.stack([b["keys"], b["vals"].astype(np.uint64)], 1).view([("k", "u8"), ("v", "u8")]).ravel())
    assert (a == c).all()


def test_strict_per_pixel_equals_per_tile():
    # each pixel's own depth-sorted list gives the same image as its tile's range (L84)
    sc, arr, cam, cfg, p = _project_scene(1)
    b = xo.bin_sort(p, cam, cfg)
    f = xo.rasterize_fwd(p, b, cam, cfg)
    s = xo.rasterize_fwd_strict(p, cam, cfg)
    for k in ("image", "final_T", "n_contrib"):
        np.testing.assert_array_equal(f[k], s[k])


# ------------------------------------------------------------------------------------------------
# P4: tiling invariance ("removing these entries is equivalent to keeping them with alpha=0", L683):
#     with the exact alpha >= 1/255 box (C7) the image cannot depend on the tile size.
# ------------------------------------------------------------------------------------------------
def test_p4_tiling_invariance():
    sc = scenes.make_scene(1)
    arr = dict(means=sc.means, scales=sc.scales, quats=sc.quats, opacities=sc.opacities, sh=sc.sh)
    cam = xo.make_camera(sc.cameras[0])
    d = scenes.default_render_config(sc)
    out = {}
    for ts in (8, 16, 64):
        out[ts] = xo.render(arr, cam, xo.make_config(dict(d, tile=ts)), np.float64)
    ok = (out[16]["fwd"]["fragile"] | out[8]["fwd"]["fragile"]) == 0
    assert ok.mean() > 0.99
    for ts in (8, 64):
        np.testing.assert_allclose(out[ts]["fwd"]["image"][ok], out[16]["fwd"]["image"][ok], rtol=0, atol=1e-12)
        np.testing.assert_allclose(out[ts]["fwd"]["final_T"][ok], out[16]["fwd"]["final_T"][ok], rtol=0, atol=1e-12)
    assert out[8]["binned"]["num_pairs"] > out[16]["binned"]["num_pairs"] > out[64]["binned"]["num_pairs"]


# ------------------------------------------------------------------------------------------------
# P7, P8: unscented transform
# ------------------------------------------------------------------------------------------------
def test_p7_ut_exact_for_affine_map():
    rng = np.random.default_rng(5)
    w2c = scenes.look_at((0.5, 0.2, -3.0), (0, 0, 0)).astype(np.float64)
    co = cam_obj(model=2, W=128, H=128, fx=30.0, fy=25.0, w2c=w2c)
    cam = xo.make_camera(co)
    cfg = xo.make_config(cfg_dict(projection=1, lowpass=0.0))
    Aff = np.diag([co.fx, co.fy]) @ w2c[:2, :3]
    for _ in range(5):
        mu = rng.uniform(-0.5, 0.5, 3); s = rng.uniform(0.05, 0.4, 3)
        q = rng.standard_normal(4); q /= np.linalg.norm(q)
        p = xo.project(**one_gaussian(mu, s, q), cam=cam, cfg=cfg, dtype=np.float64)
        R = rot_from_quat_lib(q)
        cov = Aff @ R @ np.diag(s ** 2) @ R.T @ Aff.T
        K = np.linalg.inv(cov)
        m = Aff @ mu + np.diag([co.fx, co.fy]) @ w2c[:2, 3] + [co.cx, co.cy]
        assert p["tile_count"][0] > 0
        np.testing.assert_allclose(p["mean2d"][0], m, rtol=1e-12)
        np.testing.assert_allclose(p["conic"][0], [K[0, 0], K[0, 1], K[1, 1]], rtol=1e-9)


def test_p8_ut_tends_to_ewa_for_small_scales():
    rng = np.random.default_rng(6)
    co = cam_obj(W=256, H=256, fx=300.0, fy=300.0)
    cam = xo.make_camera(co)
    errs = []
    for scale in (1e-2, 1e-3):
        mu = np.array([0.3, -0.2, 3.0]); s = scale * np.array([1.0, 0.5, 2.0])
        q = rng.standard_normal(4); q /= np.linalg.norm(q)
        g = one_gaussian(mu, s, q)
        pe = xo.project(**g, cam=cam, cfg=xo.make_config(cfg_dict(projection=0, lowpass=0.0)), dtype=np.float64)
        pu = xo.project(**g, cam=cam, cfg=xo.make_config(cfg_dict(projection=1, lowpass=0.0)), dtype=np.float64)
        errs.append(np.abs(pu["conic"][0] / pe["conic"][0] - 1).max())
        np.testing.assert_allclose(pu["mean2d"][0], pe["mean2d"][0], atol=50 * scale ** 2 * 300)
    assert errs[0] < 1e-3 and errs[1] < errs[0] / 30       # O(s^2) agreement


def test_ut_weights_follow_alpha_beta_kappa():
    # kappa != 0 -> lambda != 0: the centre point gets mean weight lambda/(n+lambda); the estimate of an
    # affine map must stay exact for any (alpha, beta, kappa).
    co = cam_obj(model=2, W=128, H=128, fx=30.0, fy=30.0)
    cam = xo.make_camera(co)
    g = one_gaussian((0.1, 0.2, 3.0), (0.3, 0.1, 0.2), (0.8, 0.2, 0.1, -0.5))
    ref = xo.project(**g, cam=cam, cfg=xo.make_config(cfg_dict(projection=1)), dtype=np.float64)
    alt = xo.project(**g, cam=cam, cfg=xo.make_config(cfg_dict(projection=1, ut_alpha=0.7, ut_beta=1.0, ut_kappa=1.5)), dtype=np.float64)
    np.testing.assert_allclose(alt["conic"], ref["conic"], rtol=1e-10)
    np.testing.assert_allclose(alt["mean2d"], ref["mean2d"], rtol=1e-12)


# ------------------------------------------------------------------------------------------------
# P9: fisheye-equidistant special cases (BASELINE.json:configs[3])
# ------------------------------------------------------------------------------------------------
def test_p9_fisheye_special_cases():
    f = 200.0
    cam0 = xo.make_camera(cam_obj(model=1, W=512, H=512, fx=f, fy=f))
    for th in (0.1, 0.7, 1.3):
        for phi in (0.0, 1.0, 2.5):
            p = np.array([math.sin(th) * math.cos(phi), math.sin(th) * math.sin(phi), math.cos(th)]) * 3.0
            pix = xo.camera_project(cam0, p) - 256.0
            np.testing.assert_allclose(np.hypot(*pix), f * th, rtol=1e-12)        # radius = f theta when k = 0
            np.testing.assert_allclose(math.atan2(pix[1], pix[0]), math.atan2(p[1], p[0]), atol=1e-12)
    # on-axis limit equals the pinhole
    camp = xo.make_camera(cam_obj(model=0, W=512, H=512, fx=f, fy=f))
    p = np.array([1e-9, -2e-9, 2.0])
    np.testing.assert_allclose(xo.camera_project(cam0, p), xo.camera_project(camp, p), atol=1e-9)
    np.testing.assert_allclose(xo.camera_project(cam0, np.array([0.0, 0.0, 2.0])), [256.0, 256.0])
    # distortion polynomial theta_d = theta (1 + k1 th^2 + k2 th^4 + k3 th^6 + k4 th^8)
    k = (0.03, -0.02, 0.01, 0.04)
    camk = xo.make_camera(cam_obj(model=1, W=512, H=512, fx=f, fy=f, k=k))
    th = 0.9
    p = np.array([math.sin(th), 0.0, math.cos(th)])
    thd = th * (1 + k[0] * th ** 2 + k[1] * th ** 4 + k[2] * th ** 6 + k[3] * th ** 8)
    np.testing.assert_allclose(xo.camera_project(camk, p)[0] - 256.0, f * thd, rtol=1e-12)
    # fp32 mode goes through fp64 for atan2 (R2): agrees to fp32 rounding
    np.testing.assert_allclose(xo.camera_project(camk, p.astype(np.float32), np.float32), xo.camera_project(camk, p), rtol=3e-7)


# ------------------------------------------------------------------------------------------------
# P10: spherical harmonics (reading C5) against scipy's complex harmonics and by quadrature
# ------------------------------------------------------------------------------------------------
def test_p10_sh_against_scipy_and_orthonormal():
    from scipy.special import sph_harm_y
    rng = np.random.default_rng(3)
    for _ in range(20):
        d = rng.standard_normal(3); d /= np.linalg.norm(d)
        theta, phi = math.acos(d[2]), math.atan2(d[1], d[0])
        Y = xo.sh_basis(d)
        for l in range(4):
            for m in range(-l, l + 1):
                y = sph_harm_y(l, abs(m), theta, phi)      # includes the Condon-Shortley phase
                ref = y.real if m == 0 else math.sqrt(2) * (y.real if m > 0 else y.imag)
                np.testing.assert_allclose(Y[l * l + l + m], ref, rtol=1e-10, atol=1e-13)
    # Gram matrix = I by Gauss-Legendre x uniform-phi quadrature
    xs, ws = np.polynomial.legendre.leggauss(16)
    phis = np.arange(32) * (2 * math.pi / 32)
    G = np.zeros((16, 16))
    for ct, w in zip(xs, ws):
        st = math.sqrt(1 - ct * ct)
        for ph in phis:
            Y = xo.sh_basis(np.array([st * math.cos(ph), st * math.sin(ph), ct]))
            G += w * (2 * math.pi / 32) * np.outer(Y, Y)
    np.testing.assert_allclose(G, np.eye(16), atol=1e-12)


def test_p10_degree0_colour_and_clamp():
    cam = xo.make_camera(cam_obj()); cfg = xo.make_config(cfg_dict())
    p = xo.project(**one_gaussian((0, 0, 4), (0.1,) * 3, rgb=(0.3, -0.2, 1.4)), cam=cam, cfg=cfg, dtype=np.float64)
    np.testing.assert_allclose(p["rgb"][0], [0.3, 0.0, 1.4], rtol=1e-12)     # rgb = max(0, 1/2 + c0 sh0)
    assert (p["flags"][0] >> 3) & 7 == 0b101


def test_sh_degree3_colour_matches_basis_dot():
    # view direction d = (mu - cam_pos)/|.| ; rgb = max(0, 1/2 + sum_k Y_k(d) sh_k)
    rng = np.random.default_rng(8)
    w2c = scenes.look_at((1.0, -0.5, -3.0), (0, 0, 0)).astype(np.float64)
    cam = xo.make_camera(cam_obj(W=128, H=128, fx=100, fy=100, w2c=w2c))
    cfg = xo.make_config(cfg_dict(sh_degree=3))
    mu = np.array([0.2, 0.1, 0.3])
    sh = rng.normal(0, 0.3, (1, 16, 3))
    g = dict(means=mu.reshape(1, 3), scales=np.full((1, 3), 0.1), quats=np.array([[1.0, 0, 0, 0]]), opacities=np.array([0.7]), sh=sh)
    p = xo.project(cam=cam, cfg=cfg, dtype=np.float64, **g)
    cam_pos = -w2c[:, :3].T @ w2c[:, 3]
    np.testing.assert_allclose(cam_pos, [1.0, -0.5, -3.0], atol=1e-12)
    d = (mu - cam_pos) / np.linalg.norm(mu - cam_pos)
    ref = np.maximum(0, 0.5 + xo.sh_basis(d) @ sh[0])
    np.testing.assert_allclose(p["rgb"][0], ref, rtol=1e-12)


# ------------------------------------------------------------------------------------------------
# P12: fp32 parity mode vs fp64 self-check mode (bounds the tolerance budget, R1-R3)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("config,kw", [(1, {}), (2, dict(n_override=20000, image_override=(320, 320)))])
def test_p12_fp32_vs_fp64(config, kw):
    sc = scenes.make_scene(config, **kw)
    arr = dict(means=sc.means, scales=sc.scales, quats=sc.quats, opacities=sc.opacities, sh=sc.sh)
    cam = xo.make_camera(sc.cameras[0]); cfg = xo.make_config(scenes.default_render_config(sc), fragile_rel=1e-4)
    r32 = xo.render(arr, cam, cfg, np.float32)
    r64 = xo.render(arr, cam, cfg, np.float64)
    # binning decisions agree except for a handful of boundary cases
    same = (r32["proj"]["tile_rect"] == r64["proj"]["tile_rect"]).all(axis=1)
    assert same.mean() > 0.999
    ok = (r32["fwd"]["fragile"] | r64["fwd"]["fragile"]) == 0
    assert ok.mean() > 0.9
    # the image is compared UNCONDITIONALLY: a Gaussian whose rectangle differs between the two precisions only
    # changes the lists of the tiles of either rectangle, so those tiles are left out and every other pixel counts
    ts = int(cfg.tile)
    H, W = int(cam.height), int(cam.width)
    hit = np.zeros(((H + ts - 1) // ts, (W + ts - 1) // ts), bool)
    for g in np.nonzero(~same)[0]:
        for rr in (r32["proj"]["tile_rect"][g], r64["proj"]["tile_rect"][g]):
            hit[rr[1]:rr[3], rr[0]:rr[2]] = True
    ok &= ~np.kron(hit, np.ones((ts, ts), bool))[:H, :W]
    assert ok.mean() > 0.85
    err = np.abs(r32["fwd"]["image"].astype(np.float64) - r64["fwd"]["image"])[ok]
    assert err.max() < 1e-5
    # (n_contrib is a list POSITION: two depths that round to one fp32 value may swap places between the two
    # precisions, so it is not compared here; the image and final_T are)
    assert np.abs(r32["fwd"]["final_T"].astype(np.float64) - r64["fwd"]["final_T"])[ok].max() < 1e-5


def test_golden_single_gaussian():
    """tests/golden/single_gaussian.txt (closed form written by tests/golden/make_golden.py)."""
    import os
    rows = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "single_gaussian.txt"))
    cam = xo.make_camera(cam_obj(fx=80.0, fy=80.0)); cfg = xo.make_config(cfg_dict())
    g = one_gaussian((0, 0, 4.0), (0.25,) * 3, o=0.8, rgb=(0.2, 0.5, 0.9))
    for dt, tol in ((np.float64, 1e-12), (np.float32, 1e-6)):
        r = xo.render(g, cam, cfg, dt)
        for px, py, a, cr, cg, cb in rows:
            np.testing.assert_allclose(r["fwd"]["image"][int(py), int(px)], [cr, cg, cb], atol=tol)
            np.testing.assert_allclose(1 - r["fwd"]["final_T"][int(py), int(px)], a, atol=tol)


# ------------------------------------------------------------------------------------------------
# P17: the Mip-Splatting opacity factor of `antialias` (PAPER L472-473 `o = p.o * mip_splatting_2D(det_orig, det)`,
# reading C19: rho = sqrt(max(0, det_raw / det))).  Pinned by (a) the closed form of an isotropic on-axis
# Gaussian, where cov_raw = sigma^2 I (EWA: J = f/z I on the axis; UT: the six outer sigma points sit at
# +-sqrt(3) s on the axes, so sum w_c dy dy^T = sigma^2 I as well), hence rho = sigma^2 / (sigma^2 + 0.3) and
# the pixel value is rgb * o * rho * exp(-r^2 / 2 (sigma^2 + 0.3)); (b) what the factor is FOR: the low-pass
# filter is a convolution with a unit-mass kernel, which preserves the integral of the splat over the image
# plane -- sum over pixels of alpha equals 2 pi o sqrt(det cov_raw) with the factor, and
# 2 pi o sqrt(det (cov_raw + 0.3 I)) without it.  A forward without the square root, with det / det_raw, or
# with the factor applied to anything but the opacity fails (a) and (b).
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("projection", [0, 1])
def test_p17_antialias_isotropic_on_axis_closed_form(projection):
    f, z0, s, o = 80.0, 4.0, 0.05, 0.8           # sigma^2 = 1: rho = 1 / 1.3, far from 1
    rgb = np.array([0.2, 0.5, 0.9])
    cam = xo.make_camera(cam_obj(fx=f, fy=f))
    g = one_gaussian((0, 0, z0), (s, s, s), o=o, rgb=rgb)
    r = xo.render(g, cam, xo.make_config(cfg_dict(antialias=1, projection=projection)), np.float64)
    var_raw = (f * s / z0) ** 2
    rho = var_raw / (var_raw + 0.3)
    p = r["proj"]
    assert p["tile_count"][0] > 0
    np.testing.assert_allclose(p["opac_eff"][0], o * rho, rtol=1e-11)
    np.testing.assert_allclose(p["conic"][0], [1 / (var_raw + 0.3), 0.0, 1 / (var_raw + 0.3)], rtol=1e-11, atol=1e-14)
    np.testing.assert_allclose(p["lnv"][0], math.log(255 * o * rho), rtol=1e-12)
    ys, xs = np.mgrid[0:64, 0:64]
    r2 = (xs + 0.5 - 32.0) ** 2 + (ys + 0.5 - 32.0) ** 2
    a = o * rho * np.exp(-0.5 * r2 / (var_raw + 0.3))
    a = np.where(a >= AT, a, 0.0)
    assert a.max() > 0.5
    np.testing.assert_allclose(r["fwd"]["image"], a[..., None] * rgb, rtol=1e-10, atol=1e-14)
    # without the flag the same Gaussian keeps its opacity
    r0 = xo.render(g, cam, xo.make_config(cfg_dict(antialias=0, projection=projection)), np.float64)
    np.testing.assert_allclose(r0["proj"]["opac_eff"][0], o, rtol=1e-14)


@pytest.mark.parametrize("projection", [0, 1])
def test_p17_antialias_preserves_the_integral_of_the_splat(projection):
    f, z0 = 300.0, 5.0
    q = np.array([0.9, 0.1, -0.3, 0.2]); q /= np.linalg.norm(q)
    s = np.array([0.03, 0.012, 0.012])          # raw sigmas 0.72 .. 1.8 px: the 0.3 px^2 filter matters
    o = 0.5
    R = rot_from_quat_lib(q)
    cov_raw = (f / z0) ** 2 * (R @ np.diag(s ** 2) @ R.T)[:2, :2]      # on the axis J = f/z [I | 0]
    cam = xo.make_camera(cam_obj(W=96, H=96, fx=f, fy=f))
    g = one_gaussian((0, 0, z0), s, q, o=o, rgb=(1.0, 1.0, 1.0))
    tiny = 1e-9                                                            # gate far below every visible pixel
    out = {}
    for aa in (0, 1):
        r = xo.render(g, cam, xo.make_config(cfg_dict(antialias=aa, projection=projection, alpha_thresh=tiny)), np.float64)
        assert r["proj"]["tile_count"][0] >= 4                            # the box of {alpha >= 1e-9}, inside the image
        out[aa] = float(r["fwd"]["image"][..., 0].sum())                   # rgb = 1, one Gaussian: image = alpha
    with_factor = 2 * math.pi * o * math.sqrt(np.linalg.det(cov_raw))
    without = 2 * math.pi * o * math.sqrt(np.linalg.det(cov_raw + 0.3 * np.eye(2)))
    assert without > 1.15 * with_factor                                   # the two are well apart on this case
    # pixel sums of a Gaussian with sigma >= 0.9 px (filtered) equal its integral to ~1e-6; UT differs from the linearised
    # covariance at second order in s/z
    tol = 1e-5 if projection == 0 else 2e-3
    np.testing.assert_allclose(out[1], with_factor, rtol=tol)
    np.testing.assert_allclose(out[0], without, rtol=tol)
