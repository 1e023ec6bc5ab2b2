"""Pin P15 of the ORACLE's rendered depth / accumulated opacity (Table 2; reading
C31: D = sum_k z_k alpha_k T_k, A = sum_k alpha_k T_k, no background).  The pins use what is already fixed:
the pinned colour pass (a feature is a colour channel), the transmittance identity A = 1 - T_final, a constant-depth
plane, and central finite differences in fp64 of the oracle's own *forward* for the hand-derived backward.
"""
import numpy as np
import pytest

import xpr_oracle as xo
from paper_2606_11529_b200 import scenes
from test_oracle_backward_pins import cam_obj, cfg_dict, draw_scene

PARAMS = ("means", "scales", "quats", "opacities", "sh")
NAMES = dict(means="g_means", scales="g_scales", quats="g_quats", opacities="g_opacities", sh="g_sh")


def _scene(seed, n=60, K=4, **kw):
    w2c = scenes.look_at((0.2, -0.1, -1.0), (0.0, 0.05, 3.0)).astype(np.float64)
    co = cam_obj(w2c=w2c, W=48, H=40, cx=23.0, cy=20.5)
    return draw_scene(seed, n, K, **kw), co


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_p15_depth_and_alpha_are_colour_channels(dtype):
    # a feature blended with the colour's weights IS a colour channel of the pinned pass (bit for bit: same
    # arithmetic, same order) once rgb := (z, 1, 2 z) and bg = 0
    arr, co = _scene(7, opac_boost=1.0)
    cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=1, bg=(0.3, 0.6, 0.9)))
    r = xo.render_da(arr, cam, cfg, dtype)
    assert (r["fwd"]["n_contrib"] > 3).any()
    p2 = dict(r["proj"])
    z = r["proj"]["depth"]
    p2["rgb"] = np.stack([z, np.ones_like(z), 2 * z], 1).astype(dtype)
    cfg0 = xo.make_config(cfg_dict(sh_degree=1, bg=(0.0, 0.0, 0.0)))
    f2 = xo.rasterize_fwd(p2, r["binned"], cam, cfg0, dtype)
    assert np.array_equal(f2["n_contrib"], r["fwd"]["n_contrib"])          # the walk does not depend on the feature
    assert np.array_equal(f2["image"][..., 0], r["fwd"]["depth_img"])
    assert np.array_equal(f2["image"][..., 1], r["fwd"]["alpha_img"])
    assert r["fwd"]["depth_img"].max() > 1.0


def test_p15_alpha_is_one_minus_final_transmittance():
    # sum_k alpha_k T_k = 1 - prod_k (1 - alpha_k) (telescoping), also when the exit test stopped the walk
    arr, co = _scene(11, n=80, ls=(-1.0, 0.3), opac_boost=4.0)
    cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=1))
    r = xo.render_da(arr, cam, cfg, np.float64)
    f = r["fwd"]
    assert (f["final_T"] < 0.01).any() and (f["final_T"] > 0.5).any()
    assert np.abs(f["alpha_img"] - (1.0 - f["final_T"])).max() < 1e-13
    assert (f["depth_img"][f["n_contrib"] == 0] == 0).all()


def test_p15_constant_depth_plane():
    # all centres on the plane z_cam = z0 (identity pose): D = z0 A exactly up to rounding
    arr = draw_scene(5, 40, 1, opac_boost=0.5)
    arr["means"][:, 2] = 3.25
    co = cam_obj(W=48, H=40)
    cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=0))
    f = xo.render_da(arr, cam, cfg, np.float64)["fwd"]
    assert f["alpha_img"].max() > 0.3
    assert np.abs(f["depth_img"] - 3.25 * f["alpha_img"]).max() < 1e-12


def test_p15_backward_reduces_to_colour_backward():
    # gD = gA = 0: exactly rasterize_bwd
    arr, co = _scene(3)
    cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=1))
    r = xo.render_da(arr, cam, cfg, np.float64)
    rng = np.random.default_rng(0)
    Gw = rng.normal(0, 1, (co.height, co.width, 3))
    Z = np.zeros((co.height, co.width))
    a = xo.rasterize_bwd_da(r["proj"], r["binned"], r["fwd"], Gw, Z, Z, cam, cfg, np.float64)
    b = xo.rasterize_bwd(r["proj"], r["binned"], r["fwd"], Gw, cam, cfg, np.float64)
    for k in b:
        assert np.allclose(a[k], b[k], rtol=1e-13, atol=1e-15), k
    assert (a["g_depth"] == 0).all()


def _loss(arr, cam, cfg, Gw, Gd, Ga):
    r = xo.render_da(arr, cam, cfg, np.float64)
    f = r["fwd"]
    return float((f["image"] * Gw).sum() + (f["depth_img"] * Gd).sum() + (f["alpha_img"] * Ga).sum()), r


@pytest.mark.parametrize("which", ["depth", "alpha", "all"])
def test_p15_finite_differences(which):
    # d/dtheta of the forward, numerically, against backward_da; every parameter of every Gaussian
    found = None
    for seed in range(40):
        w2c = scenes.look_at((0.3, -0.2, -1.0), (0.0, 0.1, 3.0)).astype(np.float64)
        co = cam_obj(w2c=w2c, cx=19.0, cy=13.5, fy=66.0)
        arr = draw_scene(500 + seed, 6, 4, z=(1.5, 4.5), opac_boost=1.0)
        cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=1), fragile_rel=1e-4)
        rng = np.random.default_rng(seed)
        Gw = rng.normal(0, 1, (co.height, co.width, 3)) * (which == "all")
        Gd = rng.normal(0, 1, (co.height, co.width)) * (which in ("depth", "all"))
        Ga = rng.normal(0, 1, (co.height, co.width)) * (which in ("alpha", "all"))
        L0, r = _loss(arr, cam, cfg, Gw, Gd, Ga)
        if (r["fwd"]["fragile"] == 0).all() and (r["proj"]["tile_count"] > 0).sum() >= 5 and (r["fwd"]["n_contrib"] > 2).any():
            found = (arr, cam, cfg, Gw, Gd, Ga, r)
            break
    assert found is not None
    arr, cam, cfg, Gw, Gd, Ga, r = found
    g = xo.backward_da(arr, r, Gw, Gd, Ga, cam, cfg, np.float64)
    assert np.abs(g["g_depth"]).max() > 0 or which == "alpha"
    scale_all = max(np.abs(g[NAMES[k]]).max() for k in PARAMS)
    h_rel = 1e-6
    for k in PARAMS:
        if k == "sh" and which != "all":
            assert (g["g_sh"] == 0).all()
            continue
        base, an = arr[k], g[NAMES[k]]
        fd = np.zeros_like(base)
        it = np.nditer(base, flags=["multi_index"])
        for _ in it:
            idx = it.multi_index
            h = h_rel * max(1.0, abs(base[idx])) if k != "scales" else h_rel * abs(base[idx]) * 10
            ap = {kk: v.copy() for kk, v in arr.items()}; ap[k][idx] += h
            am = {kk: v.copy() for kk, v in arr.items()}; am[k][idx] -= h
            fd[idx] = (_loss(ap, cam, cfg, Gw, Gd, Ga)[0] - _loss(am, cam, cfg, Gw, Gd, Ga)[0]) / (2 * h)
        err = np.abs(fd - an)
        tol = 2e-6 * np.maximum(np.abs(an), np.abs(fd)) + 1e-7 * scale_all + 1e-9
        assert not (err > tol).any(), (k, np.argwhere(err > tol)[:5], fd[err > tol][:5], an[err > tol][:5])


# ---- P16: N-channel features (xpr_oracle_rasterize_fwd_featn / _bwd_featn) -------------------------------------------

def test_p16_three_channels_are_the_colour_pass():
    # C = 3, feat = rgb, bg = 0: forward and backward reproduce the pinned colour pass (P1, P2, P6)
    arr, co = _scene(21, opac_boost=1.0)
    cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=1, bg=(0.0, 0.0, 0.0)))
    for dtype in (np.float32, np.float64):
        r = xo.render(arr, cam, cfg, dtype)
        F = xo.rasterize_fwd_featn(r["proj"], r["binned"], r["proj"]["rgb"], cam, cfg, dtype)
        assert np.array_equal(F, r["fwd"]["image"]) and F.max() > 0.1
    rng = np.random.default_rng(1)
    Gw = rng.normal(0, 1, (co.height, co.width, 3))
    a = xo.rasterize_bwd_featn(r["proj"], r["binned"], r["fwd"], r["proj"]["rgb"], Gw, cam, cfg, np.float64)
    b = xo.rasterize_bwd(r["proj"], r["binned"], r["fwd"], Gw, cam, cfg, np.float64)
    for ka, kb in (("g_mean2d", "g_mean2d"), ("g_conic", "g_conic"), ("g_opac_eff", "g_opac_eff"), ("g_feat", "g_rgb")):
        assert np.allclose(a[ka], b[kb], rtol=1e-13, atol=1e-15), ka
        assert np.abs(b[kb]).max() > 0


def test_p16_depth_and_one_are_the_p15_passes():
    # C = 2, feat = (z, 1): the P15-pinned depth image and accumulated opacity, forward and backward; the colour
    # argument of the shared walk (a non-zero background here) does not enter
    arr, co = _scene(7, opac_boost=1.0)
    cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=1, bg=(0.3, 0.6, 0.9)))
    r = xo.render_da(arr, cam, cfg, np.float64)
    z = r["proj"]["depth"]
    feat = np.stack([z, np.ones_like(z)], 1)
    F = xo.rasterize_fwd_featn(r["proj"], r["binned"], feat, cam, cfg, np.float64)
    assert np.array_equal(F[..., 0], r["fwd"]["depth_img"]) and np.array_equal(F[..., 1], r["fwd"]["alpha_img"])
    rng = np.random.default_rng(2)
    Gf = rng.normal(0, 1, (co.height, co.width, 2))
    a = xo.rasterize_bwd_featn(r["proj"], r["binned"], r["fwd"], feat, Gf, cam, cfg, np.float64)
    Z3 = np.zeros((co.height, co.width, 3))
    b = xo.rasterize_bwd_da(r["proj"], r["binned"], r["fwd"], Z3, Gf[..., 0], Gf[..., 1], cam, cfg, np.float64)
    for k in ("g_mean2d", "g_conic", "g_opac_eff"):
        assert np.allclose(a[k], b[k], rtol=1e-12, atol=1e-14), k
    assert np.allclose(a["g_feat"][:, 0], b["g_depth"], rtol=1e-13, atol=1e-15)
    assert (b["g_rgb"] == 0).all()


def test_p16_finite_differences_five_channels():
    # the hand-derived backward against central differences of the forward, on the compositing inputs themselves
    # (feat, o_eff, mean2d, conic; lists and lnv fixed: the gates are piecewise constant, C15)
    found = None
    for seed in range(40):
        arr, co = _scene(600 + seed, n=12, opac_boost=1.0)
        cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=1), fragile_rel=1e-4)
        r = xo.render(arr, cam, cfg, np.float64)
        if (r["fwd"]["fragile"] == 0).all() and (r["fwd"]["n_contrib"] > 2).any():
            found = (arr, co, cam, cfg, r)
            break
    assert found is not None
    arr, co, cam, cfg, r = found
    rng = np.random.default_rng(3)
    N, Cn = r["proj"]["depth"].shape[0], 5
    feat = rng.normal(0, 1, (N, Cn))
    Gf = rng.normal(0, 1, (co.height, co.width, Cn))
    g = xo.rasterize_bwd_featn(r["proj"], r["binned"], r["fwd"], feat, Gf, cam, cfg, np.float64)

    def loss(proj, f):
        return float((xo.rasterize_fwd_featn(proj, r["binned"], f, cam, cfg, np.float64) * Gf).sum())

    vis = np.flatnonzero(r["proj"]["tile_count"] > 0)
    assert vis.size >= 5
    checks = 0
    for key, gk in (("feat", "g_feat"), ("opac_eff", "g_opac_eff"), ("mean2d", "g_mean2d"), ("conic", "g_conic")):
        base = feat if key == "feat" else r["proj"][key]
        scale = np.abs(g[gk]).max()
        assert scale > 0
        for i in vis[:6]:
            for j in range(base[i].size if base.ndim > 1 else 1):
                idx = (i, j) if base.ndim > 1 else (i,)
                h = 1e-6 * max(1.0, abs(base[idx]))
                vals = []
                for sgn in (+1, -1):
                    p2, f2 = dict(r["proj"]), feat
                    pert = base.copy(); pert[idx] += sgn * h
                    if key == "feat":
                        f2 = pert
                    else:
                        p2[key] = pert
                    vals.append(loss(p2, f2))
                fd = (vals[0] - vals[1]) / (2 * h)
                assert abs(fd - g[gk][idx]) <= 2e-6 * scale + 1e-5 * abs(fd), (key, idx, fd, g[gk][idx])
                checks += 1
    assert checks > 60


# ---- P15r: depth / accumulated opacity with the ray evaluation (f3 x f2) ------------------------------------------------

def test_p15r_ray_depth_and_alpha_are_colour_channels():
    # with rgb := (z, 1, 2 z), bg = 0 the pinned ray colour pass (P14) renders D and A bit for bit
    arr, co = _scene(7, opac_boost=1.0)
    for dtype in (np.float32, np.float64):
        cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=1, bg=(0.3, 0.6, 0.9)))
        r = xo.render_ray_da(arr, cam, cfg, dtype)
        assert (r["fwd"]["n_contrib"] > 3).any()
        p2 = dict(r["proj"])
        z = r["proj"]["depth"]
        p2["rgb"] = np.stack([z, np.ones_like(z), 2 * z], 1).astype(dtype)
        f2 = xo.rasterize_ray_fwd(p2, r["binned"], cam, xo.make_config(cfg_dict(sh_degree=1, bg=(0.0, 0.0, 0.0))), dtype)
        assert np.array_equal(f2["n_contrib"], r["fwd"]["n_contrib"])
        assert np.array_equal(f2["image"][..., 0], r["fwd"]["depth_img"])
        assert np.array_equal(f2["image"][..., 1], r["fwd"]["alpha_img"])
    f = r["fwd"]
    assert np.abs(f["alpha_img"] - (1.0 - f["final_T"])).max() < 1e-13 and f["depth_img"].max() > 1.0


def test_p15r_ray_backward_reduces_and_routes_agree():
    arr, co = _scene(3, opac_boost=1.0)
    cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=1))
    r = xo.render_ray_da(arr, cam, cfg, np.float64)
    rng = np.random.default_rng(0)
    Gw, Gd, Ga = rng.normal(0, 1, (co.height, co.width, 3)), rng.normal(0, 1, (co.height, co.width)), rng.normal(0, 1, (co.height, co.width))
    Z = np.zeros((co.height, co.width))
    a = xo.rasterize_ray_bwd_da(r["proj"], r["binned"], r["fwd"], Gw, Z, Z, cam, cfg, np.float64)
    b = xo.rasterize_ray_bwd(r["proj"], r["binned"], r["fwd"], Gw, cam, cfg, np.float64)
    for k in b:                                                     # gD = gA = 0: exactly rasterize_ray_bwd
        assert np.allclose(a[k], b[k], rtol=1e-13, atol=1e-15), k
    assert (a["g_depth"] == 0).all()
    # the accumulator form and the plain record gradient give the same parameter gradients (as P14f), features included
    g1 = xo.rasterize_ray_bwd_da(r["proj"], r["binned"], r["fwd"], Gw, Gd, Ga, cam, cfg, np.float64)
    g2 = xo.rasterize_ray_bwd_da(r["proj"], r["binned"], r["fwd"], Gw, Gd, Ga, cam, cfg, np.float64, acc=True)
    tc = r["proj"]["tile_count"]
    p1 = xo.ray_bwd(arr["means"], arr["scales"], arr["quats"], tc, g1["g_ray_rec"], cam, np.float64)
    p2 = xo.ray_bwd_acc(arr["means"], arr["scales"], arr["quats"], tc, g2["g_ray_acc"], cam, np.float64)
    for k in p1:
        s = np.abs(p1[k]).max()
        assert s > 0 and np.abs(p1[k] - p2[k]).max() <= 1e-9 * s, k
    assert np.allclose(g1["g_depth"], g2["g_depth"], rtol=1e-12, atol=1e-15) and np.abs(g1["g_depth"]).max() > 0
    m = xo.rasterize_ray_bwd_da(r["proj"], r["binned"], r["fwd"], Gw, Gd, Ga, cam, cfg, np.float64, mass=True)
    assert (m["g_depth"] >= np.abs(g1["g_depth"]) * (1 - 1e-12)).all()


def _loss_ray(arr, cam, cfg, Gw, Gd, Ga):
    r = xo.render_ray_da(arr, cam, cfg, np.float64)
    f = r["fwd"]
    return float((f["image"] * Gw).sum() + (f["depth_img"] * Gd).sum() + (f["alpha_img"] * Ga).sum()), r


def test_p15r_ray_finite_differences():
    found = None
    for seed in range(60):
        w2c = scenes.look_at((0.3, -0.2, -1.0), (0.0, 0.1, 3.0)).astype(np.float64)
        co = cam_obj(w2c=w2c, cx=19.0, cy=13.5, fy=66.0)
        arr = draw_scene(800 + seed, 6, 4, z=(1.5, 4.5), opac_boost=1.0)
        cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=1), fragile_rel=1e-4)
        rng = np.random.default_rng(seed)
        Gw, Gd, Ga = rng.normal(0, 1, (co.height, co.width, 3)), rng.normal(0, 1, (co.height, co.width)), rng.normal(0, 1, (co.height, co.width))
        L0, r = _loss_ray(arr, cam, cfg, Gw, Gd, Ga)
        if (r["fwd"]["fragile"] == 0).all() and (r["proj"]["tile_count"] > 0).sum() >= 5 and (r["fwd"]["n_contrib"] > 2).any():
            found = (arr, cam, cfg, Gw, Gd, Ga, r)
            break
    assert found is not None
    arr, cam, cfg, Gw, Gd, Ga, r = found
    g = xo.backward_ray_da(arr, r, Gw, Gd, Ga, cam, cfg, np.float64)
    scale_all = max(np.abs(g[NAMES[k]]).max() for k in PARAMS)
    h_rel = 1e-6
    for k in PARAMS:
        base, an = arr[k], g[NAMES[k]]
        fd = np.zeros_like(base)
        it = np.nditer(base, flags=["multi_index"])
        for _ in it:
            idx = it.multi_index
            h = h_rel * max(1.0, abs(base[idx])) if k != "scales" else h_rel * abs(base[idx]) * 10
            ap = {kk: v.copy() for kk, v in arr.items()}; ap[k][idx] += h
            am = {kk: v.copy() for kk, v in arr.items()}; am[k][idx] -= h
            fd[idx] = (_loss_ray(ap, cam, cfg, Gw, Gd, Ga)[0] - _loss_ray(am, cam, cfg, Gw, Gd, Ga)[0]) / (2 * h)
        err = np.abs(fd - an)
        tol = 2e-6 * np.maximum(np.abs(an), np.abs(fd)) + 1e-7 * scale_all + 1e-9
        assert not (err > tol).any(), (k, np.argwhere(err > tol)[:5], fd[err > tol][:5], an[err > tol][:5])
