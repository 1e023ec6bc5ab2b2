"""Pins of the ORACLE's XPR-3DGUT ray evaluation (PAPER A.1.2 L437-444 Eq. 1, Listing 3):
P14a  the response equals the maximum of the 3D Gaussian density along the ray, found by brute force in the
      WORLD frame with an independently built covariance (scipy rotation, numpy inverse) -- pins Eq. 1, the
      camera-frame reading C27 and the record (o_c, M);
P14b  closed form for an isotropic Gaussian, single-Gaussian image incl. the `response > 0.0113` gate;
P14c  pixel_info is the inverse of the (separately pinned, P9) camera model;
P14d  central finite differences of the whole forward (fp64) against the hand-derived backward;
P14e  linearity, exact zeros, mass; fp32 parity mode vs fp64; agreement with the 2D EWA path in its limit.
"""
import numpy as np
import pytest
from scipy.optimize import minimize_scalar
from scipy.spatial.transform import Rotation

import xpr_oracle as xo
from paper_2606_11529_b200 import scenes
from test_oracle_backward_pins import PARAMS, cam_obj, cfg_dict, draw_scene

FISHEYE_K = (0.04, -0.03, 0.02, -0.01)


def world_sigma(s, q):
    R = Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix()     # scipy order is (x, y, z, w)
    return R @ np.diag(np.asarray(s) ** 2) @ R.T


@pytest.mark.parametrize("model", [0, 1])
def test_p14a_response_is_the_maximum_along_the_ray_world_frame(model):
    rng = np.random.default_rng(14 + model)
    for trial in range(40):
        w2c = scenes.look_at(rng.uniform(-1, 1, 3), rng.uniform(-0.5, 0.5, 3) + (0, 0, 4.0)).astype(np.float64)
        U, _, Vt = np.linalg.svd(w2c[:, :3])          # look_at rounds to fp32: make W a rotation to fp64 accuracy
        w2c[:, :3] = U @ Vt                           # (C27 is the rigid-pose reading: W^T = W^-1)
        co = cam_obj(model=model, w2c=w2c, W=64, H=48, fx=50.0, fy=55.0, cx=30.0, cy=25.0,
                     k=FISHEYE_K if model else (0, 0, 0, 0))
        cam = xo.make_camera(co)
        mu = rng.uniform(-1, 1, 3) + (0, 0, 4.0)
        s = np.exp(rng.normal(-1.0, 0.6, 3))
        q = rng.standard_normal(4); q /= np.linalg.norm(q)
        u, v = rng.uniform(0, 64), rng.uniform(0, 48)
        rec = xo.project_ray(mu[None], s[None], q[None], np.ones(1, np.uint32), cam, np.float64)[0]
        d_cam = xo.pixel_ray(cam, u, v)
        power = xo.ray_power(rec, d_cam)[0]
        # independent: world frame, Sigma from scipy's rotation, ray from the camera centre
        Wm, t = w2c[:, :3], w2c[:, 3]
        o_w, d_w = -Wm.T @ t, Wm.T @ d_cam
        Pinv = np.linalg.inv(world_sigma(s, q))
        f = lambda tau: 0.5 * (o_w + tau * d_w - mu) @ Pinv @ (o_w + tau * d_w - mu)
        tau_star = ((mu - o_w) @ Pinv @ d_w) / (d_w @ Pinv @ d_w)                       # Eq. 1, first form
        assert abs(-f(tau_star) - power) <= 1e-9 * max(1.0, abs(power))
        res = minimize_scalar(f, bracket=(tau_star - 1.0, tau_star + 1.0), tol=1e-13)  # brute force on tau
        assert abs(-res.fun - power) <= 1e-8 * max(1.0, abs(power))
        taus = tau_star + np.linspace(-2, 2, 2001)
        assert min(f(x) for x in taus) >= -power - 1e-9 * max(1.0, abs(power))         # nothing along the ray beats it
        # the record itself: M^T M = (W Sigma W^T)^-1 and o_c = -M p
        M = rec[:9].reshape(3, 3)
        np.testing.assert_allclose(M.T @ M, np.linalg.inv(Wm @ world_sigma(s, q) @ Wm.T), rtol=1e-9, atol=1e-9)
        np.testing.assert_allclose(rec[9:], -M @ (Wm @ mu + t), rtol=1e-12, atol=1e-12)


def test_p14b_isotropic_closed_form_and_the_response_gate():
    # one isotropic Gaussian: response = exp(-|p x d|^2 / (2 sigma^2)); pixel = o r c + (1 - o r) bg where
    # r > 0.0113 and o r >= 1/255, bg elsewhere (L500, C12)
    co = cam_obj(W=48, H=32, fx=40.0, fy=40.0)
    cam = xo.make_camera(co)
    sig, o = 0.25, 0.9
    p = np.array([0.2, -0.1, 3.0])
    arr = dict(means=p[None], scales=np.full((1, 3), sig), quats=np.array([[0.3, -0.5, 0.1, 0.8]]) / np.linalg.norm([0.3, -0.5, 0.1, 0.8]),
               opacities=np.array([o]), sh=np.zeros((1, 1, 3)))
    arr["sh"][0, 0] = (np.array([0.9, 0.5, 0.2]) - 0.5) / 0.28209479177387814
    cfg = xo.make_config(cfg_dict(sh_degree=0, lowpass=0.0))
    # enlarge the footprint so that every pixel the ray evaluation accepts is inside the tile rectangle
    r = xo.render_ray(arr, cam, cfg, np.float64)
    assert r["proj"]["tile_count"][0] == 6            # the whole 3 x 2 tile image
    ys, xs = np.mgrid[0:32, 0:48]
    d = np.stack([(xs + 0.5 - 24.0) / 40.0, (ys + 0.5 - 16.0) / 40.0, np.ones_like(xs, float)], -1)
    d /= np.linalg.norm(d, axis=-1, keepdims=True)
    np.testing.assert_allclose(r["proj"]["pixel_rays"], d, rtol=0, atol=1e-15)
    resp = np.exp(-0.5 * (np.cross(p, d) ** 2).sum(-1) / sig ** 2)
    on = (resp > 0.0113) & (o * resp >= 1 / 255)
    assert on.any() and (~on).any() and ((resp <= 0.0113) & (o * resp >= 1 / 255)).any()   # the new gate binds
    al = np.minimum(0.99, o * resp) * on
    want = al[..., None] * np.array([0.9, 0.5, 0.2]) + (1 - al[..., None]) * np.array([0.1, 0.2, 0.3])
    edge = (np.abs(resp - 0.0113) < 1e-9)
    np.testing.assert_allclose(r["fwd"]["image"][~edge], want[~edge], rtol=1e-12, atol=1e-12)
    np.testing.assert_array_equal(r["fwd"]["n_contrib"][~edge], on[~edge].astype(np.uint32))


@pytest.mark.parametrize("model", [0, 1])
def test_p14c_pixel_info_inverts_the_camera_model(model):
    co = cam_obj(model=model, W=80, H=60, fx=60.0, fy=66.0, cx=41.0, cy=28.5, k=FISHEYE_K if model else (0, 0, 0, 0))
    cam = xo.make_camera(co)
    rng = np.random.default_rng(3)
    for _ in range(200):
        u, v = rng.uniform(0, 80), rng.uniform(0, 60)
        d = xo.pixel_ray(cam, u, v)
        assert abs(np.linalg.norm(d) - 1) < 1e-14
        for lam in (0.5, 7.0):
            np.testing.assert_allclose(xo.camera_project(cam, lam * d), (u, v), rtol=0, atol=1e-9)
    rays = xo.pixel_info(cam, np.float64)
    assert rays.shape == (60, 80, 3)
    for py, px in ((0, 0), (59, 79), (17, 43)):
        np.testing.assert_array_equal(rays[py, px], xo.pixel_ray(cam, px + 0.5, py + 0.5))
    r32 = xo.pixel_info(cam, np.float32)
    np.testing.assert_array_equal(r32, rays.astype(np.float32))          # R2: fp64, rounded last
    if model == 1:   # on-axis pixel of a fisheye: straight ahead
        np.testing.assert_array_equal(xo.pixel_ray(cam, 41.0, 28.5), (0, 0, 1))


def loss_ray(arr, cam, cfg, Gw):
    r = xo.render_ray(arr, cam, cfg, np.float64)
    return float((r["fwd"]["image"] * Gw).sum()), r


def fd_check_ray(arr, cam, cfg, Gw, rtol=5e-6, h_rel=1e-6):
    L0, r = loss_ray(arr, cam, cfg, Gw)
    assert (r["fwd"]["fragile"] == 0).all()
    g = xo.backward_ray(arr, r, Gw, cam, cfg, np.float64)
    names = dict(means="g_means", scales="g_scales", quats="g_quats", opacities="g_opacities", sh="g_sh")
    scale_all = max(np.abs(g[names[k]]).max() for k in PARAMS)
    for k in PARAMS:
        base, an = arr[k], g[names[k]]
        fd = np.zeros_like(base)
        it = np.nditer(base, flags=["multi_index"])
        for _ in it:
            idx = it.multi_index
            h = h_rel * max(1.0, abs(base[idx])) if k != "scales" else h_rel * abs(base[idx]) * 10
            ap = {kk: v.copy() for kk, v in arr.items()}; ap[k][idx] += h
            am = {kk: v.copy() for kk, v in arr.items()}; am[k][idx] -= h
            rp, rm = loss_ray(ap, cam, cfg, Gw), loss_ray(am, cam, cfg, Gw)
            # the 2D footprint only tiles: a perturbation must not change the lists (else re-draw)
            assert rp[1]["binned"]["num_pairs"] == r["binned"]["num_pairs"] == rm[1]["binned"]["num_pairs"]
            fd[idx] = (rp[0] - rm[0]) / (2 * h)
        err = np.abs(fd - an)
        tol = rtol * np.maximum(np.abs(an), np.abs(fd)) + 1e-7 * scale_all + 1e-9
        bad = err > tol
        assert not bad.any(), (k, np.argwhere(bad)[:5], fd[bad][:5], an[bad][:5])
    return g, r


def find_seed_ray(make, need, tries=80):
    for seed in range(tries):
        arr, cam, cfg, Gw = make(seed)
        _, r = loss_ray(arr, cam, cfg, Gw)
        if (r["fwd"]["fragile"] == 0).all() and need(arr, r):
            return arr, cam, cfg, Gw, r
    raise AssertionError("no suitable seed")


@pytest.mark.parametrize("model,projection,antialias", [(0, 0, 0), (0, 1, 1), (1, 1, 1)])
def test_p14d_finite_differences(model, projection, antialias):
    def make(seed):
        w2c = scenes.look_at((0.2, 0.1, -0.5), (0.0, 0.0, 3.0)).astype(np.float64)
        co = cam_obj(model=model, w2c=w2c, k=FISHEYE_K if model else (0, 0, 0, 0), fx=45.0, fy=45.0)
        arr = draw_scene(1400 + seed, 5, 4, z=(1.5, 4.0))
        Gw = np.random.default_rng(seed).normal(0, 1, (co.height, co.width, 3))
        cfg = xo.make_config(cfg_dict(projection=projection, antialias=antialias, sh_degree=1), fragile_rel=1e-4)
        return arr, xo.make_camera(co), cfg, Gw

    def need(arr, r):
        return (r["proj"]["tile_count"] > 0).sum() >= 4 and (r["fwd"]["n_contrib"] > 2).any()

    arr, cam, cfg, Gw, _ = find_seed_ray(make, need)
    g, r = fd_check_ray(arr, cam, cfg, Gw)
    assert np.abs(g["ray_part"]["g_quats"]).max() > 0 and np.abs(g["ray_part"]["g_scales"]).max() > 0


def test_p14d_finite_differences_clamp_and_exit_active():
    def make(seed):
        co = cam_obj()
        arr = draw_scene(1500 + seed, 8, 4, z=(2.0, 4.0), xy=0.3, ls=(-0.9, 0.2), opac_boost=7.0)
        Gw = np.random.default_rng(seed).normal(0, 1, (co.height, co.width, 3))
        return arr, xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=1), fragile_rel=1e-4), Gw

    def need(arr, r):
        f = r["fwd"]
        tiles_max = (r["binned"]["ranges"][:, 1] - r["binned"]["ranges"][:, 0]).max()
        return (f["final_T"] < 0.011).any() and (f["n_contrib"] < tiles_max).any()

    arr, cam, cfg, Gw, _ = find_seed_ray(make, need)
    fd_check_ray(arr, cam, cfg, Gw)


def test_p14e_linearity_zeros_mass_and_fp32_mode():
    sc = scenes.make_scene(4, n_override=6000, image_override=(96, 64))
    arr = {k: getattr(sc, k).astype(np.float64).copy() for k in PARAMS}
    arr["means"][7] = [0, 0, -10.0]          # behind the camera -> culled
    cam = xo.make_camera(sc.cameras[0]); cfg = xo.make_config(scenes.default_render_config(sc))
    r = xo.render_ray(arr, cam, cfg, np.float64)
    assert r["proj"]["tile_count"][7] == 0 and (r["proj"]["ray_rec"][7] == 0).all()
    assert r["fwd"]["pp_pass"] > 1000
    rng = np.random.default_rng(1)
    G1, G2 = rng.normal(0, 1, (64, 96, 3)), rng.normal(0, 1, (64, 96, 3))
    g1, g2 = xo.backward_ray(arr, r, G1, cam, cfg, np.float64), xo.backward_ray(arr, r, G2, cam, cfg, np.float64)
    g12 = xo.backward_ray(arr, r, 2.0 * G1 - 3.0 * G2, cam, cfg, np.float64)
    for k in g1:
        if k == "ray_part":
            continue
        np.testing.assert_allclose(g12[k], 2.0 * g1[k] - 3.0 * g2[k], rtol=1e-9, atol=1e-9 * np.abs(g1[k]).max())
        assert (g1[k][7] == 0).all()
    m = xo.rasterize_ray_bwd(r["proj"], r["binned"], r["fwd"], G1, cam, cfg, np.float64, mass=True)
    for k in ("g_ray_rec", "g_opac_eff", "g_rgb"):
        assert (m[k] >= np.abs(g1[k]) * (1 - 1e-12) - 1e-300).all(), k
        assert (m[k] > np.abs(g1[k]) * 1.01).any(), k
    gp = xo.rasterize_ray_bwd(r["proj"], r["binned"], r["fwd"], np.abs(G1), cam, cfg, np.float64)
    np.testing.assert_allclose(m["g_rgb"], gp["g_rgb"], rtol=1e-13, atol=0)
    # fp32 parity mode: same decisions away from fragile pixels, image within 1e-4
    arr32 = {k: v.astype(np.float32) for k, v in arr.items()}
    r32 = xo.render_ray(arr32, cam, cfg, np.float32)
    np.testing.assert_array_equal(r32["binned"]["vals"], r["binned"]["vals"])
    ok = (r32["fwd"]["fragile"] | r["fwd"]["fragile"]) == 0
    assert ok.mean() > 0.9
    np.testing.assert_array_equal(r32["fwd"]["n_contrib"][ok], r["fwd"]["n_contrib"][ok])
    assert np.abs(r32["fwd"]["image"].astype(np.float64) - r["fwd"]["image"])[ok].max() < 1e-4


def test_p14e_agrees_with_the_2d_path_for_small_distant_gaussians():
    # EWA linearises the projection around the mean: for Gaussians that are small against their
    # distance the 2D conic response and the response along the ray coincide to first order
    rng = np.random.default_rng(8)
    n = 40
    co = cam_obj(W=64, H=48, fx=400.0, fy=400.0)
    cam = xo.make_camera(co)
    means = np.stack([rng.uniform(-0.3, 0.3, n), rng.uniform(-0.2, 0.2, n), rng.uniform(4.5, 5.5, n)], 1)
    arr = dict(means=means, scales=np.exp(rng.normal(np.log(0.02), 0.3, (n, 3))), quats=rng.standard_normal((n, 4)),
               opacities=rng.uniform(0.2, 0.7, n), sh=rng.normal(0, 0.5, (n, 1, 3)))
    arr["quats"] /= np.linalg.norm(arr["quats"], axis=1, keepdims=True)
    cfg = xo.make_config(cfg_dict(sh_degree=0, lowpass=0.0))
    a = xo.render(arr, cam, cfg, np.float64)["fwd"]["image"]
    b = xo.render_ray(arr, cam, cfg, np.float64)["fwd"]["image"]
    assert np.abs(a - np.array([0.1, 0.2, 0.3])).max() > 0.2          # something is drawn
    assert np.abs(a - b).max() < 2e-2 and np.abs(a - b).mean() < 5e-4


# ------------------------------------------------------------------------------------------------
# P14f: the accumulator form of the record gradient (what the GPU sums: S_c = sum k c c^T, D = sum 2 dL/ddd d d^T,
# sum dL/do_c) determines the same parameter gradients as the plain form (dL/dM_c, dL/do_c) of the definition:
#   dL/dM_c - dL/do_c p^T = -(S_c - tr(S_c) I) M_c^-T + M_c D      (o_c = -M_c p, d_c = M_c d, c = o_c x d_c).
# The plain route is pinned by finite differences (P14d); here the two routes must agree in fp64 on general scenes
# (EWA / UT footprints, pinhole and fisheye), and the mass of the accumulators equals the brute-force sum over
# one-pixel gradients, as for the other mass outputs (tests/test_oracle_mass_pins.py).
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("config,kw", [(1, dict(n_override=400)), (4, dict(n_override=6000, image_override=(96, 64))),
                                       (2, dict(n_override=3000, image_override=(80, 80)))])
def test_p14f_accumulator_route_equals_plain_route(config, kw):
    sc = scenes.make_scene(config, **kw)
    arr = {k: getattr(sc, k).astype(np.float64) for k in PARAMS}
    cam = xo.make_camera(sc.cameras[0]); cfg = xo.make_config(scenes.default_render_config(sc))
    r = xo.render_ray(arr, cam, cfg, np.float64)
    assert r["fwd"]["pp_pass"] > 500
    H, W = int(cam.height), int(cam.width)
    G = np.random.default_rng(3).normal(0, 1, (H, W, 3))
    plain = xo.rasterize_ray_bwd(r["proj"], r["binned"], r["fwd"], G, cam, cfg, np.float64)
    acc = xo.rasterize_ray_bwd_acc(r["proj"], r["binned"], r["fwd"], G, cam, cfg, np.float64)
    # (equal up to the order in which the tiles' contributions are added)
    np.testing.assert_allclose(acc["g_opac_eff"], plain["g_opac_eff"], rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(acc["g_rgb"], plain["g_rgb"], rtol=1e-12, atol=1e-14)
    s3 = np.abs(plain["g_ray_rec"][:, 9:12]).max()
    np.testing.assert_allclose(acc["g_ray_acc"][:, 12:15], plain["g_ray_rec"][:, 9:12], rtol=1e-12, atol=1e-13 * s3)
    tc = r["proj"]["tile_count"]
    a = xo.ray_bwd(arr["means"], arr["scales"], arr["quats"], tc, plain["g_ray_rec"], cam, np.float64)
    b = xo.ray_bwd_acc(arr["means"], arr["scales"], arr["quats"], tc, acc["g_ray_acc"], cam, np.float64)
    for k in ("g_means", "g_scales", "g_quats"):
        scale = np.abs(a[k]).max(axis=1, keepdims=True) + 1e-300
        assert np.abs(a[k]).max() > 0
        # per Gaussian: agreement to rounding of the LARGER of the two cancelling parts of the plain route
        big = (np.abs(plain["g_ray_rec"]).max(axis=1, keepdims=True) * (1 + np.abs(arr["means"]).max()) + scale)
        assert (np.abs(a[k] - b[k]) <= 1e-9 * big / np.minimum(arr["scales"].min(axis=1, keepdims=True), 1.0)).all(), k
        # and to 1e-7 relative of the Gaussian's largest component for all but a handful (plain-route cancellation in fp64)
        rel = np.abs(a[k] - b[k]) / scale
        assert np.quantile(rel, 0.99) < 1e-8, (k, np.quantile(rel, 0.99))


def test_p14f_accumulator_mass_equals_brute_force():
    from test_oracle_mass_pins import _tiny, _one_pixel
    arr, co = _tiny(24, opac_boost=1.5, ls=(-1.4, 0.4))
    cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=0))
    r = xo.render_ray(arr, cam, cfg, np.float64)
    H, W = co.height, co.width
    dL = np.random.default_rng(6).standard_normal((H, W, 3))
    bwd = lambda d: xo.rasterize_ray_bwd_acc(r["proj"], r["binned"], r["fwd"], d, cam, cfg, np.float64)
    m = xo.rasterize_ray_bwd_acc(r["proj"], r["binned"], r["fwd"], dL, cam, cfg, np.float64, mass=True)
    brute = 0.0
    for y in range(H):
        for x in range(W):
            brute = brute + np.abs(bwd(_one_pixel(dL, y, x))["g_ray_acc"])
    assert np.abs(brute).max() > 0
    np.testing.assert_allclose(m["g_ray_acc"], brute, rtol=1e-10, atol=1e-10 * np.abs(brute).max())


def test_p14g_degenerate_record_contributes_nothing_and_gets_zero_gradients():
    """Reading C30: a Gaussian whose shader record is not finite (zero scale: M_c = S^-1 (W R)^T is infinite) is never
    valid -- the image is the image of the scene WITHOUT it, and its gradient is exactly zero (not NaN) on both
    record-gradient routes; the other Gaussians' gradients are those of the scene without it."""
    co = cam_obj(W=40, H=24)
    arr = draw_scene(41, 8, 4, z=(2.0, 4.0), xy=0.4, opac_boost=1.0)
    cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=1))
    bad = {k: v.copy() for k, v in arr.items()}
    bad["scales"][2] = (0.0, 0.05, 0.05)                     # one zero scale: the 2D footprint (low-passed) still covers tiles
    r = xo.render_ray(bad, cam, cfg, np.float64)
    assert r["proj"]["tile_count"][2] > 0 and not r["proj"]["ray_rec"][2].any()
    keep = np.array([i for i in range(8) if i != 2])
    sub = {k: v[keep] for k, v in arr.items()}
    r0 = xo.render_ray(sub, cam, cfg, np.float64)
    np.testing.assert_allclose(r["fwd"]["image"], r0["fwd"]["image"], rtol=0, atol=1e-14)
    Gw = np.random.default_rng(0).normal(0, 1, (co.height, co.width, 3))
    g = xo.backward_ray(bad, r, Gw, cam, cfg, np.float64)
    g0 = xo.backward_ray(sub, r0, Gw, cam, cfg, np.float64)
    for k in ("g_means", "g_scales", "g_quats", "g_opacities", "g_sh"):
        assert np.isfinite(g[k]).all(), k
        assert not np.any(g[k][2]), k
        np.testing.assert_allclose(g[k][keep], g0[k], rtol=1e-12, atol=1e-14)
    ga = xo.rasterize_ray_bwd_acc(r["proj"], r["binned"], r["fwd"], Gw, cam, cfg, np.float64)
    pa = xo.ray_bwd_acc(bad["means"], bad["scales"], bad["quats"], r["proj"]["tile_count"], ga["g_ray_acc"], cam, np.float64)
    for k in pa:
        assert np.isfinite(pa[k]).all() and not np.any(pa[k][2]), k
