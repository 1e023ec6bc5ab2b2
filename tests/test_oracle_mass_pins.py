"""Pin of the ORACLE's `mass` outputs (xpr_oracle_rasterize_bwd_mass_*, _ray_bwd_mass_*, _bwd_da_mass_*).

mass[e] = sum over pixels of |the pixel's term of gradient element e| is the scale an fp32 sum of those terms
is conditioned on; the GPU gradient tolerance carries 2e-6 * mass, so a mass inflated by
any factor would silently widen the parity bar.  The inequality |sum| <= sum |.| does not fix its value.  This
file does: every step of the backward is linear in the incoming gradient, so the backward of a dL that is zero
outside ONE pixel is exactly that pixel's term -- mass must equal the brute-force sum over pixels of the absolute
value of those one-pixel gradients (computed with the separately pinned plain backward, P6 / P14d / P15).
For g_rgb the term of a pixel is per channel (alpha T g_ch), so the one-hot runs are per pixel AND per channel
there; the geometric elements combine the three channels inside the pixel before the absolute value
(dL/dalpha = sum_ch g_ch (...)), which is what a one-pixel dL with all its channels reproduces.
"""
import numpy as np

import xpr_oracle as xo
from paper_2606_11529_b200 import scenes
from test_oracle_backward_pins import cam_obj, cfg_dict, draw_scene

RT = 1e-10


def _tiny(seed, W=24, H=20, n=30, K=1, **kw):
    w2c = scenes.look_at((0.1, -0.05, -0.8), (0.0, 0.05, 3.0)).astype(np.float64)
    co = cam_obj(w2c=w2c, W=W, H=H, fx=36.0, fy=36.0, cx=W / 2 - 0.5, cy=H / 2 + 0.25)
    return draw_scene(seed, n, K, **kw), co


def _one_pixel(dL, y, x):
    d = np.zeros_like(dL)
    d[y, x] = dL[y, x]
    return d


def _assert_mass(mass, brute, keys):
    for k in keys:
        scale = np.abs(brute[k]).max()
        assert scale > 0, k
        np.testing.assert_allclose(mass[k], brute[k], rtol=RT, atol=RT * scale, err_msg=k)


def test_mass_equals_brute_force_sum_of_one_pixel_terms_2d():
    arr, co = _tiny(21, opac_boost=1.5, ls=(-1.4, 0.4))
    cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=0))
    r = xo.render(arr, cam, cfg, np.float64)
    assert (r["fwd"]["n_contrib"] > 3).any()
    H, W = co.height, co.width
    dL = np.random.default_rng(3).standard_normal((H, W, 3))
    bwd = lambda d: xo.rasterize_bwd(r["proj"], r["binned"], r["fwd"], d, cam, cfg, np.float64)
    m = xo.rasterize_bwd(r["proj"], r["binned"], r["fwd"], dL, cam, cfg, np.float64, mass=True)
    geo = ("g_mean2d", "g_conic", "g_opac_eff")
    brute = {k: 0.0 for k in geo + ("g_rgb",)}
    for y in range(H):
        for x in range(W):
            g = bwd(_one_pixel(dL, y, x))
            for k in geo:
                brute[k] = brute[k] + np.abs(g[k])
            for ch in range(3):           # the colour gradient's term is per (pixel, channel)
                d = np.zeros_like(dL); d[y, x, ch] = dL[y, x, ch]
                brute["g_rgb"] = brute["g_rgb"] + np.abs(bwd(d)["g_rgb"])
    _assert_mass(m, brute, geo + ("g_rgb",))
    # and the mass really differs from |gradient| (cancellation between pixels occurs on this scene)
    gfull = bwd(dL)
    assert (m["g_mean2d"] > 1.5 * np.abs(gfull["g_mean2d"])).any()


def test_mass_equals_brute_force_sum_of_one_pixel_terms_ray():
    arr, co = _tiny(22, opac_boost=1.5, ls=(-1.4, 0.4))
    cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=0))
    r = xo.render_ray(arr, cam, cfg, np.float64)
    assert (r["fwd"]["n_contrib"] > 3).any()
    H, W = co.height, co.width
    dL = np.random.default_rng(4).standard_normal((H, W, 3))
    bwd = lambda d: xo.rasterize_ray_bwd(r["proj"], r["binned"], r["fwd"], d, cam, cfg, np.float64)
    m = xo.rasterize_ray_bwd(r["proj"], r["binned"], r["fwd"], dL, cam, cfg, np.float64, mass=True)
    geo = ("g_ray_rec", "g_opac_eff")
    brute = {k: 0.0 for k in geo + ("g_rgb",)}
    for y in range(H):
        for x in range(W):
            g = bwd(_one_pixel(dL, y, x))
            for k in geo:
                brute[k] = brute[k] + np.abs(g[k])
            for ch in range(3):
                d = np.zeros_like(dL); d[y, x, ch] = dL[y, x, ch]
                brute["g_rgb"] = brute["g_rgb"] + np.abs(bwd(d)["g_rgb"])
    _assert_mass(m, brute, geo + ("g_rgb",))


def test_mass_equals_brute_force_sum_of_one_pixel_terms_depth_alpha():
    arr, co = _tiny(23, opac_boost=1.5, ls=(-1.4, 0.4))
    cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=0))
    r = xo.render_da(arr, cam, cfg, np.float64)
    H, W = co.height, co.width
    rng = np.random.default_rng(5)
    dL, gD, gA = rng.standard_normal((H, W, 3)), rng.standard_normal((H, W)), rng.standard_normal((H, W))
    bwd = lambda a, b, c: xo.rasterize_bwd_da(r["proj"], r["binned"], r["fwd"], a, b, c, cam, cfg, np.float64)
    m = xo.rasterize_bwd_da(r["proj"], r["binned"], r["fwd"], dL, gD, gA, cam, cfg, np.float64, mass=True)
    geo = ("g_mean2d", "g_conic", "g_opac_eff")
    brute = {k: 0.0 for k in geo + ("g_rgb", "g_depth")}
    z2, z3 = np.zeros((H, W)), np.zeros((H, W, 3))
    for y in range(H):
        for x in range(W):
            a, b, c = _one_pixel(dL, y, x), _one_pixel(gD, y, x), _one_pixel(gA, y, x)
            g = bwd(a, b, c)
            for k in geo:
                brute[k] = brute[k] + np.abs(g[k])
            brute["g_depth"] = brute["g_depth"] + np.abs(bwd(z3, b, z2)["g_depth"])     # term alpha T gD
            for ch in range(3):
                d = np.zeros_like(dL); d[y, x, ch] = dL[y, x, ch]
                brute["g_rgb"] = brute["g_rgb"] + np.abs(bwd(d, z2, z2)["g_rgb"])
    _assert_mass(m, brute, geo + ("g_rgb", "g_depth"))
