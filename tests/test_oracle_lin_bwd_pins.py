"""Pin P19 of the ORACLE's hand-derived XPR-LinPrim backward (oracle/xpr_oracle_lin.inc lin_rasterize_bwd,
lin_project_bwd_one).  The paper has no backward equations (it relies on AD, L106): the authority is the derivative of
the forward definition (PAPER A.1.3 L506-629), so the checks differentiate the oracle's fp64 FORWARD numerically and
use closed forms -- no backward formula is retyped here.
  a  central finite differences over every parameter (means, scales, quats, opacities, sh), general rotated camera;
  b  the same with the alpha clamp (C14) and the transmittance exit (C15) active;
  c  closed form: on the optical axis through the centre of an axis-aligned octahedron whose shortest half-axis is the
     viewing one, alpha = 0.99 o (L522-528), so d image / d o = 0.99 rgb at that pixel, and the chord 2 s_z does not
     depend on the other two half-axes to first order there (their gradient is 0);
  d  exact zeros for culled primitives, linearity in dL/dimage, mass >= |gradient| element by element.
"""
import types

import numpy as np

import xpr_oracle as xo
from paper_2606_11529_b200 import scenes

AT = 1.0 / 255.0
C0 = 0.28209479177387814
PARAMS = ("means", "scales", "quats", "opacities", "sh")
NAMES = dict(means="g_means", scales="g_scales", quats="g_quats", opacities="g_opacities", sh="g_sh")


def cam_obj(W=40, H=24, fx=60.0, fy=66.0, cx=None, cy=None, w2c=None):
    if w2c is None:
        w2c = np.array([[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 0]], np.float64)
    return types.SimpleNamespace(model=0, width=W, height=H, fx=fx, fy=fy, cx=W / 2 if cx is None else cx,
                                 cy=H / 2 if cy is None else cy, k=(0, 0, 0, 0), w2c=np.asarray(w2c, np.float64))


def cfg_dict(**kw):
    d = dict(projection=0, sh_degree=2, tile=16, antialias=0, alpha_thresh=AT, alpha_max=0.99, t_min=1e-4, z_near=0.2,
             lowpass=0.3, ut_alpha=1.0, ut_beta=2.0, ut_kappa=0.0, bg=(0.1, 0.2, 0.3), tile_cull=1)
    d.update(kw)
    return d


def draw(seed, n, K, z=(2.0, 5.0), xy=0.8, ls=(-1.2, 0.35), opac_boost=0.0):
    rng = np.random.default_rng(seed)
    means = np.stack([rng.uniform(-xy, xy, n), rng.uniform(-xy * 0.6, xy * 0.6, n), rng.uniform(z[0], z[1], n)], 1)
    scales = np.exp(rng.normal(ls[0], ls[1], (n, 3)))
    q = rng.standard_normal((n, 4)); q /= np.linalg.norm(q, axis=1, keepdims=True)
    o = 1 / (1 + np.exp(-(rng.normal(0, 1.0, n) + opac_boost)))
    sh = np.concatenate([rng.normal(0, 0.5, (n, 1, 3)), rng.normal(0, 0.25, (n, K - 1, 3))], 1) if K > 1 else rng.normal(0, 0.5, (n, 1, 3))
    return dict(means=means, scales=scales, quats=q, opacities=o, sh=sh)


def loss_fn(arr, cam, cfg, Gw):
    r = xo.render_lin(arr, cam, cfg, np.float64)
    return float((r["fwd"]["image"] * Gw).sum()), r


def fd_check(arr, cam, cfg, Gw, rtol=5e-6, h_rel=1e-6):
    L0, r = loss_fn(arr, cam, cfg, Gw)
    assert (r["fwd"]["fragile"] == 0).all()
    g = xo.backward_lin(arr, r, Gw, cam, cfg, np.float64)
    scale_all = max(np.abs(g[NAMES[k]]).max() for k in PARAMS)
    assert scale_all > 0
    for k in PARAMS:
        base, an = arr[k], g[NAMES[k]]
        fd = np.zeros_like(base)
        it = np.nditer(base, flags=["multi_index"])
        for _ in it:
            idx = it.multi_index
            h = h_rel * max(1.0, abs(base[idx])) if k != "scales" else h_rel * abs(base[idx]) * 10
            ap = {kk: v.copy() for kk, v in arr.items()}; ap[k][idx] += h
            am = {kk: v.copy() for kk, v in arr.items()}; am[k][idx] -= h
            fd[idx] = (loss_fn(ap, cam, cfg, Gw)[0] - loss_fn(am, cam, cfg, Gw)[0]) / (2 * h)
        err = np.abs(fd - an)
        tol = rtol * np.maximum(np.abs(an), np.abs(fd)) + 1e-7 * scale_all + 1e-9
        bad = err > tol
        assert not bad.any(), (k, np.argwhere(bad)[:5], fd[bad][:5], an[bad][:5])
        assert np.abs(an).max() > 0, k
    return g, r


def find_seed(make, need, tries=60):
    for seed in range(tries):
        arr, cam, cfg, Gw = make(seed)
        _, r = loss_fn(arr, cam, cfg, Gw)
        if (r["fwd"]["fragile"] == 0).all() and need(arr, r):
            return arr, cam, cfg, Gw, r
    raise AssertionError("no suitable seed")


def test_p19a_fd_general():
    def make(seed):
        w2c = scenes.look_at((0.3, -0.2, -1.0), (0.0, 0.1, 3.0)).astype(np.float64)
        co = cam_obj(w2c=w2c, cx=19.0, cy=13.5)
        arr = draw(500 + seed, 6, 9, z=(1.5, 4.5))
        Gw = np.random.default_rng(seed).normal(0, 1, (co.height, co.width, 3))
        return arr, xo.make_camera(co), xo.make_config(cfg_dict(), fragile_rel=1e-4), Gw

    def need(arr, r):
        return (r["proj"]["tile_count"] > 0).sum() >= 5 and (r["fwd"]["n_contrib"] > 2).any()

    arr, cam, cfg, Gw, _ = find_seed(make, need)
    fd_check(arr, cam, cfg, Gw)


def test_p19b_fd_clamp_and_exit_active():
    def make(seed):
        co = cam_obj()
        arr = draw(700 + seed, 8, 4, z=(2.0, 4.0), xy=0.3, ls=(-0.7, 0.5), opac_boost=6.0)
        Gw = np.random.default_rng(seed).normal(0, 1, (co.height, co.width, 3))
        return arr, xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=1, tile_cull=0), fragile_rel=1e-4), Gw

    def need(arr, r):
        f = r["fwd"]
        lens = (r["binned"]["ranges"][:, 1] - r["binned"]["ranges"][:, 0]).max()
        exited = (f["final_T"] < 0.011).any() and (f["n_contrib"] < lens).any()
        # clamp: some pixel sees sigma dtau > -log(1 - 0.99)
        rec = r["proj"]["lin_rec"]
        vis = np.flatnonzero(r["proj"]["tile_count"] > 0)
        pix = np.stack(np.meshgrid(np.arange(40) + 0.5, np.arange(24) + 0.5), -1).reshape(-1, 2)
        clamp = any((xo.lin_chord(rec[i], pix, np.float64) > -np.log(0.01)).any() for i in vis)
        return exited and clamp

    arr, cam, cfg, Gw, _ = find_seed(make, need)
    fd_check(arr, cam, cfg, Gw)


def test_p19c_closed_form_centre_pixel():
    co = cam_obj(W=32, H=32, fx=80.0, fy=80.0, cx=16.5, cy=16.5)      # pixel (16, 16) has its centre on the optical axis
    o, rgb = 0.6, np.array([0.9, 0.5, 0.3])
    arr = dict(means=np.array([[0.0, 0.0, 4.0]]), scales=np.array([[0.5, 0.4, 0.2]]), quats=np.array([[1.0, 0, 0, 0]]),
               opacities=np.array([o]), sh=((rgb - 0.5) / C0).reshape(1, 1, 3))
    cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=0, bg=(0.0, 0.0, 0.0)), fragile_rel=1e-6)
    r = xo.render_lin(arr, cam, cfg, np.float64)
    np.testing.assert_allclose(r["fwd"]["image"][16, 16], 0.99 * o * rgb, rtol=1e-12)        # alpha = 0.99 o (L522-528)
    Gw = np.zeros((32, 32, 3)); Gw[16, 16] = (1.0, 2.0, -1.0)
    g = xo.backward_lin(arr, r, Gw, cam, cfg, np.float64)
    np.testing.assert_allclose(g["g_opacities"][0], 0.99 * float(rgb @ Gw[16, 16]), rtol=1e-12)
    # image = rgb (1 - (1 - 0.99 o)^(s_z / min s)) with min s = s_z: independent of s_z, s_x, s_y at this pixel
    np.testing.assert_allclose(g["g_scales"][0], 0.0, atol=1e-12)
    # d image_ch / d sh_0ch = C0 alpha
    np.testing.assert_allclose(g["g_sh"][0, 0], C0 * 0.99 * o * Gw[16, 16], rtol=1e-12)
    # when the viewing half-axis is NOT the shortest: alpha = 1 - (1 - 0.99 o)^(s_z / s_min), closed-form scale gradients
    arr2 = dict(arr, scales=np.array([[0.5, 0.1, 0.2]]))
    r2 = xo.render_lin(arr2, cam, cfg, np.float64)
    base, p = 1 - 0.99 * o, 0.2 / 0.1
    np.testing.assert_allclose(r2["fwd"]["image"][16, 16], rgb * (1 - base ** p), rtol=1e-12)
    g2 = xo.backward_lin(arr2, r2, Gw, cam, cfg, np.float64)
    dalpha_dp = -np.log(base) * base ** p
    w = float(rgb @ Gw[16, 16])
    np.testing.assert_allclose(g2["g_scales"][0], [0.0, w * dalpha_dp * (-0.2 / 0.01), w * dalpha_dp / 0.1], rtol=1e-10, atol=1e-12)


def test_p19d_zeros_linearity_mass():
    sc = scenes.make_scene(2, n_override=1500, image_override=(96, 64))
    arr = dict(means=sc.means.astype(np.float64), scales=sc.scales.astype(np.float64) * 3, quats=sc.quats.astype(np.float64),
               opacities=sc.opacities.astype(np.float64), sh=sc.sh.astype(np.float64))
    cam = xo.make_camera(sc.cameras[0])
    cfg = xo.make_config(dict(scenes.default_render_config(sc), tile_cull=1))
    r = xo.render_lin(arr, cam, cfg, np.float32)
    rng = np.random.default_rng(3)
    G1, G2 = rng.normal(0, 1, (64, 96, 3)), rng.normal(0, 1, (64, 96, 3))
    ga, gb = xo.backward_lin(arr, r, G1, cam, cfg, np.float32), xo.backward_lin(arr, r, G2, cam, cfg, np.float32)
    gc = xo.backward_lin(arr, r, (2 * G1 - 3 * G2).astype(np.float32), cam, cfg, np.float32)
    G1f, G2f = G1.astype(np.float32).astype(np.float64), G2.astype(np.float32).astype(np.float64)
    lin = (2 * G1f - 3 * G2f)
    assert np.abs(lin - (2 * G1 - 3 * G2).astype(np.float32)).max() < 1e-6
    for k in NAMES.values():
        s = np.abs(gc[k]).max()
        np.testing.assert_allclose(gc[k], 2 * ga[k] - 3 * gb[k], rtol=0, atol=2e-5 * s)
    culled = r["proj"]["tile_count"] == 0
    assert culled.any()
    for k in NAMES.values():
        assert not ga[k][culled].any()
    assert not ga["g_lin_rec"][culled].any() and not ga["g_lin_rec"][:, [3, 19]].any()
    mass = xo.lin_rasterize_bwd(r["proj"], r["binned"], r["fwd"], G1, cam, cfg, np.float32, mass=True)
    assert (mass >= np.abs(ga["g_lin_rec"]) * (1 - 1e-12)).all() and (mass > np.abs(ga["g_lin_rec"]) * 1.5).any()
