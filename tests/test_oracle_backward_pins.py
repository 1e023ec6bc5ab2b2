"""Pins of the ORACLE's hand-derived backward pass: central finite differences in fp64 (P6),
linearity and exact zeros (P11).  The paper has no backward equations (it relies on AD, L106);
the only authority is the derivative of the forward definition itself, so the check
differentiates the oracle's *forward* numerically -- it never re-types a backward formula.
"""
import types

import numpy as np
import pytest

import xpr_oracle as xo
from paper_2606_11529_b200 import scenes

AT = 1.0 / 255.0
PARAMS = ("means", "scales", "quats", "opacities", "sh")


def cam_obj(model=0, W=40, H=24, fx=60.0, fy=60.0, cx=None, cy=None, w2c=None, k=(0, 0, 0, 0)):
    if w2c is None:
        w2c = np.array([[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 0]], np.float64)
    return types.SimpleNamespace(model=model, width=W, height=H, fx=fx, fy=fy, cx=W / 2 if cx is None else cx,
                                 cy=H / 2 if cy is None else cy, k=k, w2c=np.asarray(w2c, np.float64))


def cfg_dict(**kw):
    d = dict(projection=0, sh_degree=3, tile=16, antialias=0, alpha_thresh=AT, alpha_max=0.99, t_min=1e-4,
             z_near=0.2, lowpass=0.3, ut_alpha=1.0, ut_beta=2.0, ut_kappa=0.0, bg=(0.1, 0.2, 0.3))
    d.update(kw)
    return d


def draw_scene(seed, n, K, z=(2.0, 5.0), xy=0.8, ls=(-1.8, 0.4), opac_boost=0.0):
    rng = np.random.default_rng(seed)
    means = np.stack([rng.uniform(-xy, xy, n), rng.uniform(-xy * 0.6, xy * 0.6, n), rng.uniform(z[0], z[1], n)], 1)
    scales = np.exp(rng.normal(ls[0], ls[1], (n, 3)))
    q = rng.standard_normal((n, 4)); q /= np.linalg.norm(q, axis=1, keepdims=True)
    o = 1 / (1 + np.exp(-(rng.normal(0, 1.0, n) + opac_boost)))
    sh = np.concatenate([rng.normal(0, 0.5, (n, 1, 3)), rng.normal(0, 0.25, (n, K - 1, 3))], 1) if K > 1 else rng.normal(0, 0.5, (n, 1, 3))
    return dict(means=means, scales=scales, quats=q, opacities=o, sh=sh)


def loss_fn(arr, cam, cfg, Gw):
    r = xo.render(arr, cam, cfg, np.float64)
    return float((r["fwd"]["image"] * Gw).sum()), r


def fd_check(arr, cam, cfg, Gw, rtol=2e-6, h_rel=1e-6):
    L0, r = loss_fn(arr, cam, cfg, Gw)
    assert (r["fwd"]["fragile"] == 0).all(), "re-draw: a decision margin is too small for finite differences"
    g = xo.backward(arr, r, Gw, cam, cfg, np.float64)
    names = dict(means="g_means", scales="g_scales", quats="g_quats", opacities="g_opacities", sh="g_sh")
    worst = 0.0
    scale_all = max(np.abs(g[names[k]]).max() for k in PARAMS)
    for k in PARAMS:
        base = arr[k]
        an = g[names[k]]
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
        worst = max(worst, float((err / (np.abs(an) + 1e-7 * scale_all + 1e-9)).max()))
    return g, r, worst


def find_seed(make, need, tries=60):
    """Re-draw until the fragile mask is empty (P6 protocol) and the wanted cases are present."""
    for seed in range(tries):
        arr, cam, cfg, Gw = make(seed)
        _, r = loss_fn(arr, cam, cfg, Gw)
        if (r["fwd"]["fragile"] == 0).all() and need(arr, r):
            return arr, cam, cfg, Gw, r
    raise AssertionError("no suitable seed")


def test_p6_fd_ewa_pinhole_general():
    def make(seed):
        w2c = scenes.look_at((0.3, -0.2, -1.0), (0.0, 0.1, 3.0)).astype(np.float64)
        co = cam_obj(w2c=w2c, cx=19.0, cy=13.5, fy=66.0)
        arr = draw_scene(100 + seed, 6, 16, z=(1.5, 4.5))
        Gw = np.random.default_rng(seed).normal(0, 1, (co.height, co.width, 3))
        return arr, xo.make_camera(co), xo.make_config(cfg_dict(), fragile_rel=1e-4), Gw

    def need(arr, r):
        fl = r["proj"]["flags"]
        return (r["proj"]["tile_count"] > 0).sum() >= 5 and ((fl >> 3) & 7 != 7).any() and (r["fwd"]["n_contrib"] > 2).any()

    arr, cam, cfg, Gw, _ = find_seed(make, need)
    fd_check(arr, cam, cfg, Gw)


def test_p6_fd_alpha_clamp_and_early_exit_active():
    # opaque, large Gaussians: min(0.99, .) active (C14: true derivative is zero there) and the
    # transmittance exit fires (C15: no gradient through the exit)
    def make(seed):
        co = cam_obj()
        arr = draw_scene(300 + seed, 8, 4, z=(2.0, 4.0), xy=0.3, ls=(-0.9, 0.2), opac_boost=7.0)
        Gw = np.random.default_rng(seed).normal(0, 1, (co.height, co.width, 3))
        return arr, xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=1), fragile_rel=1e-4), Gw

    def need(arr, r):
        f = r["fwd"]
        tiles_max = (r["binned"]["ranges"][:, 1] - r["binned"]["ranges"][:, 0]).max()
        exited = (f["final_T"] < 0.011).any() and (f["n_contrib"] < tiles_max).any()
        p = r["proj"]
        d = np.array([20.5, 12.5]) - p["mean2d"]
        G = np.exp(-0.5 * (p["conic"][:, 0] * d[:, 0] ** 2 + p["conic"][:, 2] * d[:, 1] ** 2) - p["conic"][:, 1] * d[:, 0] * d[:, 1])
        return exited and (p["opac_eff"] * G > 0.99).any()

    arr, cam, cfg, Gw, _ = find_seed(make, need)
    fd_check(arr, cam, cfg, Gw)


def test_p6_fd_jacobian_clamp_active():
    # a big primitive far off-axis: x/z outside the C6 limit, zero slope through the clamp (C16)
    def make(seed):
        co = cam_obj(W=32, H=32, fx=20.0, fy=20.0)
        arr = draw_scene(500 + seed, 3, 1, z=(1.0, 1.5), xy=0.2, ls=(-1.2, 0.2))
        arr["means"][0] = [1.6, 0.1, 1.2]      # x/z = 1.33 > (16 + 4.8)/20 = 1.04
        arr["scales"][0] = [0.5, 0.4, 0.3]
        arr["means"][1] = [0.1, -1.7, 1.3]
        arr["scales"][1] = [0.4, 0.6, 0.3]
        Gw = np.random.default_rng(seed).normal(0, 1, (co.height, co.width, 3))
        return arr, xo.make_camera(co), xo.make_config(cfg_dict(sh_degree=0), fragile_rel=1e-4), Gw

    def need(arr, r):
        fl = r["proj"]["flags"]
        return (fl[0] & 3) == 3 and (fl[1] & 5) == 5

    arr, cam, cfg, Gw, r = find_seed(make, need)
    g, _, _ = fd_check(arr, cam, cfg, Gw)
    assert np.abs(g["g_means"][0]).max() > 0


@pytest.mark.parametrize("model,antialias", [(0, 0), (0, 1), (1, 1)])
def test_p6_fd_unscented_transform(model, antialias):
    def make(seed):
        w2c = scenes.look_at((0.2, 0.1, -0.5), (0.0, 0.0, 3.0)).astype(np.float64)
        k = (0.04, -0.03, 0.02, -0.01) if model == 1 else (0, 0, 0, 0)
        co = cam_obj(model=model, w2c=w2c, k=k, fx=45.0, fy=45.0)
        arr = draw_scene(700 + seed, 5, 4, z=(1.5, 4.0))
        Gw = np.random.default_rng(seed).normal(0, 1, (co.height, co.width, 3))
        return arr, xo.make_camera(co), xo.make_config(cfg_dict(projection=1, antialias=antialias, sh_degree=1), fragile_rel=1e-4), Gw

    arr, cam, cfg, Gw, _ = find_seed(make, lambda a, r: (r["proj"]["tile_count"] > 0).sum() >= 4)
    fd_check(arr, cam, cfg, Gw, rtol=5e-6)


def test_p6_fd_ewa_antialias():
    def make(seed):
        co = cam_obj()
        arr = draw_scene(900 + seed, 5, 1, z=(2.0, 6.0), ls=(-2.5, 0.5))
        Gw = np.random.default_rng(seed).normal(0, 1, (co.height, co.width, 3))
        return arr, xo.make_camera(co), xo.make_config(cfg_dict(antialias=1, sh_degree=0), fragile_rel=1e-4), Gw

    arr, cam, cfg, Gw, _ = find_seed(make, lambda a, r: (r["proj"]["tile_count"] > 0).sum() >= 4)
    fd_check(arr, cam, cfg, Gw)


def test_p11_linearity_and_exact_zero_for_culled():
    sc = scenes.make_scene(1)
    arr = dict(means=sc.means.astype(np.float64).copy(), scales=sc.scales.astype(np.float64), quats=sc.quats.astype(np.float64),
               opacities=sc.opacities.astype(np.float64), sh=sc.sh.astype(np.float64))
    arr["means"][7] = [0, 0, -10.0]          # behind the camera -> culled
    arr["means"][11] = [50.0, 0, 0.0]        # off screen
    cam = xo.make_camera(sc.cameras[0]); cfg = xo.make_config(scenes.default_render_config(sc))
    r = xo.render(arr, cam, cfg, np.float64)
    rng = np.random.default_rng(1)
    G1, G2 = rng.normal(0, 1, (64, 64, 3)), rng.normal(0, 1, (64, 64, 3))
    g1, g2 = xo.backward(arr, r, G1, cam, cfg, np.float64), xo.backward(arr, r, G2, cam, cfg, np.float64)
    g12 = xo.backward(arr, r, 2.0 * G1 - 3.0 * G2, cam, cfg, np.float64)
    for k in g1:
        np.testing.assert_allclose(g12[k], 2.0 * g1[k] - 3.0 * g2[k], rtol=1e-9, atol=1e-9 * np.abs(g1[k]).max())
        for i in (7, 11):
            assert (g1[k][i] == 0).all()
    # fp32 parity mode backward agrees with the fp64 one away from fragile pixels (same formulas,
    # forward quantities rounded to fp32)
    arr32 = {k: v.astype(np.float32) for k, v in arr.items()}
    r32 = xo.render(arr32, cam, cfg, np.float32)
    mask = ((r32["fwd"]["fragile"] | r["fwd"]["fragile"]) == 0)[..., None]
    b32 = xo.backward(arr32, r32, (G1 * mask).astype(np.float32), cam, cfg, np.float32)
    b64 = xo.backward(arr, r, G1 * mask, cam, cfg, np.float64)
    for k in ("g_means", "g_sh", "g_opacities"):
        np.testing.assert_allclose(b32[k], b64[k], rtol=2e-2, atol=2e-3 * np.abs(b64[k]).max())


def test_gradient_mass_bounds_gradient_and_equals_it_for_sign_definite_terms():
    """The mass output (sum over pixels of |term|, used only as the scale of the fp32 summation
    tolerance) must dominate |gradient| element-wise, and for g_rgb with dL >= 0 every term
    alpha T g is non-negative, so mass == gradient there (c = sum c_i alpha_i T_i)."""
    sc = scenes.make_scene(1, n_override=300)
    cam = xo.make_camera(sc.cameras[0])
    cfg = xo.make_config(scenes.default_render_config(sc))
    arrays = dict(means=sc.means, scales=sc.scales, quats=sc.quats, opacities=sc.opacities, sh=sc.sh)
    r = xo.render(arrays, cam, cfg, np.float64)
    rng = np.random.default_rng(5)
    dL = rng.standard_normal((64, 64, 3))
    g = xo.rasterize_bwd(r["proj"], r["binned"], r["fwd"], dL, cam, cfg, np.float64)
    m = xo.rasterize_bwd(r["proj"], r["binned"], r["fwd"], dL, cam, cfg, np.float64, mass=True)
    for k in ("g_mean2d", "g_conic", "g_opac_eff", "g_rgb"):
        assert (m[k] >= np.abs(g[k]) * (1 - 1e-12) - 1e-300).all(), k
        assert (m[k] > np.abs(g[k]) * 1.01).any(), k          # cancellation really occurs
    gp = xo.rasterize_bwd(r["proj"], r["binned"], r["fwd"], np.abs(dL), cam, cfg, np.float64)
    mp = xo.rasterize_bwd(r["proj"], r["binned"], r["fwd"], np.abs(dL), cam, cfg, np.float64, mass=True)
    np.testing.assert_allclose(mp["g_rgb"], gp["g_rgb"], rtol=1e-13, atol=0)
    np.testing.assert_allclose(m["g_rgb"], gp["g_rgb"], rtol=1e-13, atol=0)   # mass depends on |dL| only


def test_p6_fd_batch_of_views_is_the_gradient_of_the_summed_loss():
    """Batch of views (Table 2): the loss of a batch is the sum of the views' losses, so its gradient is
    pinned by central finite differences of that SUM through two forwards with different cameras (never by adding up
    backward formulas)."""
    def make(seed):
        cams = [xo.make_camera(cam_obj(w2c=scenes.look_at(e, (0.0, 0.1, 3.0)).astype(np.float64), cx=19.0, cy=13.5))
                for e in ((0.3, -0.2, -1.0), (-0.6, 0.3, -0.4))]
        arr = draw_scene(2100 + seed, 5, 4, z=(1.5, 4.5))
        Gws = [np.random.default_rng(10 * seed + v).normal(0, 1, (24, 40, 3)) for v in range(2)]
        return arr, cams, xo.make_config(cfg_dict(sh_degree=1), fragile_rel=1e-4), Gws

    for seed in range(40):
        arr, cams, cfg, Gws = make(seed)
        rs = xo.render_views(arr, cams, cfg, np.float64)
        if all((r["fwd"]["fragile"] == 0).all() and (r["proj"]["tile_count"] > 0).sum() >= 4 for r in rs):
            break
    else:
        raise AssertionError("no suitable seed")
    loss = lambda a: sum(float((r["fwd"]["image"] * G).sum()) for r, G in zip(xo.render_views(a, cams, cfg, np.float64), Gws))
    g = xo.backward_views(arr, rs, Gws, cams, cfg, np.float64)
    names = dict(means="g_means", scales="g_scales", quats="g_quats", opacities="g_opacities", sh="g_sh")
    scale_all = max(np.abs(g[n]).max() for n in names.values())
    for k, n in names.items():
        base, an = arr[k], g[n]
        it = np.nditer(base, flags=["multi_index"])
        for _ in it:
            idx = it.multi_index
            h = 1e-6 * max(1.0, abs(base[idx])) if k != "scales" else 1e-5 * abs(base[idx])
            ap = {kk: v.copy() for kk, v in arr.items()}; ap[k][idx] += h
            am = {kk: v.copy() for kk, v in arr.items()}; am[k][idx] -= h
            fd = (loss(ap) - loss(am)) / (2 * h)
            assert abs(fd - an[idx]) <= 2e-6 * max(abs(fd), abs(an[idx])) + 1e-7 * scale_all + 1e-9, (k, idx, fd, an[idx])
