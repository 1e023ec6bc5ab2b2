"""GPU parity of the rendered features (Table 2; reading C31):
xpr_rasterize_feat_fwd / xpr_rasterize_feat_bwd / xpr_depth_bwd through the C-ABI binding against the CPU oracle
(xpr_oracle_feat.inc, pinned by P15) on the same seeded inputs.

Bars: colour image, final_T, n_contrib as the colour pass (1e-4 max abs; n_contrib bit-exact outside fragile
pixels); accumulated opacity A within 1e-4 max abs; depth image D within 1e-4 * max(1, z_max) -- D is the colour
blend with c := z, so its error scales with the largest depth on the lists; compositing gradients,
g_depth included, every element within 1e-3 |ref| + 1e-6 + 2e-6 * mass; parameter gradients strict against the
oracle's project_bwd + depth_bwd fed the same fp32 2D gradients.
"""
import numpy as np
import pytest

import parity_util as pu
import xpr_oracle as xo
from paper_2606_11529_b200 import scenes

pytestmark = pytest.mark.gpu

PAIRS = (("g_mean2d", "g_mean2d"), ("g_conic", "g_conic"), ("g_opac", "g_opac_eff"), ("g_rgb", "g_rgb"),
         ("g_depth", "g_depth"))
PARAMS = ("g_means", "g_scales", "g_quats", "g_opacities", "g_sh")


def feat_grads(scene, view, shape):
    """Seeded dL/dD and dL/dA (a loss 'sum gD * D + sum gA * A'); the colour gradient is the config's own loss."""
    rng = np.random.default_rng(4000 + 7 * scene.N % 1000 + view)
    gD = rng.uniform(-1.0, 1.0, shape).astype(np.float32)
    gA = rng.uniform(-1.0, 1.0, shape).astype(np.float32)
    return gD, gA


def feat_parity(scene, view=0, cfg_over=None):
    import torch
    over = dict(features=1)
    if cfg_over:
        over.update(cfg_over)
    g = pu.run_gpu(scene, view, over)
    pipe = g["pipe"]
    o = pu.run_oracle(scene, view, cfg_over)
    pu.compare_projection(g, o)
    pu.compare_binning(g, o)
    pu.compare_forward(g, o)                      # colour, final_T, n_contrib of the fused kernel
    of = xo.rasterize_fwd_da(o["proj"], o["binned"], o["cam"], o["cfg"], np.float32)
    ok = (o["fwd"]["fragile"] & pu.FRAG_EXIT) == 0
    A_gpu, D_gpu = pipe.alpha_img.cpu().numpy(), pipe.depth_img.cpu().numpy()
    errA = np.abs(A_gpu.astype(np.float64) - of["alpha_img"])
    assert errA[ok].max(initial=0.0) <= pu.IMG_TOL, errA[ok].max()
    vis = o["proj"]["tile_count"] > 0
    zmax = max(1.0, float(o["proj"]["depth"][vis].max(initial=1.0)))
    errD = np.abs(D_gpu.astype(np.float64) - of["depth_img"])
    assert errD[ok].max(initial=0.0) <= pu.IMG_TOL * zmax, (errD[ok].max(), zmax)
    # invariant at any size: A = 1 - T_final up to fp32 summation
    assert np.abs(A_gpu + g["fwd"]["final_T"] - 1.0).max() <= 1e-4

    H, W = ok.shape
    _, dL = scenes.loss_and_grad(scene.loss, o["fwd"]["image"], scene.target(view))
    gD, gA = feat_grads(scene, view, (H, W))
    frag = (o["fwd"]["fragile"] & (pu.FRAG_EXIT | pu.FRAG_CLAMP)) != 0
    dL = np.where(frag[..., None], 0.0, dL).astype(np.float32)
    gD = np.where(frag, 0.0, gD).astype(np.float32); gA = np.where(frag, 0.0, gA).astype(np.float32)
    args = (o["proj"], o["binned"], o["fwd"], dL, gD, gA, o["cam"], o["cfg"], np.float32)
    og2 = xo.rasterize_bwd_da(*args)
    mass = xo.rasterize_bwd_da(*args, mass=True)
    dev = pipe.device
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    pipe.backward(t(dL), t(gD), t(gA))
    torch.cuda.synchronize()
    gg = {k: getattr(pipe, k).cpu().numpy() for k in [p[0] for p in PAIRS] + list(PARAMS)}
    for kg, ko in PAIRS:                                       # compositing, every element
        bad, err = pu.grad_violations(gg[kg], og2[ko], mass[ko])
        assert bad.sum() == 0, f"{kg}: {bad.sum()} of {bad.size} outside tolerance, max err {err.max()}"
    assert np.abs(og2["g_depth"]).max() > 0
    # parameters: the oracle's project_bwd + depth_bwd fed the GPU's own fp32 2D gradients (stage isolation)
    g2 = dict(g_mean2d=gg["g_mean2d"], g_conic=gg["g_conic"], g_opac_eff=gg["g_opac"], g_rgb=gg["g_rgb"])
    iso = xo.project_bwd(scene.means, scene.scales, scene.quats, scene.opacities, scene.sh, o["cam"], o["cfg"], g2,
                         np.float32)
    iso["g_means"] = iso["g_means"] + xo.depth_bwd(o["proj"]["tile_count"], gg["g_depth"], o["cam"])
    for k in PARAMS:
        bad, err = pu.grad_violations(gg[k], iso[k])
        assert bad.sum() == 0, f"{k} (stage-isolated): {bad.sum()} of {bad.size}, max err {err.max()}"
    culled = ~vis
    for k in PARAMS:
        assert not np.any(gg[k][culled])
    return g, o


def test_feat_config1_tiny():
    feat_parity(scenes.make_scene(1))


def test_feat_config2_reduced():
    feat_parity(scenes.make_scene(2, n_override=20000, image_override=(200, 200)))


@pytest.mark.parametrize("view", [0, 1])
def test_feat_config3_reduced(view):
    feat_parity(scenes.make_scene(3, n_override=50000, image_override=(480, 270)), view)


@pytest.mark.parametrize("wh", [(70, 50), (33, 17)])
def test_feat_ragged(wh):
    feat_parity(scenes.make_scene(1, image_override=wh))


def test_feat_background_and_tile_cull():
    feat_parity(scenes.make_scene(2, n_override=20000, image_override=(200, 200)), 0,
                dict(bg=(0.2, 0.5, 0.9), tile_cull=1))


def test_feat_config3_full_size_throughput_shape():
    # 8160 tiles: the 2-pixels-per-thread forward and the 4-pixels-per-thread backward (the launch shape of the bench)
    feat_parity(scenes.make_scene(3), 0, dict(tile_cull=1))


def test_feat_zero_feature_gradients_reduce_to_colour_backward():
    import torch
    sc = scenes.make_scene(2, n_override=20000, image_override=(200, 200))
    g = pu.run_gpu(sc, 0, dict(features=1))
    pipe = g["pipe"]
    rng = np.random.default_rng(7)
    dL = torch.from_numpy(rng.uniform(-1, 1, (200, 200, 3)).astype(np.float32)).to(pipe.device)
    z = torch.zeros(200, 200, device=pipe.device)
    pipe.backward(dL, z, z)
    a = {k: getattr(pipe, k).clone() for k in PARAMS}
    assert not bool(pipe.g_depth.any())
    pipe.backward(dL)                       # the colour kernel
    for k in PARAMS:
        ref = getattr(pipe, k)
        # two kernels, two orders of fp32 atomics: a sanity bound (the element-wise bars are in feat_parity)
        assert bool(((a[k] - ref).abs() <= 2e-3 * ref.abs() + 1e-4 * ref.abs().max()).all()), k


def test_feat_everything_culled():
    import torch
    sc = scenes.make_scene(1, n_override=500)
    sc.means[:, 2] -= 10.0          # all behind the camera
    g = pu.run_gpu(sc, 0, dict(features=1, bg=(0.1, 0.2, 0.3)))
    pipe = g["pipe"]
    assert g["binned"]["num_pairs"] == 0
    assert not bool(pipe.depth_img.any()) and not bool(pipe.alpha_img.any())
    assert torch.all(pipe.final_T == 1.0)
    one = torch.ones(64, 64, device=pipe.device)
    pipe.backward(torch.ones(64, 64, 3, device=pipe.device), one, one)
    for k in PARAMS + ("g_depth",):
        assert not bool(getattr(pipe, k).any()), k


# ---- N-channel features (xpr_rasterize_featn_fwd / _bwd) against the oracle (pin P16) ----------------------------

FLOOR_REL = 2e-5      # group-relative fp32 summation floor of the geometric gradients


def featn_parity(scene, Cn, view=0, cfg_over=None, with_colour=True):
    import torch
    g = pu.run_gpu(scene, view, cfg_over)
    pipe = g["pipe"]
    o = pu.run_oracle(scene, view, cfg_over)
    pu.compare_binning(g, o)
    pu.compare_forward(g, o)
    rng = np.random.default_rng(5000 + Cn + view)
    feat = rng.normal(0.0, 1.0, (scene.N, Cn)).astype(np.float32)
    H, W = o["fwd"]["n_contrib"].shape
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(pipe.device)
    F_gpu = pipe.rasterize_featn_fwd(t(feat)).cpu().numpy()
    F_ref = xo.rasterize_fwd_featn(o["proj"], o["binned"], feat, o["cam"], o["cfg"], np.float32)
    ok = (o["fwd"]["fragile"] & pu.FRAG_EXIT) == 0
    fmax = max(1.0, float(np.abs(feat).max()))
    err = np.abs(F_gpu.astype(np.float64) - F_ref).max(axis=2)
    assert err[ok].max(initial=0.0) <= pu.IMG_TOL * fmax, (err[ok].max(), fmax)      # |F| <= max|feat| (1 - T)
    assert np.abs(F_ref).max() > 0.1

    gF = rng.uniform(-1.0, 1.0, (H, W, Cn)).astype(np.float32)
    frag = (o["fwd"]["fragile"] & (pu.FRAG_EXIT | pu.FRAG_CLAMP)) != 0
    gF = np.where(frag[..., None], 0.0, gF).astype(np.float32)
    ref = xo.rasterize_bwd_featn(o["proj"], o["binned"], o["fwd"], feat, gF, o["cam"], o["cfg"], np.float32)
    # mass of every element = the same backward with |gF| and |feat| ... not available as a variant: bound it by the
    # oracle run on (|feat|, |gF|) for g_feat (sign-definite terms) and use the group scale for the geometric parts
    if with_colour:
        _, dL = scenes.loss_and_grad(scene.loss, o["fwd"]["image"], scene.target(view))
        dL = np.where(frag[..., None], 0.0, dL).astype(np.float32)
        col = xo.rasterize_bwd(o["proj"], o["binned"], o["fwd"], dL, o["cam"], o["cfg"], np.float32)
        mass = xo.rasterize_bwd(o["proj"], o["binned"], o["fwd"], dL, o["cam"], o["cfg"], np.float32, mass=True)
        pipe.rasterize_bwd(t(dL))
        g_feat = pipe.rasterize_featn_bwd(t(feat), t(gF))
    else:
        col = {k: 0.0 for k in ("g_mean2d", "g_conic", "g_opac_eff")}
        mass = {k: 0.0 for k in ("g_mean2d", "g_conic", "g_opac_eff")}
        g_feat = pipe.rasterize_featn_bwd(t(feat), t(gF), first=True)
    torch.cuda.synchronize()
    # g_feat: sums of alpha T gF over pixels; mass = the same sum with |gF|
    m = xo.rasterize_bwd_featn(o["proj"], o["binned"], o["fwd"], feat, np.abs(gF), o["cam"], o["cfg"], np.float32)
    bad, e = pu.grad_violations(g_feat.cpu().numpy(), ref["g_feat"], m["g_feat"])
    assert bad.sum() == 0, f"g_feat: {bad.sum()} of {bad.size}, max err {e.max()}"
    assert np.abs(ref["g_feat"]).max() > 0
    # geometric parts: colour part + feature part; the fp32 summation floor is taken relative to the Gaussian's
    # largest component of that gradient among the two parts (cancellation-aware, DESIGN.md 5 / 6.8)
    for kg, ko in (("g_mean2d", "g_mean2d"), ("g_conic", "g_conic"), ("g_opac", "g_opac_eff")):
        total = np.asarray(ref[ko] + col[ko], np.float64).reshape(scene.N, -1)
        floor = (np.abs(np.asarray(ref[ko]).reshape(scene.N, -1)).max(axis=1, keepdims=True)
                 + np.abs(np.asarray(col[ko] if with_colour else 0.0 * total).reshape(scene.N, -1)).max(axis=1, keepdims=True))
        got = getattr(pipe, kg).cpu().numpy().reshape(scene.N, -1).astype(np.float64)
        tol = pu.GRAD_RTOL * np.abs(total) + pu.GRAD_ATOL + FLOOR_REL * floor
        if with_colour:
            tol = tol + pu.GRAD_KAPPA * np.asarray(mass[ko]).reshape(scene.N, -1)
        worst = np.abs(got - total) - tol
        assert (worst <= 0).all(), f"{kg}: {(worst > 0).sum()} of {worst.size} outside tolerance, max excess {worst.max()}"
    return pipe


@pytest.mark.parametrize("Cn", [1, 3, 8, 13])
def test_featn_config1(Cn):
    featn_parity(scenes.make_scene(1), Cn)


def test_featn_config2_reduced_alone():
    featn_parity(scenes.make_scene(2, n_override=20000, image_override=(200, 200)), 5, with_colour=False)


@pytest.mark.parametrize("view", [0, 1])
def test_featn_config3_reduced(view):
    featn_parity(scenes.make_scene(3, n_override=50000, image_override=(480, 270)), 16, view, dict(tile_cull=1))


def test_featn_ragged():
    featn_parity(scenes.make_scene(1, image_override=(70, 50)), 4)


def test_featn_three_channels_of_rgb_are_the_colour_image():
    import torch
    sc = scenes.make_scene(2, n_override=20000, image_override=(200, 200))
    g = pu.run_gpu(sc, 0, dict(bg=(0.0, 0.0, 0.0)))
    pipe = g["pipe"]
    F = pipe.rasterize_featn_fwd(pipe.rgb)
    assert float((F - pipe.image).abs().max()) <= 1e-6


def test_featn_config3_full_size():
    featn_parity(scenes.make_scene(3), 8, 0, dict(tile_cull=1))
