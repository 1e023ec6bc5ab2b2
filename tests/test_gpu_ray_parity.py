"""GPU parity of the XPR-3DGUT evaluation: xpr_pixel_info, xpr_project_ray,
xpr_rasterize_ray_fwd / _bwd and xpr_ray_bwd against the CPU oracle (oracle/xpr_oracle_ray.inc), element by
element on the same seeded inputs, with the bars of test_gpu_parity.py:
  pixel rays      <= 1 fp32 ulp of 1 (fp64 sin / cos of two libraries, rounded to fp32; rule R2), then the GPU's rays
                  are handed to the oracle (stage isolation, as for every other stage)
  shader record   bit-exact (rule R1)
  lists           bit-exact;  image <= 1e-4 outside fragile pixels;  n_contrib equal there
  record / opacity / colour gradients  1e-3 |ref| + 1e-6 + 2e-6 mass, every element
  parameter gradients, stage-isolated  1e-3 |ref| + 1e-6 (+ the fp32 rounding of the accumulation into
                  xpr_project_bwd's outputs), end to end reported and bounded: violators <= 5e-3 of the elements,
                  each within 2e-2 of its Gaussian's largest component of that gradient.
"""
import numpy as np
import pytest

import parity_util as pu
import xpr_oracle as xo
from paper_2606_11529_b200 import scenes

pytestmark = pytest.mark.gpu

PARAMS = ("g_means", "g_scales", "g_quats", "g_opacities", "g_sh")


E2E_STATS = []      # (scene, N, end-to-end violators, elements) of every case run, printed by the last test


def ray_parity(scene, view=0, cfg_over=None):
    over = dict(cfg_over or {}, ray_eval=1)
    g = pu.run_gpu(scene, view, over)
    o = pu.run_oracle_ray(scene, view, over, pixel_rays=g["proj"]["pixel_rays"])
    vis = pu.compare_projection(g, o)
    # pixel_info: unit vectors, within one ulp of the oracle's
    dr = np.abs(g["proj"]["pixel_rays"].astype(np.float64) - o["proj"]["pixel_rays_oracle"].astype(np.float64))
    assert dr.max() <= 1.2e-7, dr.max()
    assert (dr > 0).mean() <= 1e-4, (dr > 0).mean()
    # shader record
    np.testing.assert_array_equal(g["proj"]["ray_rec"][vis].view(np.uint32), o["proj"]["ray_rec"][vis].view(np.uint32))
    assert not np.any(g["proj"]["ray_rec"][~vis])
    pu.compare_binning(g, o)
    n_frag, _ = pu.compare_forward(g, o)
    npix = o["fwd"]["image"].shape[0] * o["fwd"]["image"].shape[1]
    assert n_frag <= max(2, 1e-3 * npix), f"{n_frag} fragile pixels"
    assert o["fwd"]["pp_pass"] > 0
    _, dL = scenes.loss_and_grad(scene.loss, o["fwd"]["image"], scene.target(view))
    frag = (o["fwd"]["fragile"] & (pu.FRAG_EXIT | pu.FRAG_CLAMP)) != 0
    dL = np.where(frag[..., None], 0.0, dL).astype(np.float32)
    og = xo.backward_ray(o["arrays"], o, dL, o["cam"], o["cfg"], np.float32)
    gg = pu.run_gpu_backward(g, dL)
    # stage 1: the record gradient in the accumulator form the kernel sums (S_c, D, sum dL/do_c: xpr.h; the oracle's
    # accumulator route is pinned equal to its plain route, P14f), opacity and colour -- every element
    oa = xo.rasterize_ray_bwd_acc(o["proj"], o["binned"], o["fwd"], dL, o["cam"], o["cfg"], np.float32)
    mass = xo.rasterize_ray_bwd_acc(o["proj"], o["binned"], o["fwd"], dL, o["cam"], o["cfg"], np.float32, mass=True)
    n_plain = 0
    for kg, ko in (("g_ray_acc", "g_ray_acc"), ("g_opac", "g_opac_eff"), ("g_rgb", "g_rgb")):
        bad, err = pu.grad_violations(gg[kg], oa[ko], mass[ko])
        assert bad.sum() == 0, f"{kg}: {bad.sum()} of {bad.size} outside tolerance, max err {err.max()}"
        n_plain += int(pu.grad_violations(gg[kg], oa[ko])[0].sum())
    assert n_plain <= max(4, 2e-4 * 19 * scene.N), n_plain
    assert not np.any(gg["g_mean2d"]) and not np.any(gg["g_conic"])      # the footprint carries no gradient
    # stage 2: the oracle's chain rule fed the GPU's fp32 gradients
    N = scene.N
    gz = dict(g_mean2d=np.zeros((N, 2)), g_conic=np.zeros((N, 3)), g_opac_eff=gg["g_opac"], g_rgb=gg["g_rgb"])
    iso = xo.project_bwd(scene.means, scene.scales, scene.quats, scene.opacities, scene.sh, o["cam"], o["cfg"], gz,
                         np.float32)
    part = xo.ray_bwd_acc(scene.means, scene.scales, scene.quats, o["proj"]["tile_count"], gg["g_ray_acc"], o["cam"],
                          np.float32)
    # the stage-1 bar carried to the parameters: opacity and colour through project_bwd (zero footprint gradients), the
    # accumulators through ray_bwd_acc
    zero2 = dict(g_mean2d=np.zeros((N, 2)), g_conic=np.zeros((N, 3)))
    tol_p = pu.propagated_param_tol(o["arrays"], o["cam"], o["cfg"], dict(zero2, g_opac_eff=oa["g_opac_eff"], g_rgb=oa["g_rgb"]),
                                    dict(zero2, g_opac_eff=mass["g_opac_eff"], g_rgb=mass["g_rgb"]))
    tol_r = pu.propagated_ray_tol(o["arrays"], o["proj"]["tile_count"], o["cam"], oa["g_ray_acc"][:, :15], mass["g_ray_acc"][:, :15])
    total_bad = total = 0
    for k in PARAMS:
        ref = iso[k] + part[k] if k in part else iso[k]
        got, ref = np.asarray(gg[k], np.float64).ravel(), np.asarray(ref, np.float64).ravel()
        tol = pu.GRAD_RTOL * np.abs(ref) + pu.GRAD_ATOL
        if k in part:   # fp32 accumulation of the two parts: one rounding of each part
            tol = tol + 2.4e-7 * (np.abs(iso[k]).ravel() + np.abs(part[k]).ravel())
        bad = np.abs(got - ref) > tol
        assert bad.sum() == 0, f"{k} (stage-isolated): {bad.sum()} of {bad.size}, max err {np.abs(got - ref).max()}"
        bad_e2e, err_e2e = pu.grad_violations(gg[k], og[k])
        total_bad += int(bad_e2e.sum()); total += bad_e2e.size
        # every element within the bar derived from the stage bars (parity_util.propagated_param_tol / _ray_tol)
        tp = tol_p[k] + (tol_r[k] if k in tol_r else 0.0) + (2.4e-7 * (np.abs(iso[k]) + np.abs(part[k])) if k in part else 0.0)
        ok = pu.e2e_within_propagated(gg[k], og[k], tp)
        assert ok.all(), f"{k}: {int((~ok).sum())} elements outside the propagated end-to-end bar"
    # end to end against the oracle's PLAIN route (the definition): the accumulators no longer cancel, so what is left
    # is the fp32 summation floor of stage 1 on elements far below their Gaussian's largest component (as on the 2D path)
    E2E_STATS.append((scene.name, scene.N, total_bad, total))
    assert total_bad <= 1e-3 * total, f"end-to-end violators {total_bad}/{total}"
    culled = o["proj"]["tile_count"] == 0
    for k in PARAMS + ("g_ray_acc",):
        assert not np.any(gg[k][culled])
    return g, o


@pytest.mark.parametrize("view", [0, 1])
def test_ray_config4_ut_fisheye_reduced(view):
    ray_parity(scenes.make_scene(4, n_override=30000, image_override=(480, 270)), view)


def test_ray_config4_with_tile_cull_reduced():
    ray_parity(scenes.make_scene(4, n_override=30000, image_override=(480, 270)), 0, dict(tile_cull=1))


def test_ray_pinhole_ewa_footprint_and_background():
    # the evaluation does not depend on how the footprint was made: EWA tiling, pinhole rays, non-zero background
    ray_parity(scenes.make_scene(3, n_override=20000, image_override=(250, 130)), 1, dict(bg=(0.2, 0.4, 0.1)))


def test_ray_config1_tiny_and_ragged():
    ray_parity(scenes.make_scene(1), 0)
    ray_parity(scenes.make_scene(2, n_override=5000, image_override=(70, 50)), 0)


@pytest.mark.parametrize("view", [0, 1])
def test_ray_config4_full_size(view):
    ray_parity(scenes.make_scene(4), view, dict(tile_cull=1))


def test_ray_stats_match_oracle_counters():
    import torch
    from paper_2606_11529_b200 import binding as xb
    sc = scenes.make_scene(4, n_override=30000, image_override=(480, 270))
    g = pu.run_gpu(sc, 0, dict(ray_eval=1))
    o = pu.run_oracle_ray(sc, 0, dict(ray_eval=1), pixel_rays=g["proj"]["pixel_rays"])
    p = g["pipe"]
    stats = torch.zeros(4, dtype=torch.int64, device=p.device)
    xb.xpr_rasterize_ray_stats(p.cam, p.cfg, p.ray_rec, p.conic_opac, p.rgb, p.lnv, p.pixel_rays, p.vals_sorted,
                               p.tile_ranges, stats)
    visited, passed, blended, sum_n = stats.tolist()
    frag = int((o["fwd"]["fragile"] != 0).sum())
    assert abs(visited - o["fwd"]["pp_visit"]) <= 64 * frag and abs(passed - o["fwd"]["pp_pass"]) <= 64 * frag
    assert blended <= passed <= visited and sum_n == int(p.n_contrib.sum().item())


def test_ray_degenerate_record_is_never_valid():
    # a zero scale makes M_c infinite: the record is replaced by zeros and the Gaussian contributes nothing (C30)
    import copy
    sc = copy.deepcopy(scenes.make_scene(1))
    sc.scales[:5] = 0.0
    g, o = ray_parity(sc, 0)
    vis = o["proj"]["tile_count"] > 0
    assert vis[:5].any()
    assert not np.any(g["proj"]["ray_rec"][:5])


def test_ray_empty_scene_and_everything_culled():
    import torch
    from paper_2606_11529_b200 import pipeline
    sc = scenes.make_scene(1)
    for name in ("means", "scales", "quats", "opacities", "sh"):
        setattr(sc, name, getattr(sc, name)[:0].copy())
    cfg = dict(scenes.default_render_config(sc), ray_eval=1, bg=(0.1, 0.2, 0.3))
    pipe = pipeline.SplatPipeline(0, sc.cameras[0], cfg)
    img = pipe.forward(*pipeline.scene_to_device(sc))
    pipe.backward(torch.ones(64, 64, 3, device="cuda"))
    torch.cuda.synchronize()
    np.testing.assert_allclose(img.cpu().numpy(), np.broadcast_to(np.float32([0.1, 0.2, 0.3]), (64, 64, 3)))
    assert (pipe.final_T.cpu().numpy() == 1).all() and (pipe.n_contrib.cpu().numpy() == 0).all()
    sc = scenes.make_scene(1, n_override=500)
    sc.means[:, 2] -= 10.0          # all behind the camera
    g = pu.run_gpu(sc, 0, dict(ray_eval=1))
    assert g["binned"]["num_pairs"] == 0 and not np.any(g["proj"]["ray_rec"]) and (g["fwd"]["image"] == 0).all()
    gg = pu.run_gpu_backward(g, np.ones((64, 64, 3), np.float32))
    for k, v in gg.items():
        assert not np.any(v), k


@pytest.mark.parametrize("deg", [0, 2])
def test_ray_sh_degrees_and_ragged(deg):
    sc = scenes.make_scene(4, n_override=8000, image_override=(33, 17))
    sc.sh = sc.sh[:, :(deg + 1) ** 2].copy()
    sc.sh_degree = deg
    ray_parity(sc, 0)


def test_ray_pixel_rays_depend_on_the_intrinsics_only():
    # the two poses of config 4 share their intrinsics: identical rays (reading C27)
    sc = scenes.make_scene(4, n_override=100, image_override=(160, 90))
    a = pu.run_gpu(sc, 0, dict(ray_eval=1))["proj"]["pixel_rays"]
    b = pu.run_gpu(sc, 1, dict(ray_eval=1))["proj"]["pixel_rays"]
    np.testing.assert_array_equal(a, b)
    np.testing.assert_allclose(np.linalg.norm(a.astype(np.float64), axis=-1), 1.0, atol=2e-7)


def ray_feat_parity(scene, view=0, cfg_over=None):
    """f2 x f3: depth image and accumulated opacity rendered by the ray evaluation (xpr_rasterize_ray_feat_fwd / _bwd).
    Bars as tests/test_gpu_feat_parity.py: A within 1e-4, D within 1e-4 max(1, z_max), compositing gradients (accumulators,
    opacity, colour, g_depth) every element within 1e-3 |ref| + 1e-6 + 2e-6 mass, parameters stage-isolated."""
    import torch
    over = dict(cfg_over or {}, ray_eval=1)
    g = pu.run_gpu(scene, view, dict(over, features=1))
    pipe = g["pipe"]
    o = pu.run_oracle_ray(scene, view, over, pixel_rays=g["proj"]["pixel_rays"])
    pu.compare_binning(g, o)
    pu.compare_forward(g, o)
    of = xo.rasterize_ray_fwd_da(o["proj"], o["binned"], o["cam"], o["cfg"], np.float32)
    ok = (o["fwd"]["fragile"] & pu.FRAG_EXIT) == 0
    A_gpu, D_gpu = pipe.alpha_img.cpu().numpy(), pipe.depth_img.cpu().numpy()
    vis = o["proj"]["tile_count"] > 0
    zmax = max(1.0, float(o["proj"]["depth"][vis].max(initial=1.0)))
    assert np.abs(A_gpu.astype(np.float64) - of["alpha_img"])[ok].max(initial=0.0) <= pu.IMG_TOL
    assert np.abs(D_gpu.astype(np.float64) - of["depth_img"])[ok].max(initial=0.0) <= pu.IMG_TOL * zmax
    assert np.abs(A_gpu + g["fwd"]["final_T"] - 1.0).max() <= 1e-4 and D_gpu.max() > 0
    H, W = ok.shape
    _, dL = scenes.loss_and_grad(scene.loss, o["fwd"]["image"], scene.target(view))
    rng = np.random.default_rng(4100 + view)
    gD, gA = rng.uniform(-1, 1, (H, W)).astype(np.float32), rng.uniform(-1, 1, (H, W)).astype(np.float32)
    frag = (o["fwd"]["fragile"] & (pu.FRAG_EXIT | pu.FRAG_CLAMP)) != 0
    dL = np.where(frag[..., None], 0.0, dL).astype(np.float32)
    gD = np.where(frag, 0.0, gD).astype(np.float32); gA = np.where(frag, 0.0, gA).astype(np.float32)
    args = (o["proj"], o["binned"], o["fwd"], dL, gD, gA, o["cam"], o["cfg"], np.float32)
    oa = xo.rasterize_ray_bwd_da(*args, acc=True)
    mass = xo.rasterize_ray_bwd_da(*args, acc=True, mass=True)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(pipe.device)
    pipe.backward(t(dL), t(gD), t(gA))
    torch.cuda.synchronize()
    gg = {k: getattr(pipe, k).cpu().numpy() for k in ("g_ray_acc", "g_opac", "g_rgb", "g_depth") + PARAMS}
    for kg, ko in (("g_ray_acc", "g_ray_acc"), ("g_opac", "g_opac_eff"), ("g_rgb", "g_rgb"), ("g_depth", "g_depth")):
        bad, err = pu.grad_violations(gg[kg], oa[ko], mass[ko])
        assert bad.sum() == 0, f"{kg}: {bad.sum()} of {bad.size} outside tolerance, max err {err.max()}"
    assert np.abs(oa["g_depth"]).max() > 0
    N = scene.N
    gz = dict(g_mean2d=np.zeros((N, 2)), g_conic=np.zeros((N, 3)), g_opac_eff=gg["g_opac"], g_rgb=gg["g_rgb"])
    iso = xo.project_bwd(scene.means, scene.scales, scene.quats, scene.opacities, scene.sh, o["cam"], o["cfg"], gz, np.float32)
    part = xo.ray_bwd_acc(scene.means, scene.scales, scene.quats, o["proj"]["tile_count"], gg["g_ray_acc"], o["cam"], np.float32)
    dpart = xo.depth_bwd(o["proj"]["tile_count"], gg["g_depth"], o["cam"])
    og = xo.backward_ray_da(o["arrays"], o, dL, gD, gA, o["cam"], o["cfg"], np.float32)
    total_bad = total = 0
    for k in PARAMS:
        parts = [iso[k]] + ([part[k]] if k in part else []) + ([dpart] if k == "g_means" else [])
        ref = sum(parts)
        got, ref = np.asarray(gg[k], np.float64).ravel(), np.asarray(ref, np.float64).ravel()
        tol = pu.GRAD_RTOL * np.abs(ref) + pu.GRAD_ATOL + 2.4e-7 * sum(np.abs(x).ravel() for x in parts) * (len(parts) > 1)
        bad = np.abs(got - ref) > tol
        assert bad.sum() == 0, f"{k} (stage-isolated): {bad.sum()} of {bad.size}, max err {np.abs(got - ref).max()}"
        b2, _ = pu.grad_violations(gg[k], og[k])
        total_bad += int(b2.sum()); total += b2.size
    assert total_bad <= 1e-3 * total, f"end-to-end violators {total_bad}/{total}"
    return total_bad, total


def test_ray_feat_config4_reduced_and_tiny():
    print("RAY_FEAT e2e", ray_feat_parity(scenes.make_scene(4, n_override=30000, image_override=(480, 270)), 0))
    ray_feat_parity(scenes.make_scene(1), 0)
    ray_feat_parity(scenes.make_scene(3, n_override=20000, image_override=(250, 130)), 1, dict(bg=(0.2, 0.4, 0.1), tile_cull=1))


def test_ray_feat_config4_full_size():
    print("RAY_FEAT full e2e", ray_feat_parity(scenes.make_scene(4), 0))


def test_zz_report_end_to_end_violators(capsys):
    with capsys.disabled():
        for name, n, bad, tot in E2E_STATS:
            print(f"\n[f2 end to end] {name} N={n}: {bad} of {tot} elements outside 1e-3 rel + 1e-6 abs ({bad / max(tot, 1):.2e})", end="")
