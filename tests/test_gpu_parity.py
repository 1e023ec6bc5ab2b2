"""GPU parity: the CUDA path (through the C-ABI binding) against the CPU oracle, element by element,
on the same seeded inputs.  Bars (BASELINE.json:north_star): tile lists and sorted keys bit-exact,
images within 1e-4 max abs (fp32), gradients within 1e-3 relative + 1e-6 absolute.

Gradient parity is asserted per kernel on identical inputs:
  stage 1  xpr_rasterize_bwd  vs oracle rasterize_bwd            -> every element, tolerance
           1e-3 |ref| + 1e-6 + 2e-6 * mass (mass = sum_pixels |term|, from the oracle)
  stage 2  xpr_project_bwd    vs oracle project_bwd fed the SAME fp32 2D gradients -> strict
and the end-to-end composition is reported (its few violators are elements whose value is
cancelled by the covariance chain rule; they are bounded group-relative: within 1 % of the Gaussian's
largest component of that gradient -- the chain rule G2 = -K G_K K amplifies the fp32 summation floor of
stage 1 by the conditioning of K, and which elements are hit depends on the order of the atomics).
"""
import numpy as np
import pytest

import parity_util as pu
import xpr_oracle as xo
from paper_2606_11529_b200 import scenes

pytestmark = pytest.mark.gpu

PAIRS_2D = (("g_mean2d", "g_mean2d"), ("g_conic", "g_conic"), ("g_opac", "g_opac_eff"), ("g_rgb", "g_rgb"))
PARAMS = ("g_means", "g_scales", "g_quats", "g_opacities", "g_sh")


E2E_STATS = []      # per case: elements outside 1e-3 |ref| + 1e-6 -- 2D stage (GPU, CPU fp32), end to end (GPU, CPU fp32)


def full_parity(scene, view=0, cfg_over=None, expect_pairs=True):
    g = pu.run_gpu(scene, view, cfg_over)
    o = pu.run_oracle(scene, view, cfg_over)
    pu.compare_projection(g, o)
    pu.compare_binning(g, o)
    n_frag, _ = pu.compare_forward(g, o)
    npix = o["fwd"]["image"].shape[0] * o["fwd"]["image"].shape[1]
    assert n_frag <= max(2, 1e-3 * npix), f"{n_frag} fragile pixels"   # reported, never hidden: see compare_forward
    if expect_pairs:
        assert o["binned"]["num_pairs"] > 0
    # backward: dL from the ORACLE image so that both sides get identical inputs
    _, dL = scenes.loss_and_grad(scene.loss, o["fwd"]["image"], scene.target(view))
    frag = (o["fwd"]["fragile"] & (pu.FRAG_EXIT | pu.FRAG_CLAMP)) != 0
    dL = np.where(frag[..., None], 0.0, dL).astype(np.float32)   # fragile pixels carry no gradient on either side
    og = xo.backward(o["arrays"], o, dL, o["cam"], o["cfg"], np.float32)
    gg = pu.run_gpu_backward(g, dL)
    mass = xo.rasterize_bwd(o["proj"], o["binned"], o["fwd"], dL, o["cam"], o["cfg"], np.float32, mass=True)
    n_plain = 0
    for kg, ko in PAIRS_2D:                                       # stage 1, every element
        bad, err = pu.grad_violations(gg[kg], og[ko], mass[ko])
        assert bad.sum() == 0, f"{kg}: {bad.sum()} of {bad.size} outside tolerance, max err {err.max()}"
        n_plain += int(pu.grad_violations(gg[kg], og[ko])[0].sum())
    # without the mass term only cancellation-dominated elements may fail (the oracle's own fp32 and
    # fp64 modes disagree there too): a handful per million
    assert n_plain <= max(4, 2e-5 * 9 * scene.N), n_plain         # measured: 0-2 of 9 M (config 3), 0 of 27 M (config 5), 8 of 0.9 M (config 2)
    g2 = dict(g_mean2d=gg["g_mean2d"], g_conic=gg["g_conic"], g_opac_eff=gg["g_opac"], g_rgb=gg["g_rgb"])
    iso = xo.project_bwd(scene.means, scene.scales, scene.quats, scene.opacities, scene.sh, o["cam"], o["cfg"], g2,
                         np.float32)
    total_bad = total = 0
    tol_p = pu.propagated_param_tol(o["arrays"], o["cam"], o["cfg"], og, mass)     # stage-1 bar carried to the parameters
    for k in PARAMS:
        bad, err = pu.grad_violations(gg[k], iso[k])              # stage 2, strict
        assert bad.sum() == 0, f"{k} (stage-isolated): {bad.sum()} of {bad.size}, max err {err.max()}"
        bad_e2e, err_e2e = pu.grad_violations(gg[k], og[k])       # end to end: counted against north_star's plain bar ...
        total_bad += int(bad_e2e.sum()); total += bad_e2e.size
        ok = pu.e2e_within_propagated(gg[k], og[k], tol_p[k])     # ... and EVERY element within the derived bar
        assert ok.all(), f"{k}: {int((~ok).sum())} elements outside the propagated end-to-end bar"
    assert total_bad <= max(4, 2e-5 * total), f"end-to-end violators {total_bad}/{total}"     # measured <= 4e-6
    # The same count for a CPU that keeps its sums in fp32 (the oracle's loops with float accumulators, then the same
    # fp64 chain rule): north_star's bar is met end to end by neither on cancellation-dominated elements, and the GPU
    # (fp32 registers, shuffles, atomics in arbitrary order) must not be worse than that by more than a small factor
    c32 = xo.rasterize_bwd(o["proj"], o["binned"], o["fwd"], dL, o["cam"], o["cfg"], np.float32, acc32=True)
    cpu32 = xo.project_bwd(scene.means, scene.scales, scene.quats, scene.opacities, scene.sh, o["cam"], o["cfg"], c32,
                           np.float32)
    cpu_bad = sum(int(pu.grad_violations(cpu32[k], og[k])[0].sum()) for k in PARAMS)
    cpu_plain = sum(int(pu.grad_violations(c32[ko], og[ko])[0].sum()) for _, ko in PAIRS_2D)
    E2E_STATS.append((scene.name, scene.N, n_plain, cpu_plain, total_bad, cpu_bad, total))
    assert total_bad <= 3 * cpu_bad + max(4, 2e-5 * total), (total_bad, cpu_bad)
    culled = o["proj"]["tile_count"] == 0
    for k in PARAMS:                                              # P11: a culled Gaussian gets exactly zero
        assert not np.any(gg[k][culled])
    return g, o


def test_config1_tiny_full():
    g, o = full_parity(scenes.make_scene(1))
    assert g["binned"]["num_pairs"] == o["binned"]["num_pairs"] > 2000


def test_config2_object_reduced():
    full_parity(scenes.make_scene(2, n_override=20000, image_override=(200, 200)))


def test_config2_object_full_size():
    full_parity(scenes.make_scene(2))


@pytest.mark.parametrize("view", [0, 1])
def test_config3_unbounded_reduced(view):
    full_parity(scenes.make_scene(3, n_override=50000, image_override=(480, 270)), view)


@pytest.mark.parametrize("view", [0, 1])
def test_config4_ut_fisheye_reduced(view):
    full_parity(scenes.make_scene(4, n_override=50000, image_override=(480, 270)), view)


@pytest.mark.parametrize("view", [0, 3])
def test_config5_stress_reduced(view):
    full_parity(scenes.make_scene(5, n_override=30000, image_override=(320, 180)), view)


@pytest.mark.parametrize("wh", [(70, 50), (33, 17), (16, 16), (250, 130)])
def test_ragged_image_sizes(wh):
    full_parity(scenes.make_scene(1, n_override=600, image_override=wh))


@pytest.mark.parametrize("deg", [0, 1, 2, 3])
def test_sh_degrees(deg):
    sc = scenes.make_scene(2, n_override=3000, image_override=(96, 96))
    K = (deg + 1) ** 2
    sc.sh = np.ascontiguousarray(sc.sh[:, :K, :])
    sc.sh_degree = deg
    full_parity(sc)


def test_antialias_ewa_and_background():
    sc = scenes.make_scene(3, n_override=20000, image_override=(320, 180))
    full_parity(sc, 1, dict(antialias=1, bg=(0.25, 0.5, 0.75)))


def test_ut_pinhole():
    sc = scenes.make_scene(3, n_override=20000, image_override=(320, 180))
    full_parity(sc, 1, dict(projection=1, antialias=1))


def test_config3_full_size_bench_configuration():
    """BASELINE.json configs[2] at full size (1M Gaussians, 1920x1080), the launch configuration
    bench.py times: every stage against the oracle, every element."""
    g, o = full_parity(scenes.make_scene(3))
    assert o["binned"]["num_pairs"] > 5_000_000


def test_config5_full_size_stress_view():
    """BASELINE.json configs[4] at full size (3M Gaussians, 1920x1080, > 10^8 tile-Gaussian pairs in one
    view): every stage against the oracle, every element (the oracle needs about a minute)."""
    g, o = full_parity(scenes.make_scene(5), view=0)
    assert o["binned"]["num_pairs"] > 50_000_000


@pytest.mark.parametrize("view", [0, 1])
def test_config4_full_size_ut_fisheye(view):
    """BASELINE.json configs[3] at full size (1M Gaussians, UT with 7 sigma points through the seeded
    fisheye camera, 1920x1080), both poses."""
    g, o = full_parity(scenes.make_scene(4), view=view)
    assert o["binned"]["num_pairs"] > 1_000_000


def test_config3_full_size_second_pose():
    full_parity(scenes.make_scene(3), view=1)


# ---- f1: tile_cull ("Cull", L268-281, L435; C8) -------------------------------------
CULL = dict(tile_cull=1)


@pytest.mark.parametrize("config,kw,view", [(1, {}, 0), (2, dict(n_override=20000, image_override=(200, 200)), 0),
                                            (3, dict(n_override=50000, image_override=(480, 270)), 1),
                                            (4, dict(n_override=50000, image_override=(480, 270)), 0),
                                            (5, dict(n_override=30000, image_override=(320, 180)), 3)])
def test_tile_cull_reduced(config, kw, view):
    g, o = full_parity(scenes.make_scene(config, **kw), view, CULL)
    assert g["binned"]["num_pairs"] == o["binned"]["num_pairs"] < o["binned"]["num_candidates"]


def test_tile_cull_image_equals_uncut_image_on_gpu():
    """PAPER L683 on the GPU path itself: same image, final_T and gradients with and without culling."""
    sc = scenes.make_scene(3, n_override=50000, image_override=(480, 270))
    a = pu.run_gpu(sc, 0)
    b = pu.run_gpu(sc, 0, CULL)
    assert b["binned"]["num_pairs"] < a["binned"]["num_pairs"]
    np.testing.assert_array_equal(a["fwd"]["image"], b["fwd"]["image"])
    np.testing.assert_array_equal(a["fwd"]["final_T"], b["fwd"]["final_T"])
    dL = np.sign(a["fwd"]["image"] - sc.target(0)).astype(np.float32)
    ga, gb = pu.run_gpu_backward(a, dL), pu.run_gpu_backward(b, dL)
    for k in PARAMS:      # same terms, another order of the fp32 atomics: only cancelled elements may move
        bad, _ = pu.grad_violations(gb[k], ga[k])
        assert bad.mean() <= 1e-4, (k, int(bad.sum()))


def test_tile_cull_ragged_and_edge():
    full_parity(scenes.make_scene(1, n_override=600, image_override=(70, 50)), 0, CULL)
    full_parity(scenes.make_scene(1, n_override=600, image_override=(33, 17)), 0, CULL)


@pytest.mark.parametrize("wh", [(1924, 1083), (1925, 1081)])
@pytest.mark.parametrize("cull", [0, 1])
def test_throughput_shapes_on_ragged_widths(wh, cull):
    """>= 4096 tiles select the throughput shapes of the compositing kernels (forward: pixel pairs (x, x + 8); backward: 8
    consecutive pixels per thread, one warp per tile, per-pixel inputs as 128-bit words when W % 4 == 0).  Widths that are not
    a multiple of 8 (a thread's pixels straddle the image edge) or of 4 (no vector loads) and a ragged last tile row, with
    and without tile_cull (the branch-free and the branching forward blend)."""
    sc = scenes.make_scene(3, n_override=40000, image_override=wh)
    assert ((wh[0] + 15) // 16) * ((wh[1] + 15) // 16) >= 4096
    full_parity(sc, 0, dict(tile_cull=cull))


def test_tile_cull_config3_full_size_bench_configuration():
    g, o = full_parity(scenes.make_scene(3), 0, CULL)
    assert o["binned"]["num_pairs"] < 0.75 * o["binned"]["num_candidates"]


def test_tile_cull_config5_full_size():
    g, o = full_parity(scenes.make_scene(5), 0, CULL)
    assert o["binned"]["num_pairs"] > 50_000_000


def test_zz_report_gradient_violators(capsys):
    """Prints, for every case of this file, how many gradient elements miss north_star's plain bar 1e-3 |ref| + 1e-6 on
    the GPU and for a CPU fp32 sum of the same terms (DESIGN.md 5 quotes these numbers)."""
    with capsys.disabled():
        for name, n, g1, c1, g2, c2, tot in E2E_STATS:
            print(f"\n[2D gradients] {name} N={n}: compositing stage GPU {g1} / CPU-fp32 {c1} of {9 * n}; "
                  f"end to end GPU {g2} / CPU-fp32 {c2} of {tot}", end="")
