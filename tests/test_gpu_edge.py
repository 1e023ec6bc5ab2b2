"""GPU edge cases of the hot path: empty input, everything culled, capacity overflow and regrowth,
a full-screen Gaussian, exact depth ties (stable order), huge pair counts per Gaussian."""
import numpy as np
import pytest

import parity_util as pu
import xpr_oracle as xo
from paper_2606_11529_b200 import scenes

pytestmark = pytest.mark.gpu


def _subset(sc, idx):
    sc.means, sc.scales, sc.quats = sc.means[idx].copy(), sc.scales[idx].copy(), sc.quats[idx].copy()
    sc.opacities, sc.sh = sc.opacities[idx].copy(), sc.sh[idx].copy()
    return sc


def test_empty_scene_renders_background():
    import torch
    from paper_2606_11529_b200 import pipeline
    sc = _subset(scenes.make_scene(1), np.arange(0))
    cfg = scenes.default_render_config(sc)
    cfg["bg"] = (0.1, 0.2, 0.3)
    pipe = pipeline.SplatPipeline(0, sc.cameras[0], cfg)
    img = pipe.forward(*pipeline.scene_to_device(sc))
    torch.cuda.synchronize()
    assert pipe.num_pairs == 0
    np.testing.assert_allclose(img.cpu().numpy(), np.broadcast_to(np.float32([0.1, 0.2, 0.3]), (64, 64, 3)))
    assert (pipe.final_T.cpu().numpy() == 1).all() and (pipe.n_contrib.cpu().numpy() == 0).all()


def test_everything_culled_behind_camera():
    sc = scenes.make_scene(1, n_override=500)
    sc.means[:, 2] -= 10.0          # all behind the camera at z = -4 looking +z
    g = pu.run_gpu(sc)
    o = pu.run_oracle(sc)
    assert o["binned"]["num_pairs"] == 0 and g["binned"]["num_pairs"] == 0
    assert (g["proj"]["tile_count"] == 0).all() and (g["proj"]["flags"] == 0).all()
    assert (g["fwd"]["image"] == 0).all() and (g["binned"]["ranges"] == 0).all()
    gg = pu.run_gpu_backward(g, np.ones((64, 64, 3), np.float32))
    for k, v in gg.items():
        assert not np.any(v), k


def test_capacity_error_reports_required_pairs_then_regrows():
    import torch
    from paper_2606_11529_b200 import binding as xb, pipeline
    sc = scenes.make_scene(1)
    o = pu.run_oracle(sc)
    I = o["binned"]["num_pairs"]
    cfg = scenes.default_render_config(sc)
    pipe = pipeline.SplatPipeline(sc.N, sc.cameras[0], cfg, pair_capacity=100)
    pipe.project(*pipeline.scene_to_device(sc))
    guard = torch.full((pipe.keys_sorted.numel(),), -7, dtype=torch.int64, device="cuda")
    st, need = xb.xpr_bin_sort(pipe.depth, pipe.tile_rect, pipe.tile_count, pipe.cam, pipe.cfg, 50, guard,
                               pipe.vals_sorted, pipe.tile_ranges, pipe.workspace, raise_on_capacity=False)
    torch.cuda.synchronize()
    assert st == xb.XPR_ERR_CAPACITY and need == I
    assert (guard[50:] == -7).all()          # nothing written beyond the stated capacity
    with pytest.raises(xb.XprError):
        xb.xpr_bin_sort(pipe.depth, pipe.tile_rect, pipe.tile_count, pipe.cam, pipe.cfg, 50, guard,
                        pipe.vals_sorted, pipe.tile_ranges, pipe.workspace)
    assert pipe.bin_sort() == I and pipe.pair_capacity >= I     # pipeline regrows and redoes
    np.testing.assert_array_equal(pu.u32(pipe.vals_sorted[:I]), o["binned"]["vals"])


def test_capacity_zero_is_a_size_probe_in_both_modes():
    """pair_capacity = 0 with visible Gaussians: xpr.h promises XPR_ERR_CAPACITY and the capacity that suffices --
    synchronously through *num_pairs_host, asynchronously in workspace[0:8] -- never a clean OK with empty lists."""
    import torch
    from paper_2606_11529_b200 import binding as xb, pipeline
    sc = scenes.make_scene(1)
    I = pu.run_oracle(sc)["binned"]["num_pairs"]
    cfg = scenes.default_render_config(sc)
    pipe = pipeline.SplatPipeline(sc.N, sc.cameras[0], cfg, pair_capacity=64)
    pipe.project(*pipeline.scene_to_device(sc))
    ws = torch.empty(xb.xpr_bin_sort_workspace(sc.N, 0, pipe.T), dtype=torch.uint8, device="cuda")
    guard_k = torch.full((64,), -7, dtype=torch.int64, device="cuda")
    guard_v = torch.full((64,), -7, dtype=torch.int32, device="cuda")
    st, need = xb.xpr_bin_sort(pipe.depth, pipe.tile_rect, pipe.tile_count, pipe.cam, pipe.cfg, 0, guard_k, guard_v,
                               pipe.tile_ranges, ws, raise_on_capacity=False)
    assert st == xb.XPR_ERR_CAPACITY and need == I
    ws.zero_(); pipe.tile_ranges.fill_(-1)
    xb.xpr_bin_sort(pipe.depth, pipe.tile_rect, pipe.tile_count, pipe.cam, pipe.cfg, 0, guard_k, guard_v,
                    pipe.tile_ranges, ws, sync=False)
    torch.cuda.synchronize()
    counts = ws[:16].view(torch.int64).tolist()
    assert counts == [I, 0]
    assert (guard_k == -7).all() and (guard_v == -7).all() and not pipe.tile_ranges.any()
    # a retry with the reported capacity succeeds
    pipe._alloc_pairs(need + 1)
    assert pipe.bin_sort() == I


def test_binding_rejects_a_tensor_of_the_wrong_element_type():
    import torch
    from paper_2606_11529_b200 import binding as xb, pipeline
    sc = scenes.make_scene(1, n_override=50)
    pipe = pipeline.SplatPipeline(sc.N, sc.cameras[0], scenes.default_render_config(sc))
    m, s, q, o, sh = pipeline.scene_to_device(sc)
    with pytest.raises(TypeError):
        pipe.project(m.double(), s, q, o, sh)
    with pytest.raises(TypeError):
        xb.xpr_bin_sort(pipe.depth, pipe.tile_rect.long(), pipe.tile_count, pipe.cam, pipe.cfg, pipe.pair_capacity,
                        pipe.keys_sorted, pipe.vals_sorted, pipe.tile_ranges, pipe.workspace)


def test_fullscreen_gaussian_and_depth_ties():
    """One Gaussian covering every tile plus exact duplicates (equal keys): the stable order of equal
    keys is ascending Gaussian index (C10), so sorted values must match bit-exactly."""
    sc = scenes.make_scene(2, n_override=4000, image_override=(320, 240))
    sc.means[0] = (0.0, 0.0, 0.0)
    sc.scales[0] = (5.0, 5.0, 5.0)       # covers the whole image
    sc.opacities[0] = 0.9
    for dup in range(1, 40):             # 39 exact copies of Gaussian 100 scattered over the index range
        j = 100 * dup
        sc.means[j], sc.scales[j], sc.quats[j] = sc.means[100], sc.scales[100] * 3, sc.quats[100]
    g = pu.run_gpu(sc)
    o = pu.run_oracle(sc)
    TW, TH = 20, 15
    assert o["proj"]["tile_count"][0] == TW * TH
    pu.compare_projection(g, o)
    pu.compare_binning(g, o)
    keys = o["binned"]["keys"]
    assert (np.diff(keys.astype(np.int64)) == 0).sum() >= 38       # the ties are really there
    pu.compare_forward(g, o)


def test_many_sort_tiles_and_all_digit_passes():
    """> 100 onesweep tiles (4096 pairs each) so that the decoupled look-back chains are exercised,
    and a 1920x1080 tile grid so that all six 8-bit digit passes carry information."""
    sc = scenes.make_scene(5, n_override=40000)
    g = pu.run_gpu(sc)
    o = pu.run_oracle(sc)
    assert o["binned"]["num_pairs"] > 100 * 4096
    pu.compare_projection(g, o)
    pu.compare_binning(g, o)
    keys = g["binned"]["keys"]
    assert (keys[1:] >= keys[:-1]).all()
    r = g["binned"]["ranges"].astype(np.int64)
    nz = r[:, 1] > r[:, 0]
    assert (r[nz, 1] - r[nz, 0]).sum() == o["binned"]["num_pairs"]     # ranges partition [0, I)


def test_async_bin_sort_matches_sync_and_overflow_renders_background():
    """num_pairs_host = NULL: no host read-back; I is left in the first 8 bytes of the workspace.  Same outputs
    as the synchronous call; over capacity every tile range is (0, 0) and nothing is written out of bounds."""
    import torch
    from paper_2606_11529_b200 import binding as xb, pipeline
    sc = scenes.make_scene(2, n_override=20000, image_override=(200, 200))
    cfg = scenes.default_render_config(sc)
    params = pipeline.scene_to_device(sc)
    pipe = pipeline.SplatPipeline(sc.N, sc.cameras[0], cfg)
    pipe.project(*params)
    I = pipe.bin_sort()
    keys = pipe.keys_sorted[:I].clone(); vals = pipe.vals_sorted[:I].clone(); ranges = pipe.tile_ranges.clone()
    pipe.keys_sorted.fill_(-1); pipe.vals_sorted.fill_(-1); pipe.tile_ranges.fill_(-1)
    pipe.bin_sort_async()
    assert pipe.check_capacity() == I
    assert torch.equal(pipe.keys_sorted[:I], keys) and torch.equal(pipe.vals_sorted[:I], vals)
    assert torch.equal(pipe.tile_ranges, ranges)
    # over capacity, asynchronously
    small = pipeline.SplatPipeline(sc.N, sc.cameras[0], cfg, pair_capacity=4096)
    small.project(*params)
    guard = torch.full((8192,), -7, dtype=torch.int64, device="cuda")
    xb.xpr_bin_sort(small.depth, small.tile_rect, small.tile_count, small.cam, small.cfg, 4096, guard,
                    small.vals_sorted, small.tile_ranges, small.workspace, sync=False)
    torch.cuda.synchronize()
    need, written = small.pairs_on_device()       # the capacity that suffices (xpr.h: max(I, rows + 1, 2 x supertile
    assert written == 0 and need >= I and need > 4096      # words)), nothing in the output
    exact = pipeline.SplatPipeline(sc.N, sc.cameras[0], cfg, pair_capacity=need)
    exact.project(*params)
    st, n = xb.xpr_bin_sort(exact.depth, exact.tile_rect, exact.tile_count, exact.cam, exact.cfg, need, exact.keys_sorted,
                            exact.vals_sorted, exact.tile_ranges, exact.workspace, raise_on_capacity=False)
    assert st == xb.XPR_OK and n == I and torch.equal(exact.keys_sorted[:I], keys)     # ... and it does suffice
    assert (guard[4096:] == -7).all()
    assert not small.tile_ranges.any()
    with pytest.raises(xb.XprError):
        small.check_capacity()
    small.rasterize_fwd()
    torch.cuda.synchronize()
    assert float(small.image.abs().max()) == 0.0 and float(small.final_T.min()) == 1.0


def test_more_than_65536_tiles_three_tile_digit_passes():
    """4112 x 4112 pixels = 257 x 257 = 66049 tiles: tile ids need 17 bits -> three tile-digit passes on the pairs
    (emit_kernel<3>), tile coordinates beyond 8 bits, ragged last tile row/column."""
    sc = scenes.make_scene(1, n_override=400, image_override=(4112, 4112))
    for over in (None, dict(tile_cull=1)):
        g = pu.run_gpu(sc, 0, over)
        o = pu.run_oracle(sc, 0, over)
        pu.compare_projection(g, o)
        pu.compare_binning(g, o)
        n_frag, _ = pu.compare_forward(g, o)
        assert n_frag <= 1e-3 * 4112 * 4112
        assert int(g["binned"]["keys"].max() >> np.uint64(32)) > 65536


@pytest.mark.parametrize("kind", ["l1", "l2"])
def test_loss_grad_helper_matches_the_definition(kind):
    import torch
    from paper_2606_11529_b200 import binding as xb
    rng = np.random.default_rng(3)
    for n in (0, 3, 4, 4099, 64 * 64 * 3):
        img = rng.normal(0.5, 0.3, n).astype(np.float32)
        tgt = rng.normal(0.5, 0.3, n).astype(np.float32)
        if n > 2:
            tgt[1] = img[1]                      # exact zero difference
        want = scenes.loss_and_grad(kind, img, tgt)[1]
        out = torch.full((max(n, 1),), 7.0, device="cuda")[:n]
        xb.xpr_loss_grad(kind, torch.from_numpy(img).cuda(), torch.from_numpy(tgt).cuda(), out)
        torch.cuda.synchronize()
        np.testing.assert_array_equal(out.cpu().numpy().view(np.uint32), want.view(np.uint32))


def test_tile_order_is_a_permutation_by_decreasing_length_and_changes_no_result():
    sc = scenes.make_scene(3, n_override=40000, image_override=(480, 270))
    a = pu.run_gpu(sc, 0, dict(tile_cull=1, tile_order=1))
    b = pu.run_gpu(sc, 0, dict(tile_cull=1, tile_order=0))
    assert b["pipe"].tile_order is None
    order = pu.u32(a["pipe"].tile_order)
    T = a["pipe"].T
    np.testing.assert_array_equal(np.sort(order), np.arange(T, dtype=np.uint32))
    ln = (a["binned"]["ranges"][:, 1] - a["binned"]["ranges"][:, 0]).astype(np.int64)
    shift = max(0, int(ln.max()).bit_length() - 10)
    cls = np.minimum(1023, ln[order] >> shift)
    assert (np.diff(cls) <= 0).all() and ln[order[0]] >> shift == ln.max() >> shift
    for k in ("image", "final_T", "n_contrib"):
        np.testing.assert_array_equal(a["fwd"][k], b["fwd"][k])
    dL = np.random.default_rng(0).standard_normal((270, 480, 3)).astype(np.float32)
    ga, gb = pu.run_gpu_backward(a, dL), pu.run_gpu_backward(b, dL)
    for k in ("g_means", "g_sh", "g_opacities"):
        bad, _ = pu.grad_violations(ga[k], gb[k])
        assert bad.mean() <= 1e-4, k          # the atomics' order differs, nothing else


@pytest.mark.parametrize("ray", [0, 1])
def test_captured_step_replays_the_eager_step(ray):
    """pipeline.capture_step: the whole step in one CUDA graph gives the results of the eager calls."""
    import torch
    from paper_2606_11529_b200 import pipeline
    sc = scenes.make_scene(4 if ray else 3, n_override=20000, image_override=(320, 180))
    cfg = dict(scenes.default_render_config(sc), tile_cull=1, ray_eval=ray)
    params = pipeline.scene_to_device(sc)
    target = torch.from_numpy(sc.target(0)).cuda()
    pipe = pipeline.SplatPipeline(sc.N, sc.cameras[0], cfg)
    img = pipe.forward(*params).clone()
    dL = torch.sign(img - target)
    pipe.backward(dL)
    torch.cuda.synchronize()
    want = {k: getattr(pipe, k).clone() for k in ("g_means", "g_scales", "g_quats", "g_opacities", "g_sh")}
    n = pipe.num_pairs
    graph = pipe.capture_step(*params, target, "l1", pixel_info=bool(ray))
    for k in want:
        getattr(pipe, k).fill_(7.0)
    pipe.image.fill_(7.0)
    graph.replay(); graph.replay()
    torch.cuda.synchronize()
    assert pipe.check_capacity() == n
    assert torch.equal(pipe.image, img)
    for k, v in want.items():
        bad, _ = pu.grad_violations(getattr(pipe, k).cpu().numpy(), v.cpu().numpy())
        assert bad.mean() <= 1e-4, k            # same kernels, same inputs: only the order of the atomics differs


@pytest.mark.parametrize("seed", [0, 1])
def test_tile_cull_needle_gaussians_bit_exact(seed):
    """f1 adversarial case: rows_kernel keeps, per (Gaussian, tile row), ONE interval of tiles and settles its ends with
    the exact per-tile predicate; that equals the oracle's tile-by-tile test only if the kept tiles of a row are
    contiguous.  Needles -- scale ratios 1e3 .. 1e4 (screen-space sigma up to ~900 px against the 0.55 px low-pass
    floor), rotated in the image plane by any angle incl. 45 degrees, opaque and faint, centres inside and far
    outside the image -- are where the conservative 2^-18 margin of reading C8 could open a gap.  Lists, keys and
    ranges must be bit-exact, and the image must equal the one without tile_cull."""
    import torch
    rng = np.random.default_rng(700 + seed)
    sc = scenes.make_scene(3, n_override=4000, image_override=(960, 540))
    n = sc.N
    z = rng.uniform(2.0, 9.0, n)
    sc.means = np.stack([rng.uniform(-1.6, 1.6, n) * z, rng.uniform(-1.0, 1.0, n) * z, z], 1).astype(np.float32)
    long_ = np.exp(rng.uniform(np.log(0.3), np.log(4.0), n))
    ratio = np.exp(rng.uniform(np.log(1e3), np.log(1e4), n))
    sc.scales = np.stack([long_, long_ / ratio, long_ / ratio], 1).astype(np.float32)
    ang = np.where(rng.random(n) < 0.3, np.pi / 4, rng.uniform(0, np.pi, n))      # in-plane rotation about the view axis
    tilt = rng.normal(0, 0.05, n)                                                  # slightly out of the image plane
    q = np.stack([np.cos(ang / 2), tilt * 0.5, tilt * 0.5, np.sin(ang / 2)], 1)
    sc.quats = (q / np.linalg.norm(q, axis=1, keepdims=True)).astype(np.float32)
    sc.opacities = np.where(rng.random(n) < 0.5, rng.uniform(0.9, 0.999, n), rng.uniform(0.004, 0.05, n)).astype(np.float32)
    g = pu.run_gpu(sc, 0, dict(tile_cull=1))
    o = pu.run_oracle(sc, 0, dict(tile_cull=1))
    pu.compare_projection(g, o)
    assert o["binned"]["num_pairs"] > 20000 and o["binned"]["num_pairs"] < 0.5 * o["binned"]["num_candidates"]
    pu.compare_binning(g, o)                      # bit-exact keys, values, ranges
    pu.compare_forward(g, o)
    g0 = pu.run_gpu(sc, 0, dict(tile_cull=0))
    ok = (o["fwd"]["fragile"] & pu.FRAG_EXIT) == 0
    assert np.array_equal(g0["fwd"]["image"][ok], g["fwd"]["image"][ok])          # culling changes no pixel


@pytest.mark.gpu
@pytest.mark.parametrize("mode", [4, 1, 2])
def test_overlapped_zero_fill_gives_the_same_gradients(mode):
    """xpr_project_bwd_fill on a second stream + xpr_project_bwd_filled (pipeline option overlap_fill: forked at the
    forward compositing kernel (4, the default), at the backward (1) or at the binning stage (2)) against the plain
    xpr_project_bwd: same parameter gradients bit for bit (no atomics at one view), also when captured in a CUDA graph."""
    import numpy as np
    import torch
    from paper_2606_11529_b200 import pipeline, scenes
    sc = scenes.make_scene(2, n_override=20000, image_override=(320, 240))
    cfg = scenes.default_render_config(sc)
    params = pipeline.scene_to_device(sc)
    target = torch.from_numpy(sc.target(0)).cuda()
    names = ("g_means", "g_scales", "g_quats", "g_opacities", "g_sh")
    pipe = pipeline.SplatPipeline(sc.N, sc.cameras[0], dict(cfg, overlap_fill=mode))
    pipe.OVERLAP_MIN_BYTES = 0                              # (the pipeline skips the fork for scenes this small)
    assert pipeline.SplatPipeline(sc.N, sc.cameras[0], cfg).overlap_fill == 4
    pipe.forward(*params)
    pipe.step_async(*params, target, sc.loss)               # consumes the fill a first forward may have forked
    torch.cuda.synchronize()
    for k in names:
        getattr(pipe, k).fill_(float("nan"))                # the fill must really happen
    pipe._g2.fill_(float("nan"))                            # ... and so must that of the 2D gradients (mode 4: side stream too)
    pipe.step_async(*params, target, sc.loss)               # fill on the side stream, xpr_project_bwd_filled
    torch.cuda.synchronize()
    ref = pipeline.SplatPipeline(sc.N, sc.cameras[0], dict(cfg, overlap_fill=0))
    ref.forward(*params)
    ref.step_async(*params, target, sc.loss)
    torch.cuda.synchronize()
    for k in ("g_mean2d", "g_conic", "g_opac", "g_rgb"):    # same terms, another order of the fp32 atomics
        x, y = getattr(pipe, k).cpu().numpy(), getattr(ref, k).cpu().numpy()
        assert np.isfinite(x).all() and np.allclose(x, y, rtol=1e-2, atol=1e-3 * np.abs(y).max()), k
    a = {k: getattr(pipe, k).cpu().numpy().copy() for k in names}
    for k in names:
        getattr(pipe, k).fill_(float("nan"))
    pipe.overlap_fill = 0
    pipe.project_bwd()                                      # no fork before it: the plain xpr_project_bwd on the same 2D gradients
    torch.cuda.synchronize()
    pipe.overlap_fill = mode
    for k in names:
        b = getattr(pipe, k).cpu().numpy()
        assert np.isfinite(b).all() and np.array_equal(a[k], b), k
    assert np.abs(a["g_means"]).max() > 0
    graph = pipe.capture_step(*params, target, sc.loss)     # the fork / join is captured with the step
    for k in names:
        getattr(pipe, k).fill_(float("nan"))
    graph.replay()
    torch.cuda.synchronize()
    for k in names:
        c = getattr(pipe, k).cpu().numpy()                  # (the compositing atomics may sum in another order)
        assert np.isfinite(c).all() and np.allclose(c, a[k], rtol=1e-2, atol=1e-3 * np.abs(a[k]).max()), k


@pytest.mark.gpu
def test_fused_loss_backward_on_a_batch_of_views():
    """xpr_rasterize_bwd_loss with xpr_config.views = 2: image and target are [V,H,W,3]; same comparison as the single-view
    test below (the mass of a batch is per (view, Gaussian): the oracle's, view by view)."""
    import torch
    from paper_2606_11529_b200 import binding as xb, pipeline
    sc = scenes.make_scene(3, n_override=20000, image_override=(250, 130))
    cfg = scenes.default_render_config(sc)
    params = pipeline.scene_to_device(sc)
    views = [0, 1]
    target = torch.from_numpy(np.stack([sc.target(v) for v in views])).cuda()
    pipe = pipeline.SplatPipeline(sc.N, [sc.cameras[v] for v in views], cfg)
    pipe.forward(*params)
    dL = torch.empty_like(pipe.image)
    xb.xpr_loss_grad(sc.loss, pipe.image, target, dL)
    pipe.rasterize_bwd(dL)
    torch.cuda.synchronize()
    names = ("g_mean2d", "g_conic", "g_opac", "g_rgb")
    ref = {k: getattr(pipe, k).cpu().numpy().astype(np.float64) for k in names}
    for k in names:
        getattr(pipe, k).fill_(float("nan"))
    pipe.rasterize_bwd_loss(target, sc.loss)
    torch.cuda.synchronize()
    N = sc.N
    for vi, v in enumerate(views):
        o = pu.run_oracle(sc, v)
        mass = xo.rasterize_bwd(o["proj"], o["binned"], o["fwd"], dL[vi].cpu().numpy(), o["cam"], o["cfg"], np.float32, mass=True)
        for k, ko in zip(names, ("g_mean2d", "g_conic", "g_opac_eff", "g_rgb")):
            got = getattr(pipe, k).cpu().numpy().astype(np.float64)[vi * N:(vi + 1) * N]
            r = ref[k][vi * N:(vi + 1) * N]
            assert np.isfinite(got).all() and np.abs(r).max() > 0
            tol = 1e-3 * np.abs(r) + 2e-6 + 4e-6 * mass[ko].reshape(got.shape)
            assert (np.abs(got - r) <= tol).all(), (v, k, int((np.abs(got - r) > tol).sum()))


@pytest.mark.parametrize("config,n,wh", [(1, None, None), (2, 20000, (320, 240))])
def test_fused_loss_backward_matches_separate_loss_grad(config, n, wh):
    """xpr_rasterize_bwd_loss (loss gradient formed in the kernel's prologue) against xpr_loss_grad followed by
    xpr_rasterize_bwd: the same per-pixel dL values enter the same arithmetic, so the 2D gradients agree up to the order
    of the fp32 atomics; both
    losses (config 1: sum of squares, config 2: sum of absolute differences)."""
    import torch
    from paper_2606_11529_b200 import binding as xb, pipeline
    sc = scenes.make_scene(config, n_override=n, image_override=wh)
    cfg = scenes.default_render_config(sc)
    params = pipeline.scene_to_device(sc)
    target = torch.from_numpy(sc.target(0)).cuda()
    pipe = pipeline.SplatPipeline(sc.N, sc.cameras[0], cfg)
    pipe.forward(*params)
    dL = torch.empty_like(pipe.image)
    xb.xpr_loss_grad(sc.loss, pipe.image, target, dL)
    pipe.rasterize_bwd(dL)
    torch.cuda.synchronize()
    names = ("g_mean2d", "g_conic", "g_opac", "g_rgb")
    ref = {k: getattr(pipe, k).cpu().numpy().copy() for k in names}
    for k in names:
        getattr(pipe, k).fill_(float("nan"))
    assert pipe.can_fuse_loss()
    pipe.rasterize_bwd_loss(target, sc.loss)
    torch.cuda.synchronize()
    # both runs sum the same terms with fp32 atomics in an arbitrary order: each is within the stage-1 bar of the exact sum
    # (1e-3 |ref| + 1e-6 + 2e-6 mass), so their difference is within 1e-3 |ref| + 2e-6 + 4e-6 mass -- every
    # element, with the oracle's mass for the very dL the GPU used
    o = pu.run_oracle(sc, 0)
    mass = xo.rasterize_bwd(o["proj"], o["binned"], o["fwd"], dL.cpu().numpy(), o["cam"], o["cfg"], np.float32, mass=True)
    for k, ko in zip(names, ("g_mean2d", "g_conic", "g_opac_eff", "g_rgb")):
        got = getattr(pipe, k).cpu().numpy().astype(np.float64)
        assert np.isfinite(got).all() and np.abs(ref[k]).max() > 0
        tol = 1e-3 * np.abs(ref[k]) + 2e-6 + 4e-6 * mass[ko].reshape(got.shape)
        assert (np.abs(got - ref[k]) <= tol).all(), (k, int((np.abs(got - ref[k]) > tol).sum()))


@pytest.mark.gpu
def test_shade_record_equals_the_projection_record():
    """xpr_shade_record (for a caller with its own projection) builds, from the separate projection outputs, the 48-byte record
    xpr_project writes itself: bit for bit on every visible Gaussian (layout of xpr.h: the pre-scaled conic, +lnv, log2 o)."""
    import numpy as np
    import torch
    from paper_2606_11529_b200 import binding as xb, pipeline, scenes
    for config in (3, 4):
        sc = scenes.make_scene(config, n_override=30000, image_override=(320, 180))
        pipe = pipeline.SplatPipeline(sc.N, sc.cameras[0], scenes.default_render_config(sc))
        pipe.project(*pipeline.scene_to_device(sc))
        rec = torch.full_like(pipe.shade_rec, float("nan"))
        xb.xpr_shade_record(pipe.mean2d, pipe.conic_opac, pipe.rgb, pipe.lnv, pipe.depth, pipe.tile_count, rec)
        torch.cuda.synchronize()
        vis = (pipe.tile_count > 0).cpu().numpy()
        a = pipe.shade_rec.cpu().numpy().reshape(sc.N, 12).view(np.uint32)
        b = rec.cpu().numpy().reshape(sc.N, 12).view(np.uint32)
        assert vis.sum() > 1000 and np.array_equal(a[vis], b[vis])
        assert np.isnan(rec.cpu().numpy().reshape(sc.N, 12)[~vis]).all()          # culled Gaussians are skipped
        lnv = pipe.lnv.cpu().numpy()[vis]
        assert (lnv > 0).all() and np.array_equal(a[vis][:, 5], lnv.view(np.uint32))   # the gate's limit: +lnv, positive


@pytest.mark.gpu
@pytest.mark.parametrize("wh,cull", [((48, 40), 0), ((1024, 1024), 1), ((1024, 1024), 0)])
def test_hand_built_records_on_pixel_centres(wh, cull):
    """The compositing calls on hand-built projection outputs (no xpr_project): means EXACTLY on pixel centres (power is a
    signed zero at that pixel, for either sign of B, and must pass both gates: R3's one-compare form on -power), opacities a
    hair above alpha_thresh (lnv ~ 1e-6: only the centre pixel contributes), a saturating stack (exit), the latency shapes
    (3 x 3 tiles) and the throughput shapes (4096 tiles, most of them empty), forward and backward against the oracle."""
    import types
    import numpy as np
    import torch
    import parity_util as pu
    import xpr_oracle as xo
    from paper_2606_11529_b200 import binding as xb
    W, H = wh
    TW, TH = (W + 15) // 16, (H + 15) // 16
    rng = np.random.default_rng(11)
    at = 1.0 / 255.0
    cen = [(8.5, 8.5), (24.5, 8.5), (40.5 if W > 40 else 8.5, 24.5), (W - 7.5, H - 3.5), (16.5, 15.5)]
    m, con, op, col = [], [], [], []
    for cx, cy in cen:
        for sB in (+1.0, -1.0, 0.0):
            A_, C_ = rng.uniform(0.01, 0.05, 2)
            m.append((cx, cy)); con.append((A_, sB * 0.6 * np.sqrt(A_ * C_), C_)); op.append(rng.uniform(0.2, 0.7)); col.append(rng.uniform(0, 1, 3))
        m.append((cx, cy)); con.append((0.02, 0.004, 0.03)); op.append(at * (1.0 + 1e-6)); col.append((1.0, 1.0, 1.0))   # lnv ~ 1e-6
    for _ in range(40):                                                        # a saturating stack on one tile + random ones
        m.append((rng.uniform(0, min(W, 48)), rng.uniform(0, min(H, 40)))); con.append((0.004, 0.001, 0.005)); op.append(0.9); col.append(rng.uniform(0, 1, 3))
    N = len(m)
    mean2d = np.asarray(m, np.float32); conic = np.asarray(con, np.float32); opac = np.asarray(op, np.float32)
    rgb = np.asarray(col, np.float32)
    lnv = np.log(opac.astype(np.float64) / at).astype(np.float32)
    assert (lnv > 0).all()
    # lists: every Gaussian on every tile its 3.5 sigma box touches, in index order
    sx, sy = 3.5 / np.sqrt(conic[:, 0] * (1 - 0.36)), 3.5 / np.sqrt(conic[:, 2] * (1 - 0.36))
    vals, ranges = [], np.zeros((TW * TH, 2), np.uint32)
    for t in range(TW * TH):
        tx, ty = t % TW, t // TW
        hit = (mean2d[:, 0] + sx > 16 * tx) & (mean2d[:, 0] - sx < 16 * tx + 16) & (mean2d[:, 1] + sy > 16 * ty) & (mean2d[:, 1] - sy < 16 * ty + 16)
        idx = np.flatnonzero(hit)
        ranges[t] = (len(vals), len(vals) + len(idx)); vals.extend(idx.tolist())
    vals = np.asarray(vals, np.uint32)
    camo = types.SimpleNamespace(model=0, width=W, height=H, fx=100.0, fy=100.0, cx=W / 2, cy=H / 2, k=(0, 0, 0, 0),
                                 w2c=np.eye(4)[:3])
    cfgd = dict(projection=0, sh_degree=0, tile=16, antialias=0, alpha_thresh=at, alpha_max=0.99, t_min=1e-4, z_near=0.2,
                lowpass=0.3, ut_alpha=1.0, ut_beta=2.0, ut_kappa=0.0, bg=(0.1, 0.2, 0.3), tile_cull=cull)
    proj = dict(mean2d=mean2d, conic=conic, opac_eff=opac, rgb=rgb, lnv=lnv, tile_count=np.ones(N, np.uint32))
    binned = dict(vals=vals, ranges=ranges)
    ocam, ocfg = xo.make_camera(camo), xo.make_config(cfgd)
    of = xo.rasterize_fwd(proj, binned, ocam, ocfg, np.float32)
    d = "cuda:0"
    t = lambda a, dt=torch.float32: torch.from_numpy(np.ascontiguousarray(a)).to(d, dt)
    co4 = t(np.concatenate([conic, opac[:, None]], 1))
    rec = torch.empty(N, 12, device=d)
    xb.xpr_shade_record(t(mean2d), co4, t(rgb), t(lnv), t(np.ones(N, np.float32)), t(np.ones(N), torch.int32), rec)
    cam, cfg = xb.make_camera(camo), xb.make_config(cfgd)
    image, fT, nc = torch.empty(H, W, 3, device=d), torch.empty(H, W, device=d), torch.empty(H, W, dtype=torch.int32, device=d)
    v_d, r_d = t(vals.astype(np.int32), torch.int32), t(ranges.astype(np.int32), torch.int32)
    xb.xpr_rasterize_fwd(cam, cfg, rec, v_d, r_d, image, fT, nc)
    ok = (of["fragile"] & pu.FRAG_EXIT) == 0
    np.testing.assert_array_equal(nc.cpu().numpy().view(np.uint32)[ok], of["n_contrib"][ok])
    assert np.abs(image.cpu().numpy() - of["image"])[ok].max() <= 1e-4
    for cx, cy in cen:                                  # the centre pixels: every Gaussian centred there was blended
        px, py = int(cx), int(cy)
        mine = [i for i in range(N) if m[i] == (cx, cy)]
        lst = vals[ranges[(py // 16) * TW + px // 16][0]:ranges[(py // 16) * TW + px // 16][1]]
        assert of["n_contrib"][py, px] >= 1 + max(int(np.flatnonzero(lst == i)[0]) for i in mine[:3])
    assert (of["fragile"] & pu.FRAG_EXIT).sum() < 10 and (of["final_T"] < 0.01).any()
    dL = np.where(ok[..., None], rng.normal(0, 1, (H, W, 3)), 0.0).astype(np.float32)
    og = xo.rasterize_bwd(proj, binned, of, dL, ocam, ocfg, np.float32)
    mass = xo.rasterize_bwd(proj, binned, of, dL, ocam, ocfg, np.float32, mass=True)
    g = [torch.empty(N, k, device=d) for k in (2, 3, 1, 3)]
    nc_o = t(of["n_contrib"].astype(np.int32), torch.int32)        # both sides replay the oracle's n_contrib and T
    xb.xpr_rasterize_bwd(cam, cfg, rec, v_d, r_d, t(of["final_T"]), nc_o, t(dL), g[0], g[1], g[2].view(-1), g[3])
    for got, key in zip(g, ("g_mean2d", "g_conic", "g_opac_eff", "g_rgb")):
        bad, err = pu.grad_violations(got.cpu().numpy(), og[key], mass[key])
        assert bad.sum() == 0, (key, int(bad.sum()), float(err.max()))
    assert np.abs(og["g_opac_eff"]).max() > 0
