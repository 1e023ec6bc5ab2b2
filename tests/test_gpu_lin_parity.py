"""f4 XPR-LinPrim forward (PAPER A.1.3 L506-697, Listings 4-5, Eq. 2): the CUDA path (xpr_lin_project ->
xpr_bin_sort_lin -> xpr_lin_rasterize_fwd, through the C-ABI) against the CPU oracle (oracle/xpr_oracle_lin.inc) on
the same seeded scenes.  Bars: record values that feed integers or decisions (mu2D, sigma, depth, slabs), rectangles,
counts, keys, values and ranges bit-exact, with and without tile_cull; colours within 1 ulp; image within
north_star's 1e-4 max abs outside pixels whose EXIT decision the oracle marks fragile; n_contrib equal there.
The scenes are the synthetic Gaussian scenes of DESIGN.md section 4 read as octahedra (same centres, half-axes = the
Gaussian scales times a factor, same orientations, opacities and SH): LinPrim has no scene recipe of its own in the paper."""
import numpy as np
import pytest

import parity_util as pu
import xpr_oracle as xo
from paper_2606_11529_b200 import scenes

pytestmark = pytest.mark.gpu


def run_pair(sc, scale_mul, cfg_over, view=0):
    import torch
    from paper_2606_11529_b200 import pipeline
    cfg = scenes.default_render_config(sc)
    cfg.update(cfg_over)
    scales = np.ascontiguousarray(sc.scales * np.float32(scale_mul), np.float32)
    arr = dict(means=sc.means, scales=scales, quats=sc.quats, opacities=sc.opacities, sh=sc.sh)
    ocam = xo.make_camera(sc.cameras[view])
    ocfg = xo.make_config(cfg, fragile_rel=2e-5)
    o = xo.render_lin(arr, ocam, ocfg, np.float32)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")
    pipe = pipeline.LinPrimPipeline(sc.N, sc.cameras[view], cfg)
    pipe.forward(t(sc.means), t(scales), t(sc.quats), t(sc.opacities), t(sc.sh))
    torch.cuda.synchronize()
    return pipe, o


def compare(pipe, o):
    op, ob, of = o["proj"], o["binned"], o["fwd"]
    tc = pu.u32(pipe.tile_count)
    np.testing.assert_array_equal(tc, op["tile_count"])
    vis = tc > 0
    np.testing.assert_array_equal(pipe.tile_rect.cpu().numpy()[vis], op["tile_rect"][vis])
    rec = pipe.lin_rec.cpu().numpy()
    np.testing.assert_array_equal(rec[vis, :16].view(np.uint32), op["lin_rec"][vis, :16].view(np.uint32))
    np.testing.assert_array_equal(pipe.depth.cpu().numpy()[vis].view(np.uint32), op["depth"][vis].view(np.uint32))
    assert not rec[~vis].any()
    # colour: same SH sum, the direction's normalisation may differ by an ulp
    np.testing.assert_allclose(rec[vis, 16:19], op["lin_rec"][vis, 16:19], rtol=0, atol=2e-6)
    I = pipe.num_pairs
    assert I == ob["num_pairs"]
    np.testing.assert_array_equal(pipe.keys_sorted[:I].cpu().numpy().view(np.uint64), ob["keys"])
    np.testing.assert_array_equal(pu.u32(pipe.vals_sorted[:I]), ob["vals"])
    np.testing.assert_array_equal(pu.u32(pipe.tile_ranges), ob["ranges"])
    frag = (of["fragile"] & (pu.FRAG_EXIT | pu.FRAG_CLAMP)) != 0
    ok = ~frag
    img = pipe.image.cpu().numpy()
    err = np.abs(img.astype(np.float64) - of["image"].astype(np.float64)).max(axis=2)
    assert err[ok].max(initial=0.0) <= pu.IMG_TOL, f"image max err {err[ok].max()}"
    np.testing.assert_array_equal(pu.u32(pipe.n_contrib)[ok], of["n_contrib"][ok])
    dT = np.abs(pipe.final_T.cpu().numpy().astype(np.float64) - of["final_T"].astype(np.float64))
    assert dT[ok].max(initial=0.0) <= 1e-5
    assert frag.sum() <= max(2, 1e-3 * frag.size)
    return I, float(err[ok].max(initial=0.0)), int(frag.sum())


@pytest.mark.parametrize("tile_cull", [0, 1])
@pytest.mark.parametrize("case", ["small", "ragged", "sh3"])
def test_lin_forward_parity(case, tile_cull):
    if case == "small":
        sc, mul, over = scenes.make_scene(2, n_override=4000, image_override=(160, 160)), 3.0, {}
    elif case == "ragged":      # image edges that are no multiple of the tile, several supertiles
        sc, mul, over = scenes.make_scene(1, n_override=20000, image_override=(333, 207)), 2.0, {}
    else:
        sc, mul, over = scenes.make_scene(3, n_override=30000, image_override=(320, 256)), 5.0, {}
    pipe, o = run_pair(sc, mul, dict(over, tile_cull=tile_cull))
    I, err, nfrag = compare(pipe, o)
    assert I > 1000 and (o["fwd"]["final_T"] < 0.5).any()
    print(f"LIN_PARITY case={case} cull={tile_cull} pairs={I} img_err={err:.2e} fragile={nfrag}")


def test_lin_cull_drops_pairs_and_keeps_image():
    """tile_cull changes the lists, not the image (on the GPU: bit for bit, the dropped pairs never pass the gate)."""
    sc = scenes.make_scene(2, n_override=4000, image_override=(160, 160))
    p0, _ = run_pair(sc, 3.0, dict(tile_cull=0))
    p1, _ = run_pair(sc, 3.0, dict(tile_cull=1))
    assert p1.num_pairs < p0.num_pairs
    assert np.array_equal(p0.image.cpu().numpy(), p1.image.cpu().numpy())
    assert np.array_equal(p0.final_T.cpu().numpy(), p1.final_T.cpu().numpy())


def test_lin_stats_match_oracle_counters():
    import torch
    from paper_2606_11529_b200 import binding as xb
    sc = scenes.make_scene(2, n_override=4000, image_override=(160, 160))
    pipe, o = run_pair(sc, 3.0, dict(tile_cull=1))
    stats = torch.zeros(4, dtype=torch.int64, device="cuda:0")
    xb.xpr_lin_rasterize_stats(pipe.cam, pipe.cfg, pipe.lin_rec, pipe.vals_sorted, pipe.tile_ranges, stats)
    s = stats.cpu().numpy()
    frag = (o["fwd"]["fragile"] & (pu.FRAG_EXIT | pu.FRAG_CLAMP)) != 0
    if not frag.any():
        assert int(s[0]) == o["fwd"]["pp_visit"] and int(s[1]) == o["fwd"]["pp_pass"]
        assert int(s[3]) == int(o["fwd"]["n_contrib"].astype(np.int64).sum())
    assert s[0] >= s[1] >= s[2] > 0


def test_lin_edges():
    """N = 0, everything behind the camera, unsupported cameras / batches: defined results, no launch on bad input."""
    import torch
    from paper_2606_11529_b200 import binding as xb, pipeline
    sc = scenes.make_scene(2, n_override=64, image_override=(64, 48))
    cfg = dict(scenes.default_render_config(sc), bg=(0.25, 0.5, 0.75))
    z = lambda *s: torch.zeros(*s, device="cuda:0")
    pipe = pipeline.LinPrimPipeline(0, sc.cameras[0], cfg)
    pipe.forward(z(0, 3), z(0, 3), z(0, 4), z(0), z(0, pipe_k(cfg), 3))
    torch.cuda.synchronize()
    assert pipe.num_pairs == 0
    img = pipe.image.cpu().numpy()
    assert np.array_equal(img, np.broadcast_to(np.float32([0.25, 0.5, 0.75]), img.shape))
    assert (pipe.final_T.cpu().numpy() == 1).all() and not pipe.n_contrib.cpu().numpy().any()
    # all primitives behind the camera
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")
    cam = sc.cameras[0]
    W3, tv = np.asarray(cam.w2c)[:, :3], np.asarray(cam.w2c)[:, 3]
    behind = (W3.T @ (np.array([0, 0, -5.0]) - tv)).astype(np.float32)
    means = np.tile(behind, (sc.N, 1))
    pipe = pipeline.LinPrimPipeline(sc.N, cam, cfg)
    pipe.forward(t(means), t(sc.scales), t(sc.quats), t(sc.opacities), t(sc.sh))
    torch.cuda.synchronize()
    assert pipe.num_pairs == 0 and not pipe.tile_count.cpu().numpy().any() and not pipe.lin_rec.cpu().numpy().any()
    # a batch of views and a fisheye camera are rejected before any launch
    two = xb.make_cameras([cam, cam])
    with pytest.raises(xb.XprError) as e:
        xb.xpr_lin_project(t(sc.means), t(sc.scales), t(sc.quats), t(sc.opacities), t(sc.sh), two[0],
                           xb.make_config(dict(cfg, views=2)), pipe.lin_rec, pipe.depth, pipe.tile_rect, pipe.tile_count)
    assert e.value.status == xb.XPR_ERR_UNSUPPORTED
    fcam = xb.make_camera(cam)
    fcam.model = 1
    with pytest.raises(xb.XprError) as e:
        xb.xpr_lin_project(t(sc.means), t(sc.scales), t(sc.quats), t(sc.opacities), t(sc.sh), fcam, pipe.cfg,
                           pipe.lin_rec, pipe.depth, pipe.tile_rect, pipe.tile_count)
    assert e.value.status == xb.XPR_ERR_UNSUPPORTED


def pipe_k(cfg):
    return (int(cfg["sh_degree"]) + 1) ** 2


# ---- backward (xpr_lin_rasterize_bwd, xpr_lin_project_bwd) --------------------------------------------------

PARAMS = ("g_means", "g_scales", "g_quats", "g_opacities", "g_sh")


def backward_pair(sc, mul, cfg_over):
    import torch
    pipe, o = run_pair(sc, mul, cfg_over)
    compare(pipe, o)
    cfg = dict(scenes.default_render_config(sc), **cfg_over)
    ocam, ocfg = xo.make_camera(sc.cameras[0]), xo.make_config(cfg, fragile_rel=2e-5)
    _, dL = scenes.loss_and_grad(sc.loss, o["fwd"]["image"], sc.target(0))
    frag = (o["fwd"]["fragile"] & (pu.FRAG_EXIT | pu.FRAG_CLAMP)) != 0
    dL = np.where(frag[..., None], 0.0, dL).astype(np.float32)      # fragile pixels carry no gradient on either side
    scales = np.ascontiguousarray(sc.scales * np.float32(mul), np.float32)
    arr = dict(means=sc.means, scales=scales, quats=sc.quats, opacities=sc.opacities, sh=sc.sh)
    og = xo.backward_lin(arr, o, dL, ocam, ocfg, np.float32)
    mass = xo.lin_rasterize_bwd(o["proj"], o["binned"], o["fwd"], dL, ocam, ocfg, np.float32, mass=True)
    pipe.backward(torch.from_numpy(dL).to(pipe.device))
    torch.cuda.synchronize()
    return pipe, o, og, mass, arr, ocam, ocfg


@pytest.mark.parametrize("case", ["small", "ragged", "sh3", "config3_full_size"])
def test_lin_backward_parity(case):
    """Stage 1: the record gradient against the oracle's, element by element, within 1e-3 |ref| + 1e-6 + 2e-6 mass (the fp32
    summation floor of DESIGN.md section 5).  Stage 2 (stage-isolated, strict 1e-3 |ref| + 1e-6): xpr_lin_project_bwd fed
    the GPU's own fp32 record gradient against the oracle's projection backward fed the same values.  End to end: the
    share of parameter-gradient elements outside 1e-3 |ref| + 1e-6 is reported and bounded."""
    if case == "small":
        sc, mul = scenes.make_scene(2, n_override=4000, image_override=(160, 160)), 3.0
    elif case == "ragged":
        sc, mul = scenes.make_scene(1, n_override=20000, image_override=(333, 207)), 2.0
    elif case == "sh3":
        sc, mul = scenes.make_scene(3, n_override=30000, image_override=(320, 256)), 5.0
    else:       # the workload `bench.py --linprim 3 --config 3` times: 1 M octahedra, 1920x1080, Eq. 2's cull on
        sc, mul = scenes.make_scene(3), 3.0
    pipe, o, og, mass, arr, ocam, ocfg = backward_pair(sc, mul, dict(tile_cull=1))
    g_rec = pipe.g_lin_rec.cpu().numpy()
    assert np.isfinite(g_rec).all()
    bad, err = pu.grad_violations(g_rec, og["g_lin_rec"], mass)
    assert not bad.any(), (int(bad.sum()), np.argwhere(bad.reshape(g_rec.shape))[:5])
    plain, _ = pu.grad_violations(g_rec, og["g_lin_rec"])
    assert np.abs(og["g_lin_rec"]).max() > 0
    # stage 2, isolated
    iso = xo.lin_project_bwd(arr["means"], arr["scales"], arr["quats"], arr["opacities"], arr["sh"], ocam, ocfg,
                             g_rec.astype(np.float64), np.float32)
    for k in PARAMS:
        got = getattr(pipe, k).cpu().numpy()
        b2, _ = pu.grad_violations(got, iso[k])
        assert not b2.any(), (k, int(b2.sum()))
    # end to end
    total = nbad = 0
    for k in PARAMS:
        b3, _ = pu.grad_violations(getattr(pipe, k).cpu().numpy(), og[k])
        total += b3.size; nbad += int(b3.sum())
    print(f"LIN_BWD case={case} rec_plain_violators={int(plain.sum())}/{plain.size} e2e_violators={nbad}/{total}")
    assert nbad <= max(4, 1e-3 * total)
    culled = o["proj"]["tile_count"] == 0
    for k in PARAMS:
        assert not getattr(pipe, k).cpu().numpy()[culled].any()
