"""f3 "one launch for a batch of views" (Table 2; BASELINE.json configs[4]): xpr_config.views = V renders V views
of the same Gaussians with ONE call per stage.  The batch must equal V single-view runs bit for bit up to the backward
(same arithmetic per view: projection outputs, lists with tile ids offset by v T, images), and its parameter gradients
must equal the oracle's SUM over the views of the single-view gradients (the loss of a batch is the sum of the views'
losses) within the gradient bar of tests/test_gpu_parity.py."""
import numpy as np
import pytest

import parity_util as pu
import xpr_oracle as xo
from paper_2606_11529_b200 import scenes

pytestmark = pytest.mark.gpu
PARAMS = ("g_means", "g_scales", "g_quats", "g_opacities", "g_sh")


def batch_parity(sc, views, cfg_over=None):
    import torch
    from paper_2606_11529_b200 import pipeline
    cfg = scenes.default_render_config(sc)
    cfg.update(cfg_over or {})
    V, N = len(views), sc.N
    params = pipeline.scene_to_device(sc)
    bp = pipeline.SplatPipeline(N, [sc.cameras[v] for v in views], cfg)
    bp.forward(*params)
    torch.cuda.synchronize()
    T = bp.T // V
    I_total, off = bp.num_pairs, 0
    keys = bp.keys_sorted[:I_total].cpu().numpy().view(np.uint64)
    vals = pu.u32(bp.vals_sorted[:I_total])
    ranges = pu.u32(bp.tile_ranges).reshape(V, T, 2)
    dLs, og_sum, singles, tol_sum = [], None, [], None
    for k, v in enumerate(views):
        g = pu.run_gpu(sc, v, cfg_over)                       # the single-view GPU run
        o = pu.run_oracle(sc, v, cfg_over)
        sl = slice(k * N, (k + 1) * N)
        for name, arr in (("mean2d", bp.mean2d), ("conic_opac", bp.conic_opac), ("rgb", bp.rgb), ("depth", bp.depth),
                          ("lnv", bp.lnv), ("flags", bp.flags)):
            vis = g["proj"]["tile_count"] > 0
            a = arr[sl].cpu().numpy()
            assert np.array_equal(a[vis].view(np.uint8), g["proj"][name][vis].view(np.uint8)), (name, v)
        assert np.array_equal(pu.u32(bp.tile_count[sl]), g["proj"]["tile_count"])
        rect = bp.tile_rect[sl].cpu().numpy().copy()
        rect[:, [1, 3]] -= k * bp.TH                          # rows of view k are offset by k tiles_y
        assert np.array_equal(rect[vis], g["proj"]["tile_rect"][vis])
        # lists: the view's pairs are one contiguous block of the sorted arrays, tile ids offset by k T, values by k N
        I = g["binned"]["num_pairs"]
        kk, vv = keys[off:off + I], vals[off:off + I]
        assert np.array_equal(kk - (np.uint64(k * T) << np.uint64(32)), g["binned"]["keys"])
        assert np.array_equal(vv - np.uint32(k * N), g["binned"]["vals"])
        r = ranges[k].astype(np.int64)
        nz = (r[:, 1] > r[:, 0])
        assert np.array_equal((r - off)[nz], g["binned"]["ranges"].astype(np.int64)[nz]) and not r[~nz].any()
        off += I
        pick = (lambda t: t[k]) if V > 1 else (lambda t: t)       # a batch of one has no leading view dimension
        assert np.array_equal(pick(bp.image).cpu().numpy(), g["fwd"]["image"])
        assert np.array_equal(pick(bp.final_T).cpu().numpy(), g["fwd"]["final_T"])
        assert np.array_equal(pu.u32(pick(bp.n_contrib)), g["fwd"]["n_contrib"])
        _, dL = scenes.loss_and_grad(sc.loss, o["fwd"]["image"], sc.target(v))
        frag = (o["fwd"]["fragile"] & (pu.FRAG_EXIT | pu.FRAG_CLAMP)) != 0
        dL = np.where(frag[..., None], 0.0, dL).astype(np.float32)
        dLs.append(dL)
        og = xo.backward(o["arrays"], o, dL, o["cam"], o["cfg"], np.float32)
        og_sum = {p: og[p].copy() for p in PARAMS} if og_sum is None else {p: og_sum[p] + og[p] for p in PARAMS}
        mass = xo.rasterize_bwd(o["proj"], o["binned"], o["fwd"], dL, o["cam"], o["cfg"], np.float32, mass=True)
        tp = pu.propagated_param_tol(o["arrays"], o["cam"], o["cfg"], og, mass)     # the view's stage-1 bar at the parameters
        tol_sum = tp if tol_sum is None else {p: tol_sum[p] + tp[p] for p in PARAMS}
        singles.append((g, dL))
    assert off == I_total
    bp.backward(torch.from_numpy(np.stack(dLs) if V > 1 else dLs[0]).to(bp.device))
    torch.cuda.synchronize()
    total_bad = total = 0
    for p in PARAMS:
        got = getattr(bp, p).cpu().numpy()
        bad, err = pu.grad_violations(got, og_sum[p])
        total_bad += int(bad.sum()); total += bad.size
        # every element within the bar DERIVED from the stage bars (parity_util.propagated_param_tol; the sum over the
        # views carries one fp32 rounding per added view: 2.4e-7 of the magnitudes)
        ok = pu.e2e_within_propagated(got, og_sum[p], tol_sum[p] + 2.4e-7 * V * np.abs(og_sum[p]))
        assert ok.all(), (p, int((~ok).sum()))
    assert total_bad <= max(4, 2e-5 * total), (total_bad, total)
    # and against the sum of the single-view GPU gradients: the same kernels, but the fp32 atomics of the compositing
    # backward land in another order, so agreement is at the bar of the oracle comparison, not bit for bit
    acc = None
    for g, dL in singles:
        gg = pu.run_gpu_backward(g, dL)
        acc = {p: gg[p].astype(np.float64) for p in PARAMS} if acc is None else {p: acc[p] + gg[p] for p in PARAMS}
    nb = sum(int(pu.grad_violations(getattr(bp, p).cpu().numpy(), acc[p])[0].sum()) for p in PARAMS)
    assert nb <= max(4, 4e-5 * total), (nb, total)
    return bp


def test_batch_of_two_views_config3_reduced():
    batch_parity(scenes.make_scene(3, n_override=20000, image_override=(250, 130)), [0, 1])


def test_batch_of_two_views_with_tile_cull():
    batch_parity(scenes.make_scene(3, n_override=20000, image_override=(250, 130)), [1, 0], dict(tile_cull=1))


def test_batch_of_four_views_config5_reduced():
    batch_parity(scenes.make_scene(5, n_override=30000, image_override=(480, 270)), [0, 1, 2, 3], dict(tile_cull=1))


def test_batch_of_one_is_the_single_view_path():
    sc = scenes.make_scene(1)
    batch_parity(sc, [0])


def test_batch_ut_fisheye_views():
    batch_parity(scenes.make_scene(4, n_override=20000, image_override=(250, 130)), [0, 1], dict(tile_cull=1))


def test_batch_of_four_views_config5_full_size_equals_single_views():
    """BASELINE.json configs[4] at full size (3 M Gaussians, four 1080p views, > 4 x 10^8 candidate pairs) in the launch
    configuration `bench.py --config 5 --views 4` times: every view of the batch equals its single-view run bit for bit
    (lists, image, final_T, n_contrib; the single-view runs are checked against the oracle element by element in
    tests/test_gpu_parity.py), and the summed gradients agree with the sum of the single-view gradients."""
    import torch
    from paper_2606_11529_b200 import pipeline
    sc = scenes.make_scene(5)
    cfg = dict(scenes.default_render_config(sc), tile_cull=1)
    params = pipeline.scene_to_device(sc)
    V, N = 4, sc.N
    bp = pipeline.SplatPipeline(N, sc.cameras[:V], cfg)
    bp.forward(*params)
    T = bp.T // V
    gen = torch.Generator(device="cpu").manual_seed(9)
    dL = (torch.rand(V, bp.H, bp.W, 3, generator=gen) * 2 - 1).to(bp.device)
    bp.backward(dL)
    torch.cuda.synchronize()
    off = 0
    acc = {p: torch.zeros_like(getattr(bp, p), dtype=torch.float64) for p in PARAMS}
    for k in range(V):
        sp = pipeline.SplatPipeline(N, sc.cameras[k], cfg)
        sp.forward(*params)
        I = sp.num_pairs
        assert torch.equal(bp.keys_sorted[off:off + I] - ((k * T) << 32), sp.keys_sorted[:I])
        assert torch.equal(bp.vals_sorted[off:off + I] - k * N, sp.vals_sorted[:I])
        assert torch.equal(bp.image[k], sp.image) and torch.equal(bp.final_T[k], sp.final_T)
        assert torch.equal(bp.n_contrib[k], sp.n_contrib)
        off += I
        sp.backward(dL[k].contiguous())
        for p in PARAMS:
            acc[p] += getattr(sp, p).double()
        del sp
    assert off == bp.num_pairs > 2.5e8
    total = nb = 0
    for p in PARAMS:
        bad, _ = pu.grad_violations(getattr(bp, p).cpu().numpy(), acc[p].cpu().numpy())
        nb += int(bad.sum()); total += bad.size
    assert nb <= 4e-5 * total, (nb, total)


def test_batch_of_two_views_with_rendered_features():
    """f3 x f3: depth image and accumulated opacity for a batch of views (FEAT kernels over V T tiles, xpr_depth_bwd once
    per view).  Per view the forward equals the single-view GPU run bit for bit; the parameter gradients of the loss
    sum_v (L_v + sum gD_v D_v + sum gA_v A_v) equal the oracle's sum over the views of backward_da (reading C31, C32)."""
    import torch
    from paper_2606_11529_b200 import pipeline
    sc = scenes.make_scene(3, n_override=20000, image_override=(250, 130))
    views, N = [0, 1], sc.N
    cfg = dict(scenes.default_render_config(sc), tile_cull=1, features=1)
    params = pipeline.scene_to_device(sc)
    bp = pipeline.SplatPipeline(N, [sc.cameras[v] for v in views], cfg)
    bp.forward(*params)
    torch.cuda.synchronize()
    rng = np.random.default_rng(77)
    dLs, gDs, gAs, og_sum = [], [], [], None
    for k, v in enumerate(views):
        g = pu.run_gpu(sc, v, dict(tile_cull=1, features=1))
        p1 = g["pipe"]
        assert torch.equal(bp.image[k], p1.image) and torch.equal(bp.final_T[k], p1.final_T)
        assert torch.equal(bp.depth_img[k], p1.depth_img) and torch.equal(bp.alpha_img[k], p1.alpha_img)
        assert float(bp.depth_img[k].max()) > 0
        o = pu.run_oracle(sc, v, dict(tile_cull=1))
        o["fwd"].update(xo.rasterize_fwd_da(o["proj"], o["binned"], o["cam"], o["cfg"], np.float32))
        _, dL = scenes.loss_and_grad(sc.loss, o["fwd"]["image"], sc.target(v))
        H, W = dL.shape[:2]
        gD, gA = rng.uniform(-1, 1, (H, W)).astype(np.float32), rng.uniform(-1, 1, (H, W)).astype(np.float32)
        frag = (o["fwd"]["fragile"] & (pu.FRAG_EXIT | pu.FRAG_CLAMP)) != 0
        dL = np.where(frag[..., None], 0.0, dL).astype(np.float32)
        gD = np.where(frag, 0.0, gD).astype(np.float32); gA = np.where(frag, 0.0, gA).astype(np.float32)
        dLs.append(dL); gDs.append(gD); gAs.append(gA)
        og = xo.backward_da(o["arrays"], o, dL, gD, gA, o["cam"], o["cfg"], np.float32)
        og_sum = {p: og[p].copy() for p in PARAMS} if og_sum is None else {p: og_sum[p] + og[p] for p in PARAMS}
    t = lambda a: torch.from_numpy(np.stack(a)).to(bp.device)
    bp.backward(t(dLs), t(gDs), t(gAs))
    torch.cuda.synchronize()
    total = bad = 0
    for p in PARAMS:
        got = getattr(bp, p).cpu().numpy()
        assert np.isfinite(got).all()
        b, _ = pu.grad_violations(got, og_sum[p])
        bad += int(b.sum()); total += b.size
    assert np.abs(og_sum["g_means"]).max() > 0
    assert bad <= max(4, 2e-5 * total), (bad, total)
