"""Pins P13 for the oracle's tile_cull ("Cull", Listing 1, A.1.1 L435; C8).

The oracle's keep/drop decision is pinned by things other than itself:
  (a) the maximum of alpha over the tile, found by dense sampling of the rectangle in fp64 (brute force),
      agrees with the decision except inside the stated conservative margin;
  (b) no dropped pair has a pixel that passes the per-pixel gate ("alpha(x,y) < alpha_thresh for
      every pixel of a culled primitive-tile pair") -- checked with a formula retyped here, not the oracle's;
  (c) closed forms: an isotropic Gaussian keeps exactly the tiles within distance sigma sqrt(2 lnv) of its mean;
  (d) PAPER L683: removing the entries leaves the composited image unchanged -- bit for bit in fp32.
"""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, os.path.join(ROOT, "oracle"))
sys.path.insert(0, ROOT)

import xpr_oracle as xo  # noqa: E402
from paper_2606_11529_b200 import scenes  # noqa: E402

TS = 16


def random_pairs(rng, n):
    """Gaussians around a tile: means within a few tiles of it, anisotropic conics, lnv in (0, ln 255]."""
    tile = rng.integers(0, 20, (n, 2)).astype(np.int32)
    centre = TS * tile + TS / 2.0
    mean = centre + rng.normal(0, 30.0, (n, 2))
    sig = np.exp(rng.normal(np.log(8.0), 0.9, (n, 2)))
    th = rng.uniform(0, np.pi, n)
    c, s = np.cos(th), np.sin(th)
    cov = np.empty((n, 2, 2))
    cov[:, 0, 0] = c * c * sig[:, 0] ** 2 + s * s * sig[:, 1] ** 2
    cov[:, 1, 1] = s * s * sig[:, 0] ** 2 + c * c * sig[:, 1] ** 2
    cov[:, 0, 1] = cov[:, 1, 0] = c * s * (sig[:, 0] ** 2 - sig[:, 1] ** 2)
    K = np.linalg.inv(cov)
    conic = np.stack([K[:, 0, 0], K[:, 0, 1], K[:, 1, 1]], axis=1)
    lnv = np.log(255.0 * rng.uniform(1.0 / 255.0, 1.0, n))
    return mean, conic, lnv, tile


def brute_min_q(mean, conic, tile, grid=129):
    """min over the pixel-centre hull of the tile of 1/2 d^T K d by dense sampling (fp64)."""
    u = np.linspace(0.5, TS - 0.5, grid)
    gx, gy = np.meshgrid(u, u)
    out = np.empty(len(mean))
    for i in range(len(mean)):
        dx = TS * tile[i, 0] + gx - mean[i, 0]
        dy = TS * tile[i, 1] + gy - mean[i, 1]
        q = 0.5 * (conic[i, 0] * dx * dx + 2 * conic[i, 1] * dx * dy + conic[i, 2] * dy * dy)
        out[i] = q.min()
    return out


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_p13a_decision_matches_dense_sampling_of_the_tile(dtype):
    rng = np.random.default_rng(11)
    mean, conic, lnv, tile = random_pairs(rng, 4000)
    keep = xo.tile_keep(mean, conic, lnv, tile, TS, dtype)
    qmin = brute_min_q(mean, conic, tile)          # sampling can only over-estimate the true minimum
    assert 0.2 < keep.mean() < 0.8                 # both outcomes are exercised
    # dropped => the true minimum exceeds lnv (conservative): sampled min >= true min > lnv
    assert (qmin[~keep] > lnv[~keep]).all()
    # kept => the minimum is within the margin of lnv; the sampled minimum over-estimates by at most the grid step
    h = (TS - 1.0) / 128.0
    lam = 0.5 * (conic[:, 0] + conic[:, 2]) + np.sqrt(0.25 * (conic[:, 0] - conic[:, 2]) ** 2 + conic[:, 1] ** 2)
    slack = np.sqrt(2 * lam * np.maximum(qmin, 0)) * h * np.sqrt(2) + lam * h * h + 1e-3 * (1 + qmin)
    assert (qmin[keep] <= lnv[keep] + slack[keep]).all()
    # and the decision is tight: almost every pair whose sampled minimum is clearly above lnv is dropped
    clearly_out = qmin > lnv * (1 + 1e-3) + slack
    assert (~keep[clearly_out]).mean() > 0.999


def test_p13c_isotropic_closed_form():
    # isotropic Gaussian, sigma = 10 px, o = 0.5: alpha >= 1/255 within r = sigma sqrt(2 ln(255 o))
    sigma, o = 10.0, 0.5
    lnv = np.log(255.0 * o)
    r = sigma * np.sqrt(2 * lnv)
    mean = np.array([100.3, 77.7])
    tiles = np.array([(x, y) for x in range(0, 14) for y in range(0, 12)], np.int32)
    n = len(tiles)
    conic = np.tile([1 / sigma ** 2, 0.0, 1 / sigma ** 2], (n, 1))
    keep = xo.tile_keep(np.tile(mean, (n, 1)), conic, np.full(n, lnv), tiles, TS, np.float64)
    # distance from the mean to the pixel-centre hull of each tile
    lo = TS * tiles + 0.5
    hi = TS * tiles + TS - 0.5
    d = np.linalg.norm(np.maximum(np.maximum(lo - mean, mean - hi), 0.0), axis=1)
    np.testing.assert_array_equal(keep, d <= r * (1 + 1e-5))
    assert keep.sum() not in (0, n)


@pytest.mark.parametrize("config,kw", [(1, {}), (2, dict(n_override=4000, image_override=(160, 160))),
                                       (3, dict(n_override=20000, image_override=(240, 135)))])
def test_p13bd_dropped_pairs_have_no_passing_pixel_and_image_is_unchanged(config, kw):
    sc = scenes.make_scene(config, **kw)
    arr = dict(means=sc.means, scales=sc.scales, quats=sc.quats, opacities=sc.opacities, sh=sc.sh)
    cam = xo.make_camera(sc.cameras[0])
    d = scenes.default_render_config(sc)
    full = xo.render(arr, cam, xo.make_config(dict(d, tile_cull=0)), np.float32)
    cull = xo.render(arr, cam, xo.make_config(dict(d, tile_cull=1)), np.float32)
    nf, nc = full["binned"]["num_pairs"], cull["binned"]["num_pairs"]
    assert 0 < nc < nf
    # (d) PAPER L683: the image, the final transmittance and the gradients do not change -- bit for bit
    np.testing.assert_array_equal(full["fwd"]["image"], cull["fwd"]["image"])
    np.testing.assert_array_equal(full["fwd"]["final_T"], cull["fwd"]["final_T"])
    _, dL = scenes.loss_and_grad(sc.loss, full["fwd"]["image"], sc.target(0))
    gf = xo.backward(arr, full, dL, cam, xo.make_config(dict(d, tile_cull=0)), np.float32)
    gc = xo.backward(arr, cull, dL, cam, xo.make_config(dict(d, tile_cull=1)), np.float32)
    for k in ("g_means", "g_scales", "g_quats", "g_opacities", "g_sh"):      # fp64 sums over tiles, order not fixed
        np.testing.assert_allclose(gf[k], gc[k], rtol=1e-11, atol=1e-13)
    # the surviving pairs are a sub-multiset of the candidates, same order inside every tile
    pf = set(zip((full["binned"]["keys"] >> np.uint64(32)).tolist(), full["binned"]["vals"].tolist()))
    pc = list(zip((cull["binned"]["keys"] >> np.uint64(32)).tolist(), cull["binned"]["vals"].tolist()))
    assert len(set(pc)) == nc and set(pc) <= pf
    # (b) every dropped pair: no pixel centre of the tile passes the gate power >= -lnv (formula retyped here)
    dropped = np.array(sorted(pf - set(pc)), np.int64)
    p = full["proj"]
    W, H = sc.cameras[0].width, sc.cameras[0].height
    TW = (W + TS - 1) // TS
    rng = np.random.default_rng(0)
    for t, g in dropped[rng.choice(len(dropped), size=min(3000, len(dropped)), replace=False)]:
        tx, ty = t % TW, t // TW
        xs = TS * tx + np.arange(TS) + 0.5
        ys = TS * ty + np.arange(TS) + 0.5
        dx = xs[None, :] - np.float64(p["mean2d"][g, 0])
        dy = ys[:, None] - np.float64(p["mean2d"][g, 1])
        A, B, C = [np.float64(v) for v in p["conic"][g]]
        power = -0.5 * (A * dx * dx + C * dy * dy) - B * dx * dy
        assert (power < -np.float64(p["lnv"][g])).all(), (t, g)
