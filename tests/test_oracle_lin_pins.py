"""Pin P18 of the ORACLE's XPR-LinPrim forward (oracle/xpr_oracle_lin.inc; PAPER A.1.3 L506-697, Eq. 2), against what
the geometry fixes -- never against the oracle's own formulas:
  a  the chord of the ray through a pixel equals the chord obtained by clipping that ray against the eight faces of the
     octahedron in WORLD space (numpy, independent parametrisation) for small distant primitives, where the paper's
     linearisation A = J W R diag(s) is exact to first order; on the optical axis through the centre of an axis-aligned
     octahedron it is 2 s_z, and alpha there is 1 - (1 - 0.99 o)^(s_z / min s) -- 0.99 o along the shortest axis (L522-528);
  b  Eq. 2's per-tile bound is >= the densely sampled maximum chord over the tile, and a culled pair has alpha <
     alpha_thresh at every pixel of the tile (L633-683);
  c  the footprint rectangle contains every pixel with a non-zero chord; the image is unchanged by tile_cull (L683);
  d  transmittance-product / opacity-sum invariants of the compositing loop (L86) with rgb = 1.
"""
import math
import types

import numpy as np
import pytest

import xpr_oracle as xo
from paper_2606_11529_b200 import scenes

AT = 1.0 / 255.0
C0 = 0.28209479177387814


def cam_obj(W=96, H=64, fx=300.0, fy=300.0, w2c=None):
    if w2c is None:
        w2c = np.array([[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 0]], np.float64)
    return types.SimpleNamespace(model=0, width=W, height=H, fx=fx, fy=fy, cx=W / 2, cy=H / 2, k=(0, 0, 0, 0),
                                 w2c=np.asarray(w2c, np.float64))


def cfg_dict(**kw):
    d = dict(projection=0, sh_degree=0, tile=16, antialias=0, alpha_thresh=AT, alpha_max=0.99, t_min=1e-4, z_near=0.2,
             lowpass=0.3, ut_alpha=1.0, ut_beta=2.0, ut_kappa=0.0, bg=(0.0, 0.0, 0.0), tile_cull=0)
    d.update(kw)
    return d


def prim(mu, s, q=(1, 0, 0, 0), o=0.8, rgb=(1.0, 1.0, 1.0)):
    q = np.asarray(q, np.float64); q = q / np.linalg.norm(q)
    return dict(means=np.asarray(mu, np.float64).reshape(1, 3), scales=np.asarray(s, np.float64).reshape(1, 3),
                quats=q.reshape(1, 4), opacities=np.asarray([o], np.float64),
                sh=((np.asarray(rgb, np.float64) - 0.5) / C0).reshape(1, 1, 3))


def world_chord(co, arr, px, py):
    """Chord of the camera ray through pixel centre (px, py) with the octahedron |S^-1 R^T (x - mu)|_1 <= 1, by clipping
    against its eight face half-spaces in world space; measured in Euclidean length along the ray."""
    from scipy.spatial.transform import Rotation
    w, x, y, z = arr["quats"][0]
    R = Rotation.from_quat([x, y, z, w]).as_matrix()
    Wm, t = co.w2c[:, :3], co.w2c[:, 3]
    d_cam = np.array([(px - co.cx) / co.fx, (py - co.cy) / co.fy, 1.0]); d_cam /= np.linalg.norm(d_cam)
    o_w = -Wm.T @ t
    d_w = Wm.T @ d_cam
    Minv = np.diag(1.0 / arr["scales"][0]) @ R.T
    a = Minv @ (o_w - arr["means"][0]); b = Minv @ d_w          # local coordinates u(tau) = a + tau b
    lo, hi = -np.inf, np.inf
    for e in [(s0, s1, s2) for s0 in (1, -1) for s1 in (1, -1) for s2 in (1, -1)]:
        e = np.array(e, float)
        ea, eb = e @ a, e @ b                                    # e.u <= 1
        if abs(eb) < 1e-300:
            if ea > 1: return 0.0
            continue
        tcut = (1 - ea) / eb
        if eb > 0: hi = min(hi, tcut)
        else: lo = max(lo, tcut)
    return max(0.0, hi - lo)


def test_p18a_chord_through_the_centre_and_density():
    s = (0.05, 0.02, 0.08)
    o = 0.6
    co = cam_obj()
    arr = prim((0, 0, 4.0), s, o=o)
    cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict())
    p = xo.lin_project(cam=cam, cfg=cfg, dtype=np.float64, **arr)
    assert p["tile_count"][0] > 0
    rec = p["lin_rec"][0]
    sigma = -math.log(1 - 0.99 * o) / (2 * min(s))
    np.testing.assert_allclose(rec[2], sigma, rtol=1e-13)
    np.testing.assert_allclose(p["depth"][0], 4.0, rtol=1e-14)
    np.testing.assert_allclose(rec[:2], [48.0, 32.0], atol=1e-12)
    x = xo.lin_chord(rec, [[48.0, 32.0]])[0]                      # the ray through the centre runs along local z
    np.testing.assert_allclose(x, sigma * 2 * s[2], rtol=1e-12)
    np.testing.assert_allclose(1 - math.exp(-x), 1 - (1 - 0.99 * o) ** (s[2] / min(s)), rtol=1e-12)
    # along the shortest axis alpha = 0.99 o exactly (L522-528): rotate the primitive so that local y faces the camera
    arr2 = prim((0, 0, 4.0), s, q=(math.cos(math.pi / 4), math.sin(math.pi / 4), 0, 0), o=o)
    rec2 = xo.lin_project(cam=cam, cfg=cfg, dtype=np.float64, **arr2)["lin_rec"][0]
    np.testing.assert_allclose(1 - math.exp(-xo.lin_chord(rec2, [[48.0, 32.0]])[0]), 0.99 * o, rtol=1e-12)


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_p18a_chord_equals_world_space_clipping_for_small_distant_primitives(seed):
    rng = np.random.default_rng(40 + seed)
    w2c = scenes.look_at((0.3, -0.2, -1.0), (0.05, 0.1, 3.0)).astype(np.float64)
    co = cam_obj(W=160, H=128, fx=2500.0, fy=2500.0, w2c=w2c)
    cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict())
    mu = np.array([0.05, 0.1, 3.0]) + rng.normal(0, 0.02, 3)
    s = np.exp(rng.uniform(np.log(0.008), np.log(0.03), 3))      # 5-20 px at distance ~4: the linearisation error is O(s / z)
    arr = prim(mu, s, q=rng.standard_normal(4), o=0.7)
    p = xo.lin_project(cam=cam, cfg=cfg, dtype=np.float64, **arr)
    assert p["tile_count"][0] > 0
    rec = p["lin_rec"][0]
    cx0, cy0 = int(rec[0]), int(rec[1])
    ys, xs = np.mgrid[max(0, cy0 - 40):min(128, cy0 + 40), max(0, cx0 - 40):min(160, cx0 + 40)]
    pix = np.stack([xs.ravel() + 0.5, ys.ravel() + 0.5], 1)
    got = xo.lin_chord(rec, pix) / rec[2]
    ref = np.array([world_chord(co, arr, a, b) for a, b in pix])
    assert ref.max() > 1.2 * s.min() and (ref > 0).sum() > 30
    # first-order agreement: errors scale with s / z (here ~3e-3) times the chord scale
    assert np.abs(got - ref).max() < 0.03 * ref.max(), np.abs(got - ref).max() / ref.max()
    inside = ref > 0.2 * ref.max()
    assert np.abs(got - ref)[inside].mean() < 0.01 * ref.max()
    # footprint (L3): every pixel with a chord lies inside the tile rectangle
    r = p["tile_rect"][0]
    hit = pix[got > 0]
    assert (hit[:, 0] >= 16 * r[0]).all() and (hit[:, 0] < 16 * r[2]).all()
    assert (hit[:, 1] >= 16 * r[1]).all() and (hit[:, 1] < 16 * r[3]).all()


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_p18b_eq2_bound_dominates_the_chord_and_culled_pairs_are_invisible(seed):
    rng = np.random.default_rng(60 + seed)
    co = cam_obj(W=128, H=96, fx=400.0, fy=400.0)
    cam, cfg = xo.make_camera(co), xo.make_config(cfg_dict(tile_cull=1))
    req = -math.log(1 - AT)
    n_cull = n_keep = 0
    for _ in range(30):
        mu = np.array([rng.uniform(-0.5, 0.5), rng.uniform(-0.4, 0.4), rng.uniform(2.0, 4.0)])
        s = np.exp(rng.uniform(np.log(0.005), np.log(0.25), 3))     # flat and needle-like shapes included
        arr = prim(mu, s, q=rng.standard_normal(4), o=float(rng.choice([0.01, 0.02, 0.3, 0.95])))
        p = xo.lin_project(cam=cam, cfg=cfg, dtype=np.float64, **arr)
        if p["tile_count"][0] == 0:
            continue
        rec = p["lin_rec"][0]
        r = p["tile_rect"][0]
        tiles = [(tx, ty) for ty in range(r[1], r[3]) for tx in range(r[0], r[2])]
        keep = xo.lin_tile_keep(rec, tiles, cfg, np.float64)
        for (tx, ty), k in zip(tiles, keep):
            u = np.linspace(0.5, 16.5, 65)                       # dense sampling of the closed tile of Eq. 2 (L6)
            gx, gy = np.meshgrid(16 * tx + u, 16 * ty + u)
            dense = xo.lin_chord(rec, np.stack([gx.ravel(), gy.ravel()], 1)).max()
            centres = np.stack(np.meshgrid(16 * tx + np.arange(16) + 0.5, 16 * ty + np.arange(16) + 0.5), -1).reshape(-1, 2)
            x_pix = xo.lin_chord(rec, centres)
            if k:
                n_keep += 1
            else:
                n_cull += 1
                assert dense < req                               # the bound is an upper bound: culled => max chord below the gate
                assert (1 - np.exp(-x_pix) < AT).all()           # ... hence alpha < alpha_thresh at every pixel (L676-683)
    assert n_cull >= 5 and n_keep > 20


def test_p18c_image_unchanged_by_tile_cull_and_invariants():
    sc = scenes.make_scene(2, n_override=4000, image_override=(160, 160))
    arr = dict(means=sc.means, scales=sc.scales * 3.0, quats=sc.quats, opacities=sc.opacities, sh=sc.sh)
    cam = xo.make_camera(sc.cameras[0])
    d = scenes.default_render_config(sc)
    r0 = xo.render_lin(arr, cam, xo.make_config(dict(d, tile_cull=0)), np.float32)
    r1 = xo.render_lin(arr, cam, xo.make_config(dict(d, tile_cull=1)), np.float32)
    assert 1000 < r1["binned"]["num_pairs"] < r0["binned"]["num_pairs"] - 100      # the boxes of octahedra are tight: a few % culled
    np.testing.assert_array_equal(r0["fwd"]["image"], r1["fwd"]["image"])
    np.testing.assert_array_equal(r0["fwd"]["final_T"], r1["fwd"]["final_T"])
    # P2 analogue: rgb = 1, bg = 0 => image = 1 - final_T (sum alpha_k T_k telescopes)
    arr1 = dict(arr, sh=np.full((sc.N, 1, 3), 0.5 / C0, np.float32))
    r = xo.render_lin(arr1, cam, xo.make_config(dict(d, tile_cull=1, sh_degree=0)), np.float64)
    np.testing.assert_allclose(r["fwd"]["image"][..., 0], 1 - r["fwd"]["final_T"], atol=1e-12)
    assert (r["fwd"]["final_T"] < 0.9).any()
    # keys sorted, ranges partition the pairs
    k = r1["binned"]["keys"]
    assert (np.diff(k.astype(np.int64) >> 32) >= 0).all()
    rg = r1["binned"]["ranges"].astype(np.int64)
    assert (rg[:, 1] - rg[:, 0]).sum() == r1["binned"]["num_pairs"]
