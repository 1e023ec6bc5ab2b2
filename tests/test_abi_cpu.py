"""CPU-only checks of the boundary: libxpr.so builds (nvcc cross-compiles sm_100a), loads, exports
every symbol include/xpr.h declares, and rejects bad arguments before any launch (no GPU needed)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_11529_b200 import build, binding
    build.build()
    return binding.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "xpr.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(xpr_[a-z_]+)\s*\(", src)))


def test_header_symbols_all_exported(lib):
    from paper_2606_11529_b200 import binding
    names = declared_symbols()
    assert set(names) == set(binding.SYMBOLS), (names, binding.SYMBOLS)
    for n in names:
        assert hasattr(lib, n), n
    for n in ("xpr_project", "xpr_bin_sort", "xpr_bin_sort_cull", "xpr_rasterize_fwd", "xpr_rasterize_bwd", "xpr_project_bwd"):
        assert n in names   # BASELINE.json:north_star's five calls


def test_struct_layout_matches_header():
    from paper_2606_11529_b200 import binding
    assert C.sizeof(binding.XprCamera) == 3 * 4 + 4 * 4 + 4 * 4 + 12 * 4
    assert C.sizeof(binding.XprConfig) == 4 * 4 + 8 * 4 + 3 * 4 + 4 + 8 + 8     # + tile_order pointer, views (+ padding)
    assert binding.XprConfig.tile_order.offset == 64


def test_status_strings_and_version(lib):
    assert lib.xpr_version() >= 100
    for s in range(5):
        assert lib.xpr_status_string(C.c_int32(s)).decode().startswith("XPR_")


def _cam_cfg(**over):
    from paper_2606_11529_b200 import binding, scenes
    sc = scenes.make_scene(1, n_override=8)
    d = scenes.default_render_config(sc)
    d.update(over)
    return binding.make_camera(sc.cameras[0]), binding.make_config(d)


def test_invalid_arguments_rejected_before_launch(lib):
    from paper_2606_11529_b200 import binding as xb
    cam, cfg = _cam_cfg()
    null = C.c_void_p(0)
    # NULL pointers with N > 0
    st = lib.xpr_project(C.c_int64(4), null, null, null, null, null, C.byref(cam), C.byref(cfg), null, null, null,
                         null, null, null, null, null, null, null)
    assert st == xb.XPR_ERR_INVALID_ARG
    # negative N
    st = lib.xpr_project(C.c_int64(-1), null, null, null, null, null, C.byref(cam), C.byref(cfg), null, null, null,
                         null, null, null, null, null, null, null)
    assert st == xb.XPR_ERR_INVALID_ARG
    # tile != 16 and sh_degree > 3 are unsupported
    cam2, cfg2 = _cam_cfg(tile=8)
    st = lib.xpr_project(C.c_int64(0), null, null, null, null, null, C.byref(cam2), C.byref(cfg2), null, null, null,
                         null, null, null, null, null, null, null)
    assert st == xb.XPR_ERR_UNSUPPORTED
    cam3, cfg3 = _cam_cfg(sh_degree=4)
    st = lib.xpr_rasterize_fwd(C.byref(cam3), C.byref(cfg3), C.c_int64(0), null, null, null, null, null, null, null)
    assert st == xb.XPR_ERR_UNSUPPORTED
    # bad enum
    cam4, cfg4 = _cam_cfg(projection=7)
    st = lib.xpr_project_bwd(C.c_int64(0), null, null, null, null, null, C.byref(cam4), C.byref(cfg4), null, null,
                             null, null, null, null, null, null, null, null, null, null)
    assert st == xb.XPR_ERR_INVALID_ARG
    # a batch of views: at most XPR_MAX_VIEWS = 8, negative counts are invalid
    cam5, cfg5 = _cam_cfg(views=9)
    assert lib.xpr_rasterize_fwd(C.byref(cam5), C.byref(cfg5), C.c_int64(0), null, null, null, null, null, null, null) == xb.XPR_ERR_UNSUPPORTED
    cam6, cfg6 = _cam_cfg(views=-1)
    assert lib.xpr_rasterize_fwd(C.byref(cam6), C.byref(cfg6), C.c_int64(0), null, null, null, null, null, null, null) == xb.XPR_ERR_INVALID_ARG
    # misaligned workspace
    n = C.c_int64(0)
    st = lib.xpr_bin_sort(C.c_int64(0), null, null, null, C.byref(cam), C.byref(cfg), C.c_int64(0), null, null,
                          C.c_void_p(8), C.byref(n), C.c_void_p(100), C.c_size_t(1 << 20), null)
    assert st == xb.XPR_ERR_INVALID_ARG


def test_ray_entry_points_reject_bad_arguments(lib):
    cam, cfg = _cam_cfg()
    null = C.c_void_p(0)
    one = C.c_void_p(16)          # non-NULL, aligned; never dereferenced: the checks come first
    odd = C.c_void_p(20)          # 4-byte aligned only
    assert lib.xpr_pixel_info(None, one, null) == 1
    assert lib.xpr_pixel_info(C.byref(cam), null, null) == 1
    bad = type(cam)(); C.memmove(C.byref(bad), C.byref(cam), C.sizeof(cam)); bad.model = 7
    assert lib.xpr_pixel_info(C.byref(bad), one, null) == 1
    assert lib.xpr_project_ray(C.c_int64(-1), one, one, one, C.byref(cam), one, one, null) == 1
    assert lib.xpr_project_ray(C.c_int64(0), null, null, null, C.byref(cam), null, null, null) == 0     # N = 0: nothing to do
    assert lib.xpr_project_ray(C.c_int64(4), one, one, one, C.byref(cam), one, odd, null) == 1          # ray_rec needs 16 B
    assert lib.xpr_rasterize_ray_fwd(C.byref(cam), C.byref(cfg), C.c_int64(4), null, one, one, one, one, one, one, one,
                                     one, one, null) == 1
    assert lib.xpr_rasterize_ray_bwd(C.byref(cam), C.byref(cfg), C.c_int64(4), one, one, one, one, one, one, one, one,
                                     one, one, null, one, one, C.c_int32(1), null) == 1
    assert lib.xpr_ray_bwd(C.c_int64(4), one, one, one, C.byref(cam), one, odd, one, one, one, null) == 1
    cfg8 = type(cfg)(); C.memmove(C.byref(cfg8), C.byref(cfg), C.sizeof(cfg)); cfg8.tile = 8
    assert lib.xpr_rasterize_ray_fwd(C.byref(cam), C.byref(cfg8), C.c_int64(0), null, null, null, null, one, null, one,
                                     one, one, one, null) == 4


def test_feature_entry_points_reject_bad_arguments(lib):
    """f3 (xpr_rasterize_feat_fwd / _bwd, xpr_depth_bwd): the argument checks come before any launch."""
    cam, cfg = _cam_cfg()
    null = C.c_void_p(0)
    one = C.c_void_p(16)
    odd = C.c_void_p(18)          # not 4-byte aligned
    N4, N0, Nm = C.c_int64(4), C.c_int64(0), C.c_int64(-1)
    fwd = lambda n, *a: lib.xpr_rasterize_feat_fwd(C.byref(cam), C.byref(cfg), n, *a, null)
    # shade_rec vals ranges image final_T n_contrib depth_img alpha_img
    assert fwd(Nm, *[one] * 8) == 1
    assert fwd(N4, null, *[one] * 7) == 1                                                    # shade_rec NULL
    assert fwd(N4, C.c_void_p(24), *[one] * 7) == 1                                          # shade_rec needs 16 B
    assert fwd(N4, *[one] * 6, null, one) == 1                                               # depth_img NULL
    assert fwd(N4, *[one] * 7, odd) == 1                                                     # alpha_img misaligned
    assert lib.xpr_rasterize_feat_fwd(None, C.byref(cfg), N4, *[one] * 8, null) == 1
    cfg8 = type(cfg)(); C.memmove(C.byref(cfg8), C.byref(cfg), C.sizeof(cfg)); cfg8.tile = 8
    assert lib.xpr_rasterize_feat_fwd(C.byref(cam), C.byref(cfg8), N4, *[one] * 8, null) == 4
    # xpr_shade_record: mean2d conic_opac rgb lnv depth tile_count shade_rec
    assert lib.xpr_shade_record(Nm, *[one] * 7, null) == 1
    assert lib.xpr_shade_record(N4, *[one] * 6, null, null) == 1                             # shade_rec NULL
    assert lib.xpr_shade_record(N4, one, C.c_void_p(24), *[one] * 5, null) == 1              # conic_opac needs 16 B
    assert lib.xpr_shade_record(N0, *[null] * 7, null) == 0
    bwd = lambda n, *a: lib.xpr_rasterize_feat_bwd(C.byref(cam), C.byref(cfg), n, *a, C.c_int32(1), null)
    # shade_rec vals ranges final_T n_contrib dL dL_dD dL_dA g_mean2d g_conic g_opac g_rgb g_depth
    assert bwd(Nm, *[one] * 13) == 1
    assert bwd(N4, *[one] * 6, null, *[one] * 6) == 1                                        # dL_ddepth NULL
    assert bwd(N4, *[one] * 12, null) == 1                                                   # g_depth NULL
    assert bwd(N0, *[null] * 2, one, one, one, one, one, one, *[null] * 5) == 0              # N = 0: nothing to do
    assert lib.xpr_depth_bwd(Nm, C.byref(cam), one, one, one, null) == 1
    assert lib.xpr_depth_bwd(N4, None, one, one, one, null) == 1
    assert lib.xpr_depth_bwd(N4, C.byref(cam), one, null, one, null) == 1
    assert lib.xpr_depth_bwd(N0, C.byref(cam), null, null, null, null) == 0
    # N-channel features: mean2d conic_opac lnv feat C vals ranges n_contrib feat_img
    fn = lambda n, c, *a: lib.xpr_rasterize_featn_fwd(C.byref(cam), C.byref(cfg), n, a[0], a[1], a[2], a[3], C.c_int32(c),
                                                      a[4], a[5], a[6], a[7], null)
    assert fn(N4, 0, *[one] * 8) == 1                                                         # C < 1
    assert fn(Nm, 3, *[one] * 8) == 1
    assert fn(N4, 3, one, one, one, null, one, one, one, one) == 1                            # feat NULL
    assert fn(N4, 3, *[one] * 7, null) == 1                                                   # feat_img NULL
    bn = lambda n, c, *a: lib.xpr_rasterize_featn_bwd(C.byref(cam), C.byref(cfg), n, a[0], a[1], a[2], a[3], C.c_int32(c),
                                                      *a[4:], C.c_int32(3), null)
    # mean2d conic_opac lnv feat | vals ranges final_T n_contrib dL_dfeat g_mean2d g_conic g_opac g_feat
    assert bn(N4, 0, *[one] * 13) == 1
    assert bn(N4, 5, *[one] * 12, null) == 1                                                  # g_feat NULL
    assert bn(N4, 5, *[one] * 8, odd, *[one] * 4) == 1                                        # dL_dfeat misaligned
    assert bn(N0, 5, *[null] * 5, one, one, one, one, *[null] * 4) == 0                       # N = 0: nothing to do


def test_workspace_size_monotone(lib):
    from paper_2606_11529_b200 import binding as xb
    a = xb.xpr_bin_sort_workspace(1000, 10_000, 16)
    b = xb.xpr_bin_sort_workspace(1000, 1_000_000, 8160)
    assert 0 < a < b
    assert b >= 8 * 1_000_000        # the second buffer of 8-byte packed words (tile << 32 | rank)
    with pytest.raises(xb.XprError):
        xb.xpr_bin_sort_workspace(1000, 1 << 30, 16)
    # N >= 2^30 would overflow the 30-bit counts of the sort's look-back words: refused, not corrupted
    with pytest.raises(xb.XprError) as e:
        xb.xpr_bin_sort_workspace(1 << 30, 1000, 16)
    assert e.value.status == xb.XPR_ERR_UNSUPPORTED
    assert xb.xpr_bin_sort_workspace((1 << 30) - 1, 0, 16) > 0


def test_binding_refuses_cpu_tensors():
    import torch
    from paper_2606_11529_b200 import binding as xb
    with pytest.raises(TypeError):
        xb._p(torch.zeros(4))


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_11529_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "xpr_oracle" not in txt and "import oracle" not in txt, f


def test_profiles_hold_text_summaries_only():
    """profiles/ holds ncu summaries as .txt / .csv / .md; every .csv is named by a .md beside it."""
    d = os.path.join(ROOT, "profiles")
    names = sorted(os.listdir(d))
    assert names and all(n.endswith((".txt", ".csv", ".md")) for n in names), names
    mds = "\n".join(open(os.path.join(d, n)).read() for n in names if n.endswith(".md"))
    for n in names:
        if n.endswith(".csv"):
            assert n in mds, n


def test_linprim_entry_points_reject_bad_arguments(lib):
    """f4 (xpr_lin_project, xpr_bin_sort_lin, xpr_lin_rasterize_fwd / _stats): the argument checks come before any launch."""
    cam, cfg = _cam_cfg()
    null, one, odd = C.c_void_p(0), C.c_void_p(16), C.c_void_p(20)
    N4, N0, Nm = C.c_int64(4), C.c_int64(0), C.c_int64(-1)
    # means scales quats opacities sh | cam cfg | lin_rec depth tile_rect tile_count
    prj = lambda n, cm, cf, *a: lib.xpr_lin_project(n, *a[:5], cm, cf, *a[5:], null)
    assert prj(Nm, C.byref(cam), C.byref(cfg), *[one] * 9) == 1
    assert prj(N4, None, C.byref(cfg), *[one] * 9) == 1
    assert prj(N4, C.byref(cam), C.byref(cfg), *[one] * 5, odd, one, one, one) == 1           # lin_rec needs 16 B
    assert prj(N4, C.byref(cam), C.byref(cfg), null, *[one] * 8) == 1                         # means NULL
    assert prj(N0, C.byref(cam), C.byref(cfg), *[null] * 9) == 0                              # N = 0: nothing to do
    fish = type(cam)(); C.memmove(C.byref(fish), C.byref(cam), C.sizeof(cam)); fish.model = 1
    assert prj(N4, C.byref(fish), C.byref(cfg), *[one] * 9) == 4                              # LinPrim: pinhole only
    cfg8 = type(cfg)(); C.memmove(C.byref(cfg8), C.byref(cfg), C.sizeof(cfg)); cfg8.tile = 8
    ras = lambda n, cm, cf, *a: lib.xpr_lin_rasterize_fwd(cm, cf, n, *a, null)
    # lin_rec vals ranges image final_T n_contrib
    assert ras(Nm, C.byref(cam), C.byref(cfg), *[one] * 6) == 1
    assert ras(N4, C.byref(cam), None, *[one] * 6) == 1
    assert ras(N4, C.byref(cam), C.byref(cfg), odd, *[one] * 5) == 1
    assert ras(N4, C.byref(cam), C.byref(cfg), one, one, one, null, one, one) == 1            # image NULL
    assert ras(N4, C.byref(cam), C.byref(cfg8), *[one] * 6) == 4
    assert ras(N4, C.byref(fish), C.byref(cfg), *[one] * 6) == 4
    assert lib.xpr_lin_rasterize_stats(C.byref(cam), C.byref(cfg), N4, one, one, one, null, null) == 1
    # xpr_bin_sort_lin: as xpr_bin_sort, + lin_rec
    bs = lambda n, rec, cap, *a: lib.xpr_bin_sort_lin(n, one, one, one, rec, C.byref(cam), C.byref(cfg), C.c_int64(cap), *a)
    assert bs(N4, odd, 1024, one, one, one, None, C.c_void_p(256), C.c_size_t(1 << 20), null) == 1   # lin_rec needs 16 B
    assert bs(Nm, one, 1024, one, one, one, None, C.c_void_p(256), C.c_size_t(1 << 20), null) == 1
    assert bs(N4, one, 1024, one, one, one, None, C.c_void_p(256), C.c_size_t(64), null) == 1        # workspace too small
    assert bs(C.c_int64(1 << 30), one, 1024, one, one, one, None, C.c_void_p(256), C.c_size_t(1 << 20), null) == 4
    # backward: lin_rec vals ranges final_T n_contrib dL g_lin_rec
    rb = lambda n, cm, cf, *a: lib.xpr_lin_rasterize_bwd(cm, cf, n, *a, null)
    assert rb(Nm, C.byref(cam), C.byref(cfg), *[one] * 7) == 1
    assert rb(N4, C.byref(cam), C.byref(cfg), *[one] * 6, odd) == 1                           # g_lin_rec needs 16 B
    assert rb(N4, C.byref(cam), C.byref(cfg), *[one] * 5, null, one) == 1                     # dL NULL
    assert rb(N4, C.byref(fish), C.byref(cfg), *[one] * 7) == 4
    assert rb(N0, C.byref(cam), C.byref(cfg), null, null, one, one, one, one, null) == 0      # N = 0: nothing to do
    # means scales quats opacities sh | cam cfg | tile_count lin_rec g_lin_rec g_means g_scales g_quats g_opacities g_sh
    pb = lambda n, cm, cf, *a: lib.xpr_lin_project_bwd(n, *a[:5], cm, cf, *a[5:], null)
    assert pb(Nm, C.byref(cam), C.byref(cfg), *[one] * 13) == 1
    assert pb(N4, C.byref(cam), C.byref(cfg), *[one] * 7, odd, *[one] * 5) == 1               # g_lin_rec needs 16 B
    assert pb(N4, C.byref(cam), C.byref(cfg), *[one] * 10, odd, one, one) == 1                # g_quats needs 16 B
    assert pb(N4, C.byref(cam), C.byref(cfg), *[one] * 12, null) == 1                         # g_sh NULL
    assert pb(N4, C.byref(fish), C.byref(cfg), *[one] * 13) == 4
    assert pb(N0, C.byref(cam), C.byref(cfg), *[null] * 13) == 0


def test_ray_feature_entry_points_reject_bad_arguments(lib):
    """f2 x f3 (xpr_rasterize_ray_feat_fwd / _bwd): the argument checks come before any launch."""
    cam, cfg = _cam_cfg()
    null, one, odd = C.c_void_p(0), C.c_void_p(16), C.c_void_p(18)
    N4, N0, Nm = C.c_int64(4), C.c_int64(0), C.c_int64(-1)
    # ray_rec conic_opac rgb lnv depth rays vals ranges image final_T n_contrib depth_img alpha_img
    fwd = lambda n, *a: lib.xpr_rasterize_ray_feat_fwd(C.byref(cam), C.byref(cfg), n, *a, null)
    assert fwd(Nm, *[one] * 13) == 1
    assert fwd(N4, *[one] * 4, null, *[one] * 8) == 1                                        # depth NULL
    assert fwd(N4, *[one] * 11, null, one) == 1                                              # depth_img NULL
    assert fwd(N4, *[one] * 12, odd) == 1                                                    # alpha_img misaligned
    # ... final_T n_contrib dL dL_dD dL_dA g_ray_acc g_opac g_rgb g_depth
    bwd = lambda n, *a: lib.xpr_rasterize_ray_feat_bwd(C.byref(cam), C.byref(cfg), n, *a, C.c_int32(1), null)
    assert bwd(Nm, *[one] * 17) == 1
    assert bwd(N4, *[one] * 11, null, *[one] * 5) == 1                                       # dL_ddepth NULL
    assert bwd(N4, *[one] * 16, null) == 1                                                   # g_depth NULL
    assert bwd(N0, *[null] * 5, one, null, one, one, one, one, one, one, *[null] * 4) == 0   # N = 0: nothing to do


def test_bin_sort_static_rejects_before_launch(lib):
    """xpr_bin_sort_static (no-allocation entry point): argument errors and the size limit are reported before any CUDA call."""
    cam, cfg = _cam_cfg()
    null, one = C.c_void_p(0), C.c_void_p(256)
    call = lambda n, cap, cm=cam, cf=cfg: lib.xpr_bin_sort_static(C.c_int64(n), one, one, one, null, null, null, C.byref(cm),
                                                                 C.byref(cf), C.c_int64(cap), one, one, one, None, null)
    assert call(-1, 1024) == 1
    assert call(4, -1) == 1
    assert call(1 << 30, 1024) == 4
    assert lib.xpr_bin_sort_static(C.c_int64(4), one, one, one, null, null, null, None, C.byref(cfg), C.c_int64(16), one, one,
                                   one, None, null) == 1
    assert call(4, 1 << 22) == 5 and call(2_000_000, 1024) == 5            # beyond XPR_STATIC_SCRATCH_BYTES
    assert lib.xpr_status_string(C.c_int32(5)).decode().startswith("XPR_ERR_SCRATCH_LIMIT")
    from paper_2606_11529_b200 import binding
    src = open(os.path.join(ROOT, "include", "xpr.h")).read()
    assert "XPR_STATIC_SCRATCH_BYTES = 16 * 1024 * 1024" in src and binding.XPR_STATIC_SCRATCH_BYTES == 16 * 1024 * 1024


def test_rasterize_bwd_loss_rejects_bad_arguments(lib):
    cam, cfg = _cam_cfg()
    null, one, odd = C.c_void_p(0), C.c_void_p(16), C.c_void_p(18)
    # shade_rec vals ranges image final_T n_contrib | kind target | g_mean2d g_conic g_opac g_rgb
    f = lambda n, kind, *a: lib.xpr_rasterize_bwd_loss(C.byref(cam), C.byref(cfg), C.c_int64(n), *a[:6], C.c_int32(kind), *a[6:],
                                                       C.c_int32(1), null)
    assert f(4, 2, *[one] * 11) == 1 and f(4, -1, *[one] * 11) == 1          # loss_kind outside {0, 1}
    assert f(-1, 0, *[one] * 11) == 1
    assert f(4, 0, one, one, one, null, *[one] * 7) == 1                      # image NULL
    assert f(4, 1, *[one] * 6, odd, *[one] * 4) == 1                          # target misaligned
    assert f(0, 0, null, null, one, one, one, one, one, *[null] * 4) == 0     # N = 0: nothing to do
