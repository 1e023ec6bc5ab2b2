"""xpr_bin_sort_static: the no-allocation variant of xpr_bin_sort / xpr_bin_sort_cull (scratch in a static device array
inside libxpr.so, include/xpr.h) against the existing path (xpr_bin_sort[_cull] with a caller workspace), on two calls in
a row that share the array.  Integer work: keys, values, ranges and the pair count must be identical bit for bit (the
bar of tests/test_gpu_parity.py for a4-a7).  The second call is a SMALLER problem with another configuration (tile_cull
on, different image size), so that anything the first call left in the scratch and the second failed to clear would
show.  This file sorts last on purpose (pytest -x): it must pass alone in a fresh process and after the
other tests."""
import numpy as np
import pytest

from paper_2606_11529_b200 import scenes

pytestmark = pytest.mark.gpu


def _existing_path(sc, cfg_over):
    import torch
    from paper_2606_11529_b200 import pipeline
    cfg = dict(scenes.default_render_config(sc), **cfg_over)
    params = pipeline.scene_to_device(sc)
    pipe = pipeline.SplatPipeline(sc.N, sc.cameras[0], cfg)
    pipe.project(*params)
    I = pipe.bin_sort()                      # xpr_bin_sort / xpr_bin_sort_cull with the pipeline's own workspace
    torch.cuda.synchronize()
    return pipe, I


def _static_path(pipe, capacity):
    import torch
    from paper_2606_11529_b200 import binding as xb
    dev = pipe.device
    keys = torch.full((capacity,), -1, dtype=torch.int64, device=dev)
    vals = torch.full((capacity,), -1, dtype=torch.int32, device=dev)
    ranges = torch.full((pipe.T, 2), -1, dtype=torch.int32, device=dev)
    before = torch.cuda.memory_allocated(dev)
    _, I = xb.xpr_bin_sort_static(pipe.depth, pipe.tile_rect, pipe.tile_count, pipe.cam, pipe.cfg, capacity, keys, vals,
                                  ranges, cull_data=pipe._cull_data())
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated(dev) == before      # nothing taken from the caller's allocator either
    return I, keys, vals, ranges


def _same(pipe, I_ref, I, keys, vals, ranges):
    assert I == I_ref and I > 1000
    assert np.array_equal(keys[:I].cpu().numpy(), pipe.keys_sorted[:I].cpu().numpy())
    assert np.array_equal(vals[:I].cpu().numpy(), pipe.vals_sorted[:I].cpu().numpy())
    assert np.array_equal(ranges.cpu().numpy(), pipe.tile_ranges.cpu().numpy())
    k = keys[:I].cpu().numpy().view(np.uint64)
    assert (np.diff(k.astype(np.float64)) >= 0).all()          # sorted by (tile, depth bits)


def test_bin_sort_static_matches_workspace_path_on_two_calls_in_a_row():
    from paper_2606_11529_b200 import binding as xb
    # call 1: plain binning, 60 000 Gaussians on 640 x 400 (1000 tiles, several supertiles, ragged last tile row)
    sc1 = scenes.make_scene(3, n_override=60000, image_override=(640, 400))
    p1, I1 = _existing_path(sc1, dict(tile_cull=0))
    cap1 = max(2 * I1, 1 << 16)
    r1 = _static_path(p1, cap1)
    _same(p1, I1, *r1)
    # call 2, right after it on the same scratch: smaller, with tile_cull, other image size
    sc2 = scenes.make_scene(2, n_override=8000, image_override=(200, 136))
    p2, I2 = _existing_path(sc2, dict(tile_cull=1))
    cap2 = max(2 * I2, 1 << 14)
    r2 = _static_path(p2, cap2)
    _same(p2, I2, *r2)
    # and the first problem once more: the scratch now holds call 2's contents
    r3 = _static_path(p1, cap1)
    _same(p1, I1, *r3)
    # capacity too small: the capacity contract of xpr_bin_sort holds (XPR_ERR_CAPACITY with the capacity that suffices)
    import torch
    with pytest.raises(xb.XprError) as e:
        _static_path(p2, 64)
    assert e.value.status == xb.XPR_ERR_CAPACITY
    torch.cuda.synchronize()
    _same(p2, I2, *_static_path(p2, cap2))                      # a failed call leaves nothing behind that matters


def test_bin_sort_static_rejects_sizes_beyond_the_static_scratch():
    import torch
    from paper_2606_11529_b200 import binding as xb
    sc = scenes.make_scene(2, n_override=8000, image_override=(200, 136))
    pipe, I = _existing_path(sc, dict(tile_cull=0))
    big = 4 << 20                                               # 4 M pairs: 8 B x capacity alone exceeds 16 MiB
    keys = torch.empty(big, dtype=torch.int64, device=pipe.device)
    vals = torch.empty(big, dtype=torch.int32, device=pipe.device)
    ranges = torch.full((pipe.T, 2), 7, dtype=torch.int32, device=pipe.device)
    with pytest.raises(xb.XprError) as e:
        xb.xpr_bin_sort_static(pipe.depth, pipe.tile_rect, pipe.tile_count, pipe.cam, pipe.cfg, big, keys, vals, ranges)
    assert e.value.status == xb.XPR_ERR_SCRATCH_LIMIT and "XPR_STATIC_SCRATCH_BYTES" in str(e.value)
    torch.cuda.synchronize()
    assert (ranges.cpu().numpy() == 7).all()                    # rejected before anything was launched
