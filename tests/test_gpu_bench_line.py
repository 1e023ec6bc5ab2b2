"""bench.py prints one JSON line with the keys the measurement contract asks for (run on the tiny config)."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*extra):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--config", "1", "--steps", "3", "--warmup", "3",
                          *extra], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    return json.loads(lines[0])


def test_bench_line_ours():
    d = _run()
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert k in d, k
    assert d["n_gpus"] == 1 and d["steps"] == 3 and d["value"] > 0 and d["vs_baseline"] is None
    assert "workload" in d["config"] and "model" not in d["config"]
    assert d["gpu_launches"] == 3 * 15          # 11 launches of xpr_bin_sort (one supertile-digit pass); loss gradient fused
    assert d["config"]["fuse_loss"] == 1 and d["stage_ms"]["loss_grad"] < 0.005
    st = d["ms_per_step_stats"]
    # the stages are timed in a second, instrumented pass and sum to ITS step time
    assert abs(sum(d["stage_ms"].values()) - st["instrumented_ms_per_step"]) < 0.02 * st["instrumented_ms_per_step"]
    r = d["roofline"]
    assert r["bound"] in ("hbm", "alu", "tensor") and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    assert d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0 and d["e2e"]["value"] > 0
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["sample"]


def test_bench_line_reference_arm():
    d = _run("--impl", "reference")
    assert d["impl"] == "reference" and d["value"] > 0 and d["metric"] == "fwd_bwd_megapixels_per_s"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle"


def test_bench_line_ray_evaluation():
    d = _run("--config", "4", "--ray-eval", "1", "--no-cpu-baseline", "--no-e2e")
    assert d["config"]["ray_eval"] == 1 and d["value"] > 0
    assert d["roofline"]["kernel"].startswith("rasterize_ray_")
    assert d["gpu_launches"] == 3 * (16 + 3)    # 1080p: 135 supertiles, one digit pass; + pixel_info, project_ray, ray_bwd


def test_bench_line_rendered_features():
    d = _run("--config", "3", "--features", "1", "--no-cpu-baseline")
    assert d["config"]["features"] == 1 and d["value"] > 0
    assert d["rooflines"]["rasterize_bwd"]["kernel"] == "rasterize_bwd_kernel<FEAT>"
    assert d["gpu_launches"] == 3 * (16 + 1)    # + depth_bwd
    assert d["e2e"]["d2h_bytes_per_step"] > 1920 * 1080 * 4 * 5    # image, D and A all come back


def test_bench_line_reports_n_channel_feature_timings():
    d = _run("--featn", "5", "--no-cpu-baseline", "--no-e2e", "--no-graph")
    assert d["featn"]["C"] == 5 and d["featn"]["fwd_ms"] > 0 and d["featn"]["bwd_ms"] > 0
    assert d["gpu_launches"] == 3 * 15          # the step itself is unchanged


def test_bench_line_batch_of_views():
    d = _run("--config", "5", "--views", "2", "--no-cpu-baseline", "--no-e2e", "--no-graph")
    assert d["config"]["views"] == 2 and d["value"] > 0
    assert d["gpu_launches"] == 3 * 15          # a batch of views costs the launches of one view


def test_bench_line_separate_loss_kernel():
    d = _run("--fuse-loss", "0", "--no-cpu-baseline", "--no-e2e", "--no-graph", "--no-plain")
    assert d["config"]["fuse_loss"] == 0 and d["gpu_launches"] == 3 * 16 and d["stage_ms"]["loss_grad"] > 0.005


def test_bench_line_linprim():
    d = _run("--linprim", "3", "--config", "2")
    assert d["config"]["method"] == "linprim" and d["value"] > 0 and d["config"]["pairs"] > 1000
    assert set(d["stage_ms"]) == {"project", "bin_sort", "rasterize_fwd", "loss_grad", "rasterize_bwd", "project_bwd"}
    assert d["roofline"]["kernel"] == "lin_rasterize_fwd_kernel" and 0 < d["roofline"]["frac"] < 1
    assert d["counts"]["visited"] >= d["counts"]["passed"] >= d["counts"]["blended"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] > 0
