"""bench.py's reference arm runs without a GPU: one JSON line with the keys the driver reads."""
import json
import os
import re
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_json_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                          "--steps", "2", "--warmup", "1", "--ref-sample", "3000"],
                         capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert k in d, k
    assert d["impl"] == "reference" and d["metric"] == "protons_per_sec" and d["steps"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["config"]["workload"] == "config1_water64" and d["vs_baseline"] is None


def test_product_arm_refuses_to_run_without_a_gpu():
    """No CPU fallback: on a box without CUDA the product arm must fail loudly, not fall back to the oracle."""
    import torch
    if torch.cuda.is_available():
        return
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode != 0 and "no CPU fallback" in (out.stderr + out.stdout)


def test_static_ncu_counts_point_at_committed_captures():
    """roofline.traffic / roofline.ncu come from profiles/r03_counts.csv: one row per k_transport launch of one timed step of
    every config (1 / 1 / 1 / 3 / 6 launches), with the commit of the kernel; the README beside it names the ncu command."""
    sys.path.insert(0, ROOT)
    import bench
    assert bench.HEADLINE_CONFIG == 5
    for cfg, n in ((1, 1), (2, 1), (3, 1), (4, 3), (5, 6)):
        sc = bench._static_counts(cfg)
        assert sc is not None, cfg
        assert sc["n_launches"] == n and len(sc["per_launch_ms"]) == n
        assert sc["dram_bytes"] > 0 and sc["warp_instructions"] > 0 and sc["kernel_ms_under_ncu"] > 0
        assert 0 < sc["l2_tag_pct_time_weighted"] <= sc["l2_tag_pct_hottest_slice_time_weighted"] <= 100
        assert os.path.exists(os.path.join(ROOT, sc["source"]))
        assert re.fullmatch(r"[0-9a-f]{7,12}", sc["kernel_commit"])
    readme = open(os.path.join(ROOT, "profiles", "r03_README.md")).read()
    assert "r03_counts.csv" in readme and "ncu --clock-control none -k regex:k_transport" in readme and "bench.py --config" in readme
