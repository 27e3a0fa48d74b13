"""bench.py prints ONE JSON line with the keys the driver reads (task contract); run on the GPU box with `-m gpu`."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.gpu
def test_bench_line_has_the_contract_keys():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "2", "--warmup", "3", "--workload",
                          "c2_hbn_256", "--frames", "64", "--no-cpu-baseline"], capture_output=True, text=True, timeout=600,
                         cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert k in d, k
    assert d["n_gpus"] == 1 and d["steps"] == 2 and d["warmup"] >= 3 and d["value"] > 0
    assert d["config"]["workload"].startswith("c2_hbn_256") and d["gpu_launches"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0 and d["e2e"]["value"] > 0
    r = d["roofline"]
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert k in r, k
    assert r["bound"] == "hbm" and 0.0 < r["frac"] < 1.5


def test_default_workload_is_the_largest_single_gpu_configuration():
    """CPU: with no flags bench.py times config 3 (512^2, 80 slices, 10 240 atoms) on one 16-probe scan row x all 1024
    frames, and says so in config.workload."""
    sys.path.insert(0, ROOT)
    import argparse
    import bench
    args = argparse.Namespace(workload="c3_si_probe_512", frames=None, grid=None, probes_side=None, probe_chunk=16)
    src = open(os.path.join(ROOT, "bench.py")).read()
    assert 'ap.add_argument("--workload", default="c3_si_probe_512")' in src
    assert 'ap.add_argument("--probe-chunk", type=int, default=16' in src
    w = bench.build_workload(args)
    assert (w.nx, w.ny, w.n_slices, w.n_frames, w.n_probes, w.n_atoms) == (512, 512, 80, 1024, 16, 10240)
    assert "16-probe scan row x 1024 frames" in w.label
    cfg = bench.workload_config(w)
    assert cfg["workload"] == w.label and cfg["probes"] == 16 and cfg["frames"] == 1024


def test_oracle_arm_uses_all_cores_on_a_small_case():
    """CPU: `--impl reference` prints the contract line, with cores = os.cpu_count() worker processes."""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "c1_si_128",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    d = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert d["impl"] == "reference" and d["value"] > 0 and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] == min(os.cpu_count(), 64)
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"]
