"""bench.py's reference arm runs on the CPU (the oracle, as it stands): check the JSON-line contract without a GPU."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.timeout(300)
def test_reference_arm_prints_one_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0",
                          "--cpu-seconds", "1"], capture_output=True, text=True, timeout=280, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert key in d, key
    assert d["impl"] == "reference" and d["unit"] == "pairs/s" and d["value"] > 0 and d["data"] == "synthetic"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0 and "workload" in d["config"]


def test_nonzero_rank_of_reference_arm_exits_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                          "--warmup", "0"], capture_output=True, text=True, timeout=120, cwd=ROOT, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_pipe_peak_helper_builds_outside_the_library():
    """The pipe-peak microbenchmarks are a bench-only helper (bench_peak.cu -> libbench_peak.so), not part of liblsp_b200.so."""
    import ctypes
    sys.path.insert(0, ROOT)
    import bench
    lib = ctypes.CDLL(bench.build_peak_lib())
    assert hasattr(lib, "bench_pipe_peak")
    import paper_2105_04006_b200 as pkg
    assert not hasattr(pkg.load_library(), "lsp_pipe_peak") and not hasattr(pkg.load_library(), "bench_pipe_peak")


def test_roofline_traffic_is_read_from_a_committed_capture():
    sys.path.insert(0, ROOT)
    import bench
    b, src = bench.ncu_traffic("c2", "tensor", "f32")
    assert src is not None and os.path.exists(os.path.join(ROOT, src)) and b > 1e6
    assert bench.ncu_traffic("c4", "tensor", "f32") == (None, None)
