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
    # the tensor kernel's captures are keyed by its precision mode as well: another product count is another kernel
    b, src = bench.ncu_traffic("c2", "tensor", "f32", 2)
    assert src is not None and os.path.exists(os.path.join(ROOT, src)) and b > 1e6
    for key in bench.NCU_SUMMARIES:
        got = bench.ncu_traffic(*key)
        assert got == (None, None) or os.path.exists(os.path.join(ROOT, got[1]))
    assert bench.ncu_traffic("c2", "tensor", "f32") == (None, None)       # no product count: no capture is claimed
    assert bench.ncu_traffic("c4", "tensor", "f32", 3) == (None, None)


def test_bench_line_names_the_arithmetic_and_the_real_instantiation():
    """The line's `dtype` is the arithmetic of the multiply-accumulates and roofline.kernel the instantiation the library
    launched, both derived from lsp_last_call_info (tensor_shape, tensor_products), never from argv."""
    sys.path.insert(0, ROOT)
    import bench
    assert bench.arithmetic_dtype("tensor", "f32", 3) == "f16x3-split/f32acc"
    assert bench.arithmetic_dtype("tensor", "f32", 2) == "f16x2-split/f32acc"
    assert bench.arithmetic_dtype("tensor", "f32", 1) == "f16/f32acc"
    assert bench.arithmetic_dtype("factored", "f32", 0) == "f32" and bench.arithmetic_dtype("factored", "f64", 0) == "f64"
    assert bench.tensor_instantiation(3, 3) == "lsp_tensor_kernel<float,0,4,4,0,true,112>"
    assert bench.tensor_instantiation(3, 2) == "lsp_tensor_kernel<float,2,4,4,0,true,112>"
    assert bench.tensor_instantiation(1, 3) == "lsp_tensor_kernel<float,0,8,3,0>"
    assert bench.tensor_instantiation(2, 1) == "lsp_tensor_kernel<float,1,4,4,0>"
    rf = bench.roofline("tensor", "f32", False, 1e10, 0.15, 0.0, "c2", products=3, shape=3)
    assert rf["kernel"] == "lsp_tensor_kernel<float,0,4,4,0,true,112>" and rf["executed_flop_per_pair"] == 24.0
    assert abs(rf["frac_executed"] - 3 * rf["frac"]) < 1e-12 and rf["bound"] == "tensor"
    src = open(os.path.join(ROOT, "bench.py")).read()
    for key in ('"fp32_fma_pipe"', '"fp32_tensor_2products"', '"fast_vs_accurate"', '"c5"', '"io_dtype"', '"clocks"', '"e2e"'):
        assert key in src, key
