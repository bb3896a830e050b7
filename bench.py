#!/usr/bin/env python
"""bench.py -- (t,f) pair-evaluations/s of the batched Lomb-Scargle hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2|c3|c4|c5] [--dtype f32|f64] [--fast-math] [--variants]
    python bench.py --impl reference ...          # the CPU oracle, as it stands, on the box's host cores

A "step" is one pass of the whole hot path (SURVEY.md section 8(a) steps 1-6/6', and 7 for host output) over one
batch of seeded synthetic input.  Default workload: BASELINE.json configs[1] (single object, N_t = 10,000,
N_f = 1,000,000, full periodogram) in FP32 (the primary keys).  The same line then carries, as short objects,
  fp64           the same workload in FP64 (value, e2e, roofline)
  fp32_fma_pipe  the all-FP32 FFMA2 contraction on the FMA pipe (north_star's "FP32 issue-bound roofline": value, e2e, roofline, clocks)
  fp32_tensor_2products  the tensor path's two-product opt-in (faster, not safe on few-night cadences)
  c3, c4         BASELINE.json configs[2] (batch, fused best period) and configs[3] (4 GB of periodograms to pinned host
                 through the copy streams: T_compute, T_d2h, T_pipelined)
  fast_vs_accurate  MUFU (__sincosf-class) vs accurate sincos: the paper-shaped direct kernel and the tensor path
  c5             BASELINE.json configs[4], compact: pairs/s and roofline fraction of the 12 sweep points per dtype
`dtype` is the arithmetic of the multiply-accumulates ("f16x3-split/f32acc" for the default tensor path, "f32", "f64");
config.io_dtype is the element type of t, y and the powers.
and, with --variants, the comparison legs (fast_math, the paper-shaped direct kernels, the generalised mode).
  value       device-resident: inputs and output in HBM, CUDA events around each step on the launching stream
  e2e         the same pass through lsp_periodogram_batched_host: pinned HOST inputs, H2D + kernels + D2H inside
              the timed region
  roofline    the dominant kernel: tensor peak for the tcgen05 kernel, FMA / FP64 pipe peak for the FMA-pipe kernels
  cpu_baseline  the oracle timed on a bounded sample of the same workload (rank 0, N = 1 only)
Multi-GPU (torchrun, one rank per GPU): c2 -- every rank runs its own object of the same shape (seed + rank), "scaling":
"weak"; c3 -- ONE batch is cut by `sharding.partition_objects` (balanced by sum N_t), every rank runs the library on its
own CSR slice and the best periods are gathered, "scaling": "strong".  No data-path collective; device times, max over ranks.
"""
from __future__ import annotations

import argparse
import ctypes
import csv
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "lsp_pair_evals_per_s"
UNIT = "pairs/s"

# ALU roofline denominators: 148 SMs x lanes/clk/SM x 2 flop x clocks.max.sm (1965 MHz, B200_PROFILING.md)
N_SM = 148
SM_MAX_HZ = 1965e6
FP32_LANES = 128      # FP32 FMA lanes per SM per clock
FP64_LANES = 64       # FP64 FMA lanes per SM per clock
FLOP_PER_PAIR = 8.0   # factored formulation: 4 FMA per (t,f) pair ("4 FMA = 8 flop/pair")
# Tensor path: the same 4 MAC per pair as one FP16 GEMM; the accurate mode issues three products per MAC (a_hi b_hi + a_hi b_lo +
# a_lo b_hi, the library default) or two (a_hi (b_hi + b_lo); --tensor-products 2, an opt-in), fast_math one.
TENSOR_PRODUCTS = {False: 3, True: 1}
TENSOR_PEAK_FALLBACK = 1590.0     # TFLOP/s, B200_PROFILING.md fallback (bf16 burst; fp16 : bf16 nominal ratio is 1)


# roofline.traffic = dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, READ at run time from the
# committed `ncu --set full` summary of the same workload and kernel (profiles/*.csv; the commands are in the README beside
# them).  No capture for this (workload, kernel) -> null.  Newest round first.
NCU_SUMMARIES = {
    # tensor kernel: keyed by FP16 products per MAC as well (r02 captures: the two-product launches; r03: three products)
    ("c2", "tensor", "f32", 3): ("profiles/r03_ncu_full_tensor_f32_c2_3products.csv",),
    ("c3", "tensor", "f32", 3): ("profiles/r03_ncu_full_tensor_f32_c3_3products.csv",),
    ("c2", "tensor", "f32", 2): ("profiles/r02_ncu_full_tensor_f32_c2.csv",),
    ("c3", "tensor", "f32", 2): ("profiles/r02_ncu_full_tensor_f32_c3.csv",),
    ("c2", "factored", "f32"): ("profiles/r02_ncu_full_factored_ws_f32.csv",),
    ("c2", "factored", "f64"): ("profiles/r02_ncu_full_factored_ws_f64.csv",),
}


def ncu_traffic(workload: str, kernel: str, dtype: str, products: int = 0):
    """(bytes per launch, file) from the newest committed ncu summary of this workload / kernel (tensor kernel: of this
    product count; a capture of another precision mode is another kernel), or (None, None)."""
    key = (workload, kernel, dtype) if kernel != "tensor" else (workload, kernel, dtype, int(products))
    for rel in NCU_SUMMARIES.get(key, ()):
        path = os.path.join(ROOT, rel)
        if not os.path.exists(path):
            continue
        tot = {}
        with open(path, newline="") as fh:
            for row in csv.DictReader(fh):
                if row.get("metric") in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(row.get("unit", ""), None)
                    if scale is not None:
                        tot[row["metric"]] = float(row["value"]) * scale
        if len(tot) == 2:
            return sum(tot.values()), rel
    return None, None


_PEAK_LIB = None


def pipe_peak(which: int, device: int):
    """(ops_per_s, elapsed_ms) of the register-only pipe microbenchmark `which` (bench_peak.cu: 1 = FFMA2, 2 = DFMA, ...).
    A bench-only helper library built beside this file; it is not part of liblsp_b200.so."""
    global _PEAK_LIB
    if _PEAK_LIB is None:
        _PEAK_LIB = ctypes.CDLL(build_peak_lib())
        _PEAK_LIB.bench_pipe_peak.argtypes = [ctypes.c_int32, ctypes.c_int32, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
        _PEAK_LIB.bench_pipe_peak.restype = ctypes.c_int
    ops, ms = ctypes.c_double(), ctypes.c_double()
    rc = _PEAK_LIB.bench_pipe_peak(int(device), int(which), ctypes.byref(ops), ctypes.byref(ms))
    if rc != 0:
        raise RuntimeError(f"bench_pipe_peak failed with cudaError {rc}")
    return ops.value, ms.value


def build_peak_lib(force: bool = False) -> str:
    """nvcc -> libbench_peak.so beside bench.py (sm_100a; cross-compiles without a GPU)."""
    src, lib = os.path.join(ROOT, "bench_peak.cu"), os.path.join(ROOT, "libbench_peak.so")
    if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(src):
        nvcc = os.environ.get("NVCC") or "/usr/local/cuda/bin/nvcc"
        subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
                        "-shared", "-o", lib + ".tmp", src], check=True)
        os.replace(lib + ".tmp", lib)
    return lib


def measured_tensor_peak():
    """(TFLOP/s, provenance) -- the driver-written cuBLAS bf16 burst figure; FP16 runs at the same nominal rate."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["bf16_tflops"]), "of measured (MEASURED_PEAKS.json bf16_tflops, burst; fp16:bf16 = 1)"
    except Exception:
        return TENSOR_PEAK_FALLBACK, "of fallback (B200_PROFILING.md 1.59 PFLOP/s bf16 burst; fp16:bf16 = 1)"


def tensor_instantiation(shape: int, products: int) -> str:
    """The lsp_tensor_kernel instantiation launch_main picks (csrc/lsp_api.cu) for a standard call, from lsp_last_call_info:
    <T, PM (0 = three products, 2 = two, 1 = fast_math), epilogue warps, generator groups, GM = 0[, PAIR, max NL]>."""
    pm = {1: 1, 2: 2, 3: 0}.get(int(products), 0)
    if shape == 3:
        return "lsp_tensor_kernel<float,%d,4,4,0,true,112>" % pm
    return "lsp_tensor_kernel<float,%d,%s,0>" % (pm, "4,4" if shape == 2 else "8,3")


def arithmetic_dtype(kernel: str, dtype: str, products: int) -> str:
    """Machine-readable arithmetic of the contraction (the line's `dtype`): what the multiply-accumulates really are."""
    if kernel == "tensor":
        return {1: "f16/f32acc", 2: "f16x2-split/f32acc", 3: "f16x3-split/f32acc"}.get(int(products), "f16-split/f32acc")
    return dtype


def roofline(kernel: str, dtype: str, fast: bool, pairs: float, k_ms: float, pipe_ops: float, workload: str = "",
             products: int = 0, shape: int = 0):
    """Roofline object of the dominant kernel: achieved = algorithmic flop per launch
    (8 flop per (t,f) pair x pairs) / mean launch duration measured with CUDA events on the launching stream."""
    achieved = pairs * FLOP_PER_PAIR / (k_ms * 1e-3) / 1e12
    traffic, traffic_from = (None, None) if fast else ncu_traffic(workload, kernel, dtype, products)
    if kernel == "tensor":
        peak, prov = measured_tensor_peak()
        prod = products if products else TENSOR_PRODUCTS[bool(fast)]
        return {"bound": "tensor", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "traffic": traffic, "traffic_from": traffic_from,
                "kernel": tensor_instantiation(shape, prod), "flop_per_pair": FLOP_PER_PAIR,
                "peak_is": prov,
                "executed_flop_per_pair": FLOP_PER_PAIR * prod,
                "executed_tflops": achieved * prod, "frac_executed": achieved * prod / peak,
                "note": "FP16 split operands: %d tcgen05 products per algorithmic MAC" % prod}
    lanes = FP32_LANES if dtype == "f32" else FP64_LANES
    peak = N_SM * lanes * 2 * SM_MAX_HZ / 1e12
    if kernel != "factored":
        # Paper-shaped direct kernel (SURVEY.md 8(d) "Algorithmic work per pair"): FP32 fast = 2 MUFU per pair against the XU
        # pipe (16 lanes/clk/SM); FP32 accurate = ~17 FMA-pipe instructions per pair against 128 lanes/clk/SM; FP64 = ~24
        # FP64-pipe instructions per pair against 64 lanes/clk/SM.  Unit: 1e12 pipe operations per second.
        if dtype == "f32" and fast:
            ops, lanes_, what = 2.0, 16, "MUFU (XU pipe)"
        elif dtype == "f32":
            ops, lanes_, what = 17.0, 128, "FMA-pipe instructions"
        else:
            ops, lanes_, what = 24.0, 64, "FP64-pipe instructions"
        pk = N_SM * lanes_ * SM_MAX_HZ / 1e12
        ach = pairs * ops / (k_ms * 1e-3) / 1e12
        return {"bound": "alu", "achieved": ach, "peak": pk, "unit": "Top/s", "frac": ach / pk, "traffic": None,
                "kernel": "lsp_direct_kernel", "ops_per_pair": ops,
                "peak_is": "derived: 148 SMs x %d lanes/clk/SM x 1965 MHz, %s" % (lanes_, what)}
    return {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic,
            "traffic_from": traffic_from, "kernel": "lsp_factored_ws_kernel<%s>" % ("float" if dtype == "f32" else "double"),
            "flop_per_pair": FLOP_PER_PAIR,
            "peak_is": "derived: 148 SMs x %d %s FMA lanes/clk/SM x 2 flop x 1965 MHz (clocks.max.sm)" % (lanes, "FP32" if dtype == "f32" else "FP64"),
            "pipe_peak_measured": pipe_ops * 2 / 1e12, "frac_of_measured_pipe": achieved / (pipe_ops * 2 / 1e12)}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="c2", choices=["c2", "c3", "c4", "c5"])
    ap.add_argument("--dtype", default="f32", choices=["f32", "f64"], help="precision of the primary line")
    ap.add_argument("--fast-math", action="store_true", help="FP32: MUFU.SIN/COS instead of accurate sincospif")
    ap.add_argument("--kernel", default="auto", choices=["auto", "direct", "factored", "tensor"])
    ap.add_argument("--tensor-products", type=int, default=0, choices=[0, 2, 3],
                    help="tensor path, accurate mode: FP16 products per MAC (lsp_config.tensor_products; 0 = library default = 3)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-secondary", action="store_true", help="primary leg only (no fp64 / fp32_fma_pipe / c3 / c4 objects)")
    ap.add_argument("--variants", action="store_true", help="add the comparison legs: fast_math, direct kernels, generalised mode")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the cpu_baseline sample")
    return ap.parse_args()


def workload_for(name: str, dtype: str, rank: int, world: int = 1):
    """This rank's input.  c2 / c4 / c5: weak scaling, rank r draws its own object(s) from the same generator with sweep-point
    index r.  c3 with world > 1: ONE batch (the config's own seed), cut into contiguous object ranges balanced by sum N_t
    (sharding.partition_objects); rank r gets its CSR slice -- strong scaling, no data-path collective."""
    from workloads import make_config, Workload
    from workloads.configs import config_seed  # noqa: F401  (seed recipe: DESIGN.md "Input recipe")
    cfg = {"c2": 2, "c3": 3, "c4": 4, "c5": 5}[name]
    if name == "c3" and world > 1:
        from paper_2105_04006_b200 import sharding
        w = make_config(cfg, dtype=dtype)
        o0, o1 = sharding.partition_objects(w.offsets, world)[rank]
        off, t, y = sharding.slice_csr(w.offsets, w.t, w.y, o0, o1)
        return Workload(w.name, off.copy(), t, y, w.f_min, w.f_max, w.n_freq, dtype,
                        meta={"shard": [int(o0), int(o1)], "n_obj_total": int(w.n_obj), "n_obs_total": int(w.n_obs)})
    return make_config(cfg, dtype=dtype, point=rank)


# ---- clocks --------------------------------------------------------------------------------------------------------
class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""
    BAD = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "hw_power_brake": 0x80}
    NOTE = {"sw_power_cap": 0x4}

    def __init__(self, index: int, period_s: float = 0.002):
        self.samples, self.reasons = [], set()
        self.period, self.stop_flag, self.thread, self.ok = period_s, threading.Event(), None, False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = index
            if vis:
                try:
                    phys = int(vis.split(",")[index])
                except ValueError:
                    phys = index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception as exc:  # no NVML: clocks are reported as unavailable, never invented
            self.err = repr(exc)

    def _run(self):
        nv = self.nv
        while not self.stop_flag.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in {**self.BAD, **self.NOTE}.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def __enter__(self):
        if self.ok:
            self.thread = threading.Thread(target=self._run, daemon=True)
            self.thread.start()
        return self

    def __exit__(self, *exc):
        if self.thread:
            self.stop_flag.set()
            self.thread.join()

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml_unavailable"]}
        s = sorted(self.samples)
        return {"sm_mhz": float(s[len(s) // 2]), "sm_max_mhz": float(self.max_mhz), "reasons": sorted(self.reasons),
                "samples": len(s)}


# ---- the CPU oracle leg (cpu_baseline and --impl reference) ---------------------------------------------------
def oracle_sample_runner(w, seconds_per_step: float):
    """Returns (run, pairs_per_step, cores, description): `run()` evaluates the oracle, as it stands, on a bounded
    sample of workload `w`: whole objects for batches, a strided subset of the grid for a single object."""
    import numpy as np
    import oracle
    oracle.build()
    probe_k = np.linspace(0, w.n_freq - 1, 512).astype(np.int64)
    one = w.take_objects([0]) if w.n_obj > 1 else w
    t0 = time.perf_counter()
    _, cores = oracle.periodogram(one.offsets, one.t, one.y, w.f_min, w.f_max, w.n_freq, k_list=probe_k, return_threads=True)
    dt = max(time.perf_counter() - t0, 1e-4)
    rate = one.n_obs * probe_k.size / dt                 # pairs/s seen by the probe
    pairs_target = rate * seconds_per_step
    if w.n_obj == 1:
        n_k = int(min(w.n_freq, max(cores * 8, pairs_target / max(1, w.n_obs))))
        ks = np.unique(np.linspace(0, w.n_freq - 1, n_k).astype(np.int64))
        sub, desc = w, f"{ks.size} of {w.n_freq} grid frequencies (strided) x all {w.n_obs} observations"
    else:
        ks = np.unique(np.linspace(0, w.n_freq - 1, min(w.n_freq, 2000)).astype(np.int64))
        mean_nt = w.n_obs / w.n_obj
        n_o = int(min(w.n_obj, max(2 * cores, pairs_target / (mean_nt * ks.size))))
        sub = w.take_objects(np.arange(n_o))
        desc = f"first {n_o} of {w.n_obj} objects x {ks.size} of {w.n_freq} grid frequencies (strided)"

    def run():
        return oracle.periodogram(sub.offsets, sub.t, sub.y, w.f_min, w.f_max, w.n_freq, k_list=ks)

    run.sub, run.ks = sub, ks
    return run, int(sub.n_obs) * int(ks.size), int(cores), desc


def cpu_baseline(w, seconds: float, gpu_power=None):
    """The oracle timed on the host cores on a bounded sample of the workload.  `gpu_power(sub)`, if given, returns the CUDA
    path's full periodogram of the sample's objects (library defaults, as timed): the sample then doubles as a parity spot
    check of the timed configuration, max |dP| / max P over the sample (tolerances: BASELINE.json, 1e-3 FP32 / 1e-9 FP64)."""
    run, pairs, cores, desc = oracle_sample_runner(w, seconds)
    t0 = time.perf_counter()
    p_ref = run()
    dt = time.perf_counter() - t0
    out = {"value": pairs / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc, "seconds": round(dt, 3)}
    if gpu_power is not None:
        import numpy as np
        p_gpu = gpu_power(run.sub)[:, run.ks].astype(np.float64)
        err = float(np.max(np.max(np.abs(p_gpu - p_ref), axis=1) / np.max(p_ref, axis=1)))
        out["parity_sample"] = {"max_err_over_max_p": err, "tolerance": 1e-3 if w.dtype == "f32" else 1e-9,
                                "note": "CUDA path (library defaults, as timed) vs the oracle on the sampled grid points; "
                                        "max P is the sample's"}
    return out


def run_reference(args, rank: int, world: int):
    if rank != 0:
        return
    w = workload_for(args.workload, args.dtype, 0)
    n_steps = args.steps + args.warmup
    per_step = max(0.05, min(3.0, 90.0 / max(1, n_steps)))
    run, pairs, cores, desc = oracle_sample_runner(w, per_step)
    for _ in range(args.warmup):
        run()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        run()
    dt = time.perf_counter() - t0
    value = pairs * args.steps / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": describe_workload(args.workload, w), "sample_per_step": desc},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def describe_workload(name: str, w) -> str:
    if name == "c2":
        return (f"BASELINE.json configs[1]: single object, N_t={w.n_obs}, N_f={w.n_freq}, f in [{w.f_min},{w.f_max}) c/d, "
                f"full periodogram")
    if name == "c3":
        n_obj, n_obs = w.meta.get("n_obj_total", w.n_obj), w.meta.get("n_obs_total", w.n_obs)
        return (f"BASELINE.json configs[2]: {n_obj} objects, N_t in [50,500] (sum {n_obs}), N_f={w.n_freq}, "
                f"best period only")
    return (f"BASELINE.json configs[3]: {w.n_obj} objects (sum N_t {w.n_obs}), N_f={w.n_freq}, full periodogram to "
            f"pinned host over copy streams")


# ---- the B200 leg -----------------------------------------------------------------------------------------------
class Leg:
    """One precision of one workload on this rank's GPU: device-resident steps and end-to-end (host buffer) steps."""

    def __init__(self, pkg, torch, w, name: str, dtype: str, fast_math: bool, kernel: str, device: int, tensor_products: int = 0):
        self.torch, self.w, self.name, self.dtype = torch, w, name, dtype
        self.tdt = torch.float32 if dtype == "f32" else torch.float64
        self.plan = pkg.Plan(w.f_min, w.f_max, w.n_freq, dtype, fast_math=fast_math and dtype == "f32", kernel=kernel,
                             device=device, tensor_products=tensor_products)
        self.plan.set_timing(False)            # the timed steps run as a user's would: no events inside the library
        self.h_off = torch.from_numpy(w.offsets)
        self.h_t = torch.from_numpy(w.t).pin_memory()
        self.h_y = torch.from_numpy(w.y).pin_memory()
        dev = torch.device("cuda", device)
        self.d_off, self.d_t, self.d_y = self.h_off.to(dev), self.h_t.to(dev), self.h_y.to(dev)
        self.best_only = name == "c3"
        self.host_mode = name == "c4"          # the workload itself ends on the host
        n = w.n_obj
        self.d_best = (torch.empty(n, dtype=self.tdt, device=dev), torch.empty(n, dtype=self.tdt, device=dev),
                       torch.empty(n, dtype=torch.int64, device=dev))
        self.h_best = (torch.empty(n, dtype=self.tdt).pin_memory(), torch.empty(n, dtype=self.tdt).pin_memory(),
                       torch.empty(n, dtype=torch.int64).pin_memory())
        self.d_out = self.h_out = None
        if not self.best_only:
            if self.host_mode:
                self.h_out = torch.empty((n, w.n_freq), dtype=self.tdt).pin_memory()
            else:
                self.d_out = torch.empty((n, w.n_freq), dtype=self.tdt, device=dev)
                self.h_out = torch.empty((n, w.n_freq), dtype=self.tdt).pin_memory()
        self.launches = 0

    def step_device(self):
        """Inputs resident in HBM.  c2: full periodogram to HBM; c3: fused best period; c4: periodograms to pinned host."""
        if self.best_only:
            self.plan.best_period(self.d_off, self.d_t, self.d_y, out=self.d_best, h_offsets=self.h_off)
        elif self.host_mode:
            self.plan.periodogram_batched(self.d_off, self.d_t, self.d_y, host_out=self.h_out, h_offsets=self.h_off)
        else:
            self.plan.periodogram_batched(self.d_off, self.d_t, self.d_y, out=self.d_out, h_offsets=self.h_off)

    def step_e2e(self):
        if self.best_only:
            self.plan.periodogram_batched_host(self.h_off, self.h_t, self.h_y, best_out=self.h_best)
        else:
            self.plan.periodogram_batched_host(self.h_off, self.h_t, self.h_y, host_out=self.h_out)

    def e2e_bytes(self):
        h2d = self.h_off.numel() * 8 + self.h_t.numel() * self.h_t.element_size() * 2
        if self.best_only:
            d2h = sum(x.numel() * x.element_size() for x in self.h_best)
        else:
            d2h = self.h_out.numel() * self.h_out.element_size()
        return int(h2d), int(d2h)

    def note_call(self, timed: bool):
        info = self.plan.last_call_info()
        if timed:
            self.launches += info["launches"]
        return info

    def measure_kernel_ms(self, flush, steps: int):
        """Mean duration of the dominant kernel: a separate short loop with the library's own CUDA events recorded around
        that kernel on the launching stream (lsp_set_timing).  Kept out of the step timing: an event between two launches
        would also undo the programmatic overlap of the tensor path's launches."""
        self.plan.set_timing(True)
        ms = []
        for i in range(steps + 2):
            flush()
            self.step_device()
            self.torch.cuda.synchronize()
            if i >= 2:
                ms.append(self.plan.last_kernel_ms())
        self.plan.set_timing(False)
        return sum(ms) / len(ms)


def timed_loop(torch, dist, world, leg, step, steps: int, warmup: int, flush):
    """W warm-up steps, then K steps, each bracketed by CUDA events on the launching (current) stream; the L2 flush runs
    between steps, outside the event pairs.  Returns (total_ms over K steps: max over ranks, info of the last call)."""
    for _ in range(warmup):
        flush()
        step()
        leg.note_call(False)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
        torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    info = None
    for a, b in ev:
        flush()
        a.record()
        step()
        b.record()
        info = leg.note_call(True)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
        torch.cuda.synchronize()
    total_ms = sum(a.elapsed_time(b) for a, b in ev)
    if world > 1:
        tt = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        total_ms = float(tt.item())
    return total_ms, info


ARITHMETIC_3 = "fp16 hi+lo split of both operands (22-bit), 3 tcgen05 products per MAC, fp32 accumulate in TMEM; phases two-float fp32"
ARITHMETIC = {
    ("tensor", False): "fp16 generated operand (11-bit) x fp16 hi+lo tabulated operand (22-bit), 2 tcgen05 products per MAC, fp32 accumulate in TMEM; phases two-float fp32",
    ("tensor", True): "fp16 operands, 1 tcgen05 product per MAC, fp32 accumulate; MUFU sincos (fast_math)",
    ("factored", False): "all-fp32 FFMA2 contraction (fp64: DFMA)", ("factored", True): "all-fp32 FFMA2 contraction, MUFU sincos",
    ("direct", False): "one accurate sincos per pair", ("direct", True): "one MUFU sincos per pair",
}


def run_leg(args, pkg, torch, dist, rank, world, device, dtype, flush, with_clocks: bool, kernel=None, fast=None,
            with_e2e: bool = True, workload=None, steps=None, tensor_products=None):
    name = args.workload if workload is None else workload
    steps = args.steps if steps is None else steps
    w = workload_for(name, dtype, rank, world)
    kernel = args.kernel if kernel is None else kernel
    fast = bool(args.fast_math if fast is None else fast) and dtype == "f32"
    leg = Leg(pkg, torch, w, name, dtype, fast, kernel, device, args.tensor_products if tensor_products is None else tensor_products)
    pairs_step = w.pairs
    pairs_all = pairs_step
    if world > 1:
        tt = torch.tensor([float(pairs_step)], dtype=torch.float64, device="cuda")
        dist.all_reduce(tt, op=dist.ReduceOp.SUM)
        pairs_all = float(tt.item())
    sampler = ClockSampler(device) if with_clocks else None
    if sampler:
        sampler.__enter__()
    total_ms, info = timed_loop(torch, dist, world, leg, leg.step_device, steps, args.warmup, flush)
    dev_launches = leg.launches
    leg.launches = 0
    ms_step = total_ms / steps
    k_ms = leg.measure_kernel_ms(flush, max(3, min(steps, 10)))
    # measured pipe peak with the same clocks the kernels see (register-only FFMA2 / DFMA loops, bench_peak.cu)
    pipe_ops = 0.0
    if info["kernel"] == "factored":
        pipe_ops, _ = pipe_peak(1 if dtype == "f32" else 2, device)
    products = int(info.get("tensor_products", 0))     # what the library launched (0 = not the tensor kernel), never argv
    rf = roofline(info["kernel"], dtype, fast, pairs_step, k_ms, pipe_ops, name, products, int(info.get("tensor_shape", 0)))
    es = 4 if dtype == "f32" else 8
    in_bytes = w.n_obs * 2 * es + (w.n_obj + 1) * 8
    out_bytes = w.n_obj * (2 * es + 8) if leg.best_only else w.n_obj * w.n_freq * es
    rf["algorithmic_bytes"] = int(in_bytes + out_bytes)
    if not leg.best_only and not leg.host_mode:
        # achieved HBM write rate of the full-periodogram stores (north_star): N_o x N_f powers per launch of the
        # kernel that writes them
        rf["hbm_write_gbs"] = out_bytes / (k_ms * 1e-3) / 1e9
    out = {
        "dtype": dtype,
        "arithmetic_dtype": arithmetic_dtype(info["kernel"], dtype, products), "tensor_products": products,
        "value": pairs_all * steps / (total_ms * 1e-3),
        "ms_per_step": ms_step,
        "kernel": info["kernel"], "n_split": info["n_split"], "fast_math": fast, "tensor_shape": info.get("tensor_shape", 0),
        "kernel_ms_per_step": k_ms,
        "gpu_launches": dev_launches,
        "roofline": rf,
        "arithmetic": ARITHMETIC_3 if (info["kernel"] == "tensor" and products == 3) else ARITHMETIC.get((info["kernel"], fast), ""),
        "io_dtype": dtype,
    }
    if world > 1 and name == "c3":
        obs = [torch.zeros(1, dtype=torch.int64, device="cuda") for _ in range(world)]
        dist.all_gather(obs, torch.tensor([int(w.n_obs)], dtype=torch.int64, device="cuda"))
        out["rank_sum_nt"] = [int(x.item()) for x in obs]
        # the best periods of the whole batch, gathered on every rank (outside the timed region: 24 bytes per object)
        from paper_2105_04006_b200 import sharding
        counts = [b - a for a, b in sharding.partition_objects(
            __import__("workloads").make_config(3, dtype=dtype).offsets, world)]
        allb = sharding.gather_objects(leg.d_best, counts)
        out["gathered_best_periods"] = int(allb[0].numel())
    if with_e2e:
        e2e_ms, _ = timed_loop(torch, dist, world, leg, leg.step_e2e, steps, args.warmup, flush)
        h2d, d2h = leg.e2e_bytes()
        out["e2e"] = {"value": pairs_all * steps / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                      "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms / steps}
    if sampler:
        sampler.__exit__()
    if sampler:
        out["clocks"] = sampler.summary()
    leg.plan.destroy()
    return out, w


def c4_overlap(args, pkg, torch, device, flush, with_pageable: bool = True):
    """SURVEY.md 8(d) "C4 overlap": T_c = compute only (periodograms to a device buffer), T_d = D2H only of the resident
    N_o x N_f buffer with the library's chunking (chunk_bytes pieces round-robin over n_copy_streams streams into the
    pinned destination), T = the pipelined call.  hidden = (T_c + T_d - T) / min(T_c, T_d); "fully overlapped" means
    T <= 1.05 max(T_c, T_d) + one chunk's latency."""
    w = workload_for("c4", "f32", 0)
    dev = torch.device("cuda", device)
    n_streams, chunk_bytes = 3, 64 << 20
    plan = pkg.Plan(w.f_min, w.f_max, w.n_freq, "f32", kernel=args.kernel, device=device, n_copy_streams=n_streams,
                    chunk_bytes=chunk_bytes)
    h_off = torch.from_numpy(w.offsets)
    d_off, d_t, d_y = h_off.to(dev), torch.from_numpy(w.t).to(dev), torch.from_numpy(w.y).to(dev)
    d_out = torch.empty((w.n_obj, w.n_freq), dtype=torch.float32, device=dev)
    h_out = torch.empty((w.n_obj, w.n_freq), dtype=torch.float32).pin_memory()
    row = w.n_freq * 4
    objs_per_chunk = max(1, chunk_bytes // row)
    streams = [torch.cuda.Stream(device=dev) for _ in range(n_streams)]

    def t_compute():
        plan.periodogram_batched(d_off, d_t, d_y, out=d_out, h_offsets=h_off)

    def t_copy():
        cur = torch.cuda.current_stream()
        for i, o0 in enumerate(range(0, w.n_obj, objs_per_chunk)):
            st = streams[i % n_streams]
            st.wait_stream(cur)
            with torch.cuda.stream(st):
                h_out[o0:o0 + objs_per_chunk].copy_(d_out[o0:o0 + objs_per_chunk], non_blocking=True)
        for st in streams:
            cur.wait_stream(st)

    def t_pipe():
        plan.periodogram_batched(d_off, d_t, d_y, host_out=h_out, h_offsets=h_off)

    def timeit(fn, reps=3):
        for _ in range(2):
            fn()
        torch.cuda.synchronize()
        best = 1e30
        for _ in range(reps):
            flush()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn()
            b.record()
            torch.cuda.synchronize()
            best = min(best, a.elapsed_time(b))
        return best

    tc, td, tp = timeit(t_compute), timeit(t_copy), timeit(t_pipe)
    plan.destroy()
    # pageable destination (Fig. 8): pinned staging ring + host-side copies on the copy
    # streams' callback threads, against plain cudaMemcpyAsync into the pageable buffer
    h_page = None
    if with_pageable:
        h_page = torch.empty((w.n_obj, w.n_freq), dtype=torch.float32)
        h_page.fill_(0.0)                              # touch the pages once, outside the timed region
    pageable = {}
    for mode in (("staged", "plain") if with_pageable else ()):
        pl = pkg.Plan(w.f_min, w.f_max, w.n_freq, "f32", kernel=args.kernel, device=device, n_copy_streams=n_streams,
                      chunk_bytes=chunk_bytes, pageable_staged=(mode == "staged"))
        pageable[mode] = timeit(lambda: pl.periodogram_batched(d_off, d_t, d_y, host_out=h_page, h_offsets=h_off), reps=2)
        pl.destroy()
    gb = w.n_obj * row / 1e9
    out = {"T_compute_ms": tc, "T_d2h_ms": td, "T_pipelined_ms": tp, "d2h_GBps": gb / (td * 1e-3),
           "hidden_fraction": (tc + td - tp) / min(tc, td), "T_over_max": tp / max(tc, td),
           "fully_overlapped": bool(tp <= 1.05 * max(tc, td) + td / max(1, -(-w.n_obj // objs_per_chunk))),
           "value": w.pairs / (tp * 1e-3), "chunk_bytes": chunk_bytes, "n_copy_streams": n_streams, "bytes": w.n_obj * row}
    if with_pageable:
        out["T_pageable_staged_ms"], out["T_pageable_plain_ms"] = pageable["staged"], pageable["plain"]
    return out


def run_c5(args, pkg, torch, device, flush):
    """BASELINE.json configs[4]: single object, N_t x N_f sweep in FP32 and FP64; pairs/s and roofline fraction per
    point (device-resident, full periodogram; kernel time from CUDA events on the launching stream)."""
    from workloads import make_config, C5_NT, C5_NF
    dev = torch.device("cuda", device)
    rows = []
    for dtype in ("f32", "f64"):
        pipe_ops, _ = pipe_peak(1 if dtype == "f32" else 2, device)
        tdt = torch.float32 if dtype == "f32" else torch.float64
        for i, nt in enumerate(C5_NT):
            for j, nf in enumerate(C5_NF):
                w = make_config(5, dtype=dtype, n_t=nt, n_freq=nf, point=i * len(C5_NF) + j)
                plan = pkg.Plan(w.f_min, w.f_max, w.n_freq, dtype, kernel=args.kernel, fast_math=args.fast_math and dtype == "f32",
                                device=device, tensor_products=args.tensor_products)
                h_off = torch.from_numpy(w.offsets)
                d_off, d_t, d_y = h_off.to(dev), torch.from_numpy(w.t).to(dev), torch.from_numpy(w.y).to(dev)
                d_out = torch.empty((1, nf), dtype=tdt, device=dev)
                steps = max(3, min(args.steps, int(2e12 / w.pairs) + 3))
                for _ in range(max(3, args.warmup)):
                    plan.periodogram_batched(d_off, d_t, d_y, out=d_out, h_offsets=h_off)
                torch.cuda.synchronize()
                tot, kms = 0.0, 0.0
                for _ in range(steps):
                    flush()
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record()
                    plan.periodogram_batched(d_off, d_t, d_y, out=d_out, h_offsets=h_off)
                    b.record()
                    torch.cuda.synchronize()
                    tot += a.elapsed_time(b)
                plan.set_timing(True)                      # the dominant kernel alone: a separate loop (see Leg.measure_kernel_ms)
                for _ in range(3):
                    flush()
                    plan.periodogram_batched(d_off, d_t, d_y, out=d_out, h_offsets=h_off)
                    torch.cuda.synchronize()
                    kms += plan.last_kernel_ms() * steps / 3.0
                info = plan.last_call_info()
                rf = roofline(info["kernel"], dtype, args.fast_math and dtype == "f32", w.pairs, kms / steps, pipe_ops,
                              products=int(info.get("tensor_products", 0)), shape=int(info.get("tensor_shape", 0)))
                rows.append({"dtype": dtype, "n_t": nt, "n_freq": nf, "pairs": w.pairs, "kernel": info["kernel"],
                             "n_split": info["n_split"], "ms_per_step": tot / steps, "kernel_ms": kms / steps,
                             "pairs_per_s": w.pairs * steps / (tot * 1e-3), "bound": rf["bound"], "roofline_frac": rf["frac"],
                             "frac_executed": rf.get("frac_executed")})
                plan.destroy()
    # FP64 / FP32 time ratio per point (the paper's Table 4 analogue)
    f32 = {(r["n_t"], r["n_freq"]): r["ms_per_step"] for r in rows if r["dtype"] == "f32"}
    for r in rows:
        if r["dtype"] == "f64":
            r["time_vs_f32"] = r["ms_per_step"] / f32[(r["n_t"], r["n_freq"])]
    return rows


def run_generalized(args, pkg, torch, device, flush, dtype: str):
    """The generalised mode (floating mean + errors) on the same workload, device-resident: pairs/s counts
    N_t x N_f once (the paper's convention: it quotes the generalised periodogram as 2.06-2.14x the standard one's time)."""
    import numpy as np
    w = workload_for(args.workload, dtype, 0)
    dev = torch.device("cuda", device)
    rng = np.random.Generator(np.random.PCG64(977))
    sigma = (0.2 * rng.uniform(0.5, 2.0, w.n_obs)).astype(w.t.dtype)
    plan = pkg.Plan(w.f_min, w.f_max, w.n_freq, dtype, device=device)
    h_off = torch.from_numpy(w.offsets)
    d_off, d_t, d_y, d_s = h_off.to(dev), torch.from_numpy(w.t).to(dev), torch.from_numpy(w.y).to(dev), torch.from_numpy(sigma).to(dev)
    best_only = args.workload == "c3"
    out = None if best_only else torch.empty((w.n_obj, w.n_freq), dtype=d_t.dtype, device=dev)
    steps = max(3, min(args.steps, 10))

    def step():
        plan.periodogram_generalized(d_off, d_t, d_y, d_s, out=out, best=best_only, want_power=not best_only, h_offsets=h_off)

    for _ in range(3):
        step()
    torch.cuda.synchronize()
    tot = 0.0
    for _ in range(steps):
        flush()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        step()
        b.record()
        torch.cuda.synchronize()
        tot += a.elapsed_time(b)
    info = plan.last_call_info()
    plan.destroy()
    return {"dtype": dtype, "value": w.pairs * steps / (tot * 1e-3), "unit": UNIT, "ms_per_step": tot / steps, "steps": steps,
            "kernel": info["kernel"], "gpu_launches": info["launches"] * steps}


def run_b200(args, rank: int, world: int, local_rank: int):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device visible; the library has no CPU fallback (use --impl reference for the oracle)")
    import paper_2105_04006_b200 as pkg
    pkg.load_library()
    dist = None
    torch.cuda.set_device(local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2

    def flush():
        flush_buf.fill_(1)

    if args.workload == "c5":
        if rank == 0:
            rows = run_c5(args, pkg, torch, local_rank, flush)
            f32 = [r for r in rows if r["dtype"] == "f32"]
            tot_pairs = sum(r["pairs"] for r in f32)
            tot_ms = sum(r["ms_per_step"] for r in f32)
            print(json.dumps({"metric": METRIC, "value": tot_pairs / (tot_ms * 1e-3), "unit": UNIT, "n_gpus": 1,
                              "steps": args.steps, "warmup": args.warmup, "ms_per_step": tot_ms, "higher_is_better": True,
                              "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                              "config": {"workload": "BASELINE.json configs[4]: single-object sweep N_t x N_f, FP32 and FP64, "
                                                     "full periodogram; value = FP32 pairs of the 12 points / their summed time",
                                         "l2": "flushed between steps"},
                              "sweep": rows}), flush=True)
        return
    primary, w = run_leg(args, pkg, torch, dist, rank, world, local_rank, args.dtype, flush, True)
    solo = rank == 0 and world == 1
    secondary = not args.no_secondary and args.workload == "c2" and args.kernel == "auto" and not args.fast_math
    other = fma = two = c3 = c4 = fva = c5 = None
    variants = {}
    if secondary:
        other_dtype = "f64" if args.dtype == "f32" else "f32"
        other, _ = run_leg(args, pkg, torch, dist, rank, world, local_rank, other_dtype, flush, False)
        # the all-FP32 FFMA2 contraction on the FMA pipe: north_star's "FP32 issue-bound roofline" is answered by this kernel
        fma, _ = run_leg(args, pkg, torch, dist, rank, world, local_rank, "f32", flush, True, kernel="factored", fast=False,
                         with_e2e=True)
        # the two-product opt-in of the tensor path (lsp_config.tensor_products = 2): faster on long objects, not safe on
        # few-night cadences -- a labelled leg, never the headline
        if args.tensor_products != 2:
            two, _ = run_leg(args, pkg, torch, dist, rank, world, local_rank, "f32", flush, False, kernel="auto", fast=False,
                             with_e2e=False, tensor_products=2)
        if solo:
            # BASELINE.json configs[2] and configs[3], short: the driver's record then carries them too
            c3, _ = run_leg(args, pkg, torch, dist, rank, world, local_rank, "f32", flush, False, workload="c3",
                            steps=max(3, min(args.steps, 10)))
            c4 = c4_overlap(args, pkg, torch, local_rank, flush, with_pageable=False)
            # north_star: "fast-math __sincosf is compared against accurate sincos" (Table 6): the paper-shaped
            # direct kernel with MUFU sincos vs sincospif, and the tensor path's fast_math mode vs its default
            few = max(3, min(args.steps, 5))
            legs = {}
            for key, kern, fast_ in (("direct_sincosf", "direct", True), ("direct_accurate", "direct", False),
                                     ("tensor_fast_math", "auto", True)):
                legs[key], _ = run_leg(args, pkg, torch, dist, rank, world, local_rank, "f32", flush, False, kernel=kern,
                                       fast=fast_, with_e2e=False, steps=few)
            fva = {"unit": UNIT, "workload": "c2", "dtype": "f32", "cite": "PAPER.md:L423-433, Table 6 L451-459"}
            for key, v in legs.items():
                fva[key] = {"value": v["value"], "kernel_ms": v["kernel_ms_per_step"], "frac": v["roofline"]["frac"],
                            "bound": v["roofline"]["bound"], "gpu_launches": v["gpu_launches"]}
            fva["tensor_default"] = {"value": primary["value"], "kernel_ms": primary["kernel_ms_per_step"]}
            fva["direct_speedup_fast_over_accurate"] = legs["direct_sincosf"]["value"] / legs["direct_accurate"]["value"]
            fva["tensor_speedup_fast_over_default"] = legs["tensor_fast_math"]["value"] / primary["value"]
            # BASELINE.json configs[4], compact: per dtype the 12 (N_t x N_f) points' pairs/s and roofline fraction, row-major
            from workloads import C5_NT, C5_NF
            rows = run_c5(args, pkg, torch, local_rank, flush)
            c5 = {"n_t": list(C5_NT), "n_freq": list(C5_NF), "order": "n_t-major", "unit": UNIT}
            for dt in ("f32", "f64"):
                rr = [r for r in rows if r["dtype"] == dt]
                c5[dt] = {"pairs_per_s": [float("%.4g" % r["pairs_per_s"]) for r in rr],
                          "frac": [float("%.3g" % r["roofline_frac"]) for r in rr],
                          "bound": sorted({r["bound"] for r in rr}), "kernel": sorted({r["kernel"] for r in rr})}
    if args.variants and args.workload == "c2":
        # fast_math tensor mode and the paper-shaped kernel (thread = frequency, one sincos per pair): __sincosf-class vs
        # accurate sincos, the comparison north_star asks for
        variants["fp32_fast_math"], _ = run_leg(args, pkg, torch, dist, rank, world, local_rank, "f32", flush, False,
                                                kernel="auto", fast=True, with_e2e=False)
        few = max(3, min(args.steps, 5))
        for key, dt, fast in (("direct_fp32_sincosf", "f32", True), ("direct_fp32_accurate", "f32", False), ("direct_fp64", "f64", False)):
            variants[key], _ = run_leg(args, pkg, torch, dist, rank, world, local_rank, dt, flush, False, kernel="direct",
                                       fast=fast, with_e2e=False, steps=few)
    gls = None
    if args.variants and args.workload in ("c2", "c3") and solo:
        gls = {}
        for dt in (("f32", "f64") if args.workload == "c2" else ("f32",)):
            g = run_generalized(args, pkg, torch, local_rank, flush, dt)
            std_ms = primary["ms_per_step"] if dt == primary["dtype"] else (other["ms_per_step"] if other else None)
            g["time_vs_standard_same_dtype"] = (g["ms_per_step"] / std_ms) if std_ms else None
            gls[dt] = g
    overlap = None
    if args.workload == "c4" and solo:
        overlap = c4_overlap(args, pkg, torch, local_rank, flush)
    cpu = None
    if solo and not args.no_cpu_baseline:
        def gpu_power(sub):
            with pkg.Plan(sub.f_min, sub.f_max, sub.n_freq, args.dtype, kernel=args.kernel, fast_math=args.fast_math and args.dtype == "f32",
                          device=local_rank, tensor_products=args.tensor_products) as plan:
                dev = torch.device("cuda", local_rank)
                h_off = torch.from_numpy(sub.offsets)
                P, _ = plan.periodogram_batched(h_off.to(dev), torch.from_numpy(sub.t).to(dev), torch.from_numpy(sub.y).to(dev),
                                                h_offsets=h_off)
                torch.cuda.synchronize()
                return P.cpu().numpy()
        cpu = cpu_baseline(w, args.cpu_seconds, gpu_power if args.workload in ("c2", "c3") else None)
    if rank == 0:
        sharded = world > 1 and args.workload == "c3"
        rf_keys = ("bound", "achieved", "peak", "unit", "frac", "traffic", "traffic_from", "algorithmic_bytes", "hbm_write_gbs",
                   "kernel", "peak_is", "executed_flop_per_pair", "frac_executed", "frac_of_measured_pipe")

        def short_rf(rf):
            return {k: rf[k] for k in rf_keys if k in rf}

        def short_leg(v, with_e2e=True):
            o = {"value": v["value"], "dtype": v["arithmetic_dtype"], "ms_per_step": v["ms_per_step"],
                 "kernel_ms_per_step": v["kernel_ms_per_step"], "kernel": v["kernel"], "gpu_launches": v["gpu_launches"],
                 "roofline": short_rf(v["roofline"])}
            if with_e2e and "e2e" in v:
                o["e2e"] = v["e2e"]
            if "clocks" in v:
                o["clocks"] = v["clocks"]
            return o

        # the contract's keys first, so that a cut tail cannot lose them
        line = {
            "metric": METRIC, "value": primary["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": primary["ms_per_step"], "higher_is_better": True,
            "scaling": "strong" if sharded else "weak",
            # dtype = the arithmetic of the multiply-accumulates (an FP16-split tcgen05 contraction is not "f32"); io_dtype = t, y, P
            "vs_baseline": None, "dtype": primary["arithmetic_dtype"], "data": "synthetic",
            "config": {"workload": describe_workload(args.workload, w), "kernel": primary["kernel"],
                       "io_dtype": primary["io_dtype"], "tensor_products": primary["tensor_products"],
                       "arithmetic": primary["arithmetic"],
                       "fast_math": bool(args.fast_math and args.dtype == "f32"), "n_split": primary["n_split"],
                       "tensor_shape": primary["tensor_shape"],
                       "l2": "flushed between steps (256 MiB fill, outside the event pairs)",
                       "parallelism": (f"one batch sharded by object over {world} ranks (balanced by sum N_t), no collective"
                                       if sharded else f"replicas x{world} (one object set per rank, no collective)")},
            "e2e": primary["e2e"], "gpu_launches": primary["gpu_launches"],
            "kernel_ms_per_step": primary["kernel_ms_per_step"],
            "roofline": short_rf(primary["roofline"]), "clocks": primary.get("clocks"),
        }
        if "rank_sum_nt" in primary:
            line["rank_sum_nt"] = primary["rank_sum_nt"]
        if other is not None:
            line["fp64" if other["dtype"] == "f64" else "fp32"] = short_leg(other)
        if fma is not None:
            # the all-FP32 answer to north_star's "FP32 issue-bound roofline": a full leg (roofline with traffic, e2e, clocks)
            line["fp32_fma_pipe"] = short_leg(fma)
            line["fp32_fma_pipe"]["frac"] = fma["roofline"]["frac"]
        if two is not None:
            line["fp32_tensor_2products"] = short_leg(two, with_e2e=False)
            line["fp32_tensor_2products"]["note"] = "opt-in (lsp_config.tensor_products = 2); over the 1e-3 tolerance on few-night cadences"
        if c3 is not None:
            line["c3"] = {"value": c3["value"], "ms_per_step": c3["ms_per_step"], "kernel_ms_per_step": c3["kernel_ms_per_step"],
                          "frac": c3["roofline"]["frac"], "frac_executed": c3["roofline"].get("frac_executed"),
                          "e2e": c3["e2e"]["value"], "fast_math": c3["fast_math"]}
        if c4 is not None:
            line["c4"] = {k: c4[k] for k in ("value", "T_compute_ms", "T_d2h_ms", "T_pipelined_ms", "T_over_max", "d2h_GBps",
                                             "fully_overlapped")}
        if fva is not None:
            line["fast_vs_accurate"] = fva
        if c5 is not None:
            line["c5"] = c5
        if overlap is not None:
            line["d2h_overlap"] = overlap
        if cpu is not None:
            line["cpu_baseline"] = cpu
        for name, v in variants.items():
            line[name] = short_leg(v, with_e2e=False)
        if gls:
            line["generalized"] = gls
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_b200(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
