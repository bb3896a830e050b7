#!/usr/bin/env python
"""bench.py -- (t,f) pair-evaluations/s of the batched Lomb-Scargle hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2|c3|c4] [--dtype f32|f64] [--fast-math]
    python bench.py --impl reference ...          # the CPU oracle, as it stands, on the box's host cores

A "step" is one pass of the whole hot path (SURVEY.md section 8(a) steps 1-6/6', and 7 for host output) over one
batch of seeded synthetic input.  Default workload: BASELINE.json configs[1] (single object, N_t = 10,000,
N_f = 1,000,000, full periodogram), in FP32 (primary line) and FP64 (the "fp64" object of the same line).
  value       device-resident: inputs and output in HBM, CUDA events around each step on the launching stream
  e2e         the same pass through lsp_periodogram_batched_host: pinned HOST inputs, H2D + kernels + D2H inside
              the timed region
  roofline    the dominant kernel against the FMA-pipe (FP32) / FP64-pipe peak: "bound": "alu"
  cpu_baseline  the oracle timed on a bounded sample of the same workload (rank 0, N = 1 only)
Multi-GPU (torchrun, one rank per GPU): every rank runs its own object of the same shape (seed + rank), no data-path
collective ("scaling": "weak"); times are device times, max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
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
# Tensor path: the same 4 MAC per pair as one FP16 GEMM; the accurate mode issues three products per MAC
# (a_hi b_hi + a_hi b_lo + a_lo b_hi), fast_math one.
TENSOR_PRODUCTS = {False: 3, True: 1}
TENSOR_PEAK_FALLBACK = 1590.0     # TFLOP/s, B200_PROFILING.md fallback (bf16 burst; fp16 : bf16 nominal ratio is 1)


# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel on config 2, from the committed
# `ncu --set full` captures (profiles/r01_ncu_full_*.csv; commands in profiles/r01_README.md).  Other workloads: null.
NCU_TRAFFIC_C2 = {("tensor", False): 20.83e6 + 58.40e6, ("factored", "f32"): 5.94e6 + 0.37e6, ("factored", "f64"): 6.65e6 + 42.69e6}


def measured_tensor_peak():
    """(TFLOP/s, provenance) -- the driver-written cuBLAS bf16 burst figure; FP16 runs at the same nominal rate."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["bf16_tflops"]), "of measured (MEASURED_PEAKS.json bf16_tflops, burst; fp16:bf16 = 1)"
    except Exception:
        return TENSOR_PEAK_FALLBACK, "of fallback (B200_PROFILING.md 1.59 PFLOP/s bf16 burst; fp16:bf16 = 1)"


def roofline(kernel: str, dtype: str, fast: bool, pairs: float, k_ms: float, pipe_ops: float, workload: str = ""):
    """Roofline object of the dominant kernel: achieved = algorithmic flop per launch
    (8 flop per (t,f) pair x pairs) / mean launch duration measured with CUDA events on the launching stream."""
    achieved = pairs * FLOP_PER_PAIR / (k_ms * 1e-3) / 1e12
    traffic = None
    if workload == "c2":
        traffic = NCU_TRAFFIC_C2.get((kernel, bool(fast)) if kernel == "tensor" else (kernel, dtype))
    if kernel == "tensor":
        peak, prov = measured_tensor_peak()
        prod = TENSOR_PRODUCTS[bool(fast)]
        return {"bound": "tensor", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "traffic": traffic, "kernel": "lsp_tensor_kernel<float,%d>" % int(bool(fast)), "flop_per_pair": FLOP_PER_PAIR,
                "peak_is": prov,
                "executed_flop_per_pair": FLOP_PER_PAIR * prod,
                "executed_tflops": achieved * prod, "frac_executed": achieved * prod / peak,
                "note": "FP16 hi+lo split operands: %d tcgen05 products per algorithmic MAC" % prod}
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
            "kernel": "lsp_factored_ws_kernel<%s>" % ("float" if dtype == "f32" else "double"),
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
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-secondary", action="store_true", help="skip the other-precision leg")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the cpu_baseline sample")
    return ap.parse_args()


def workload_for(name: str, dtype: str, rank: int):
    from workloads import make_config
    from workloads.configs import config_seed  # noqa: F401  (seed recipe: DESIGN.md "Input recipe")
    cfg = {"c2": 2, "c3": 3, "c4": 4, "c5": 5}[name]
    # weak scaling: rank r draws its own object(s) from the same generator with sweep-point index r
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
        oracle.periodogram(sub.offsets, sub.t, sub.y, w.f_min, w.f_max, w.n_freq, k_list=ks)

    return run, int(sub.n_obs) * int(ks.size), int(cores), desc


def cpu_baseline(w, seconds: float):
    run, pairs, cores, desc = oracle_sample_runner(w, seconds)
    t0 = time.perf_counter()
    run()
    dt = time.perf_counter() - t0
    return {"value": pairs / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
            "seconds": round(dt, 3)}


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
        return (f"BASELINE.json configs[2]: {w.n_obj} objects, N_t in [50,500] (sum {w.n_obs}), N_f={w.n_freq}, "
                f"best period only")
    return (f"BASELINE.json configs[3]: {w.n_obj} objects (sum N_t {w.n_obs}), N_f={w.n_freq}, full periodogram to "
            f"pinned host over copy streams")


# ---- the B200 leg -----------------------------------------------------------------------------------------------
class Leg:
    """One precision of one workload on this rank's GPU: device-resident steps and end-to-end (host buffer) steps."""

    def __init__(self, pkg, torch, w, name: str, dtype: str, fast_math: bool, kernel: str, device: int):
        self.torch, self.w, self.name, self.dtype = torch, w, name, dtype
        self.tdt = torch.float32 if dtype == "f32" else torch.float64
        self.plan = pkg.Plan(w.f_min, w.f_max, w.n_freq, dtype, fast_math=fast_math and dtype == "f32", kernel=kernel,
                             device=device)
        self.plan.set_timing(True)
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
        self.kernel_ms = []

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
            self.kernel_ms.append(self.plan.last_kernel_ms())
        return info


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


def run_leg(args, pkg, torch, dist, rank, world, device, dtype, flush, with_clocks: bool, kernel=None, fast=None,
            with_e2e: bool = True):
    w = workload_for(args.workload, dtype, rank)
    kernel = args.kernel if kernel is None else kernel
    fast = bool(args.fast_math if fast is None else fast) and dtype == "f32"
    leg = Leg(pkg, torch, w, args.workload, dtype, fast, kernel, device)
    pairs_step = w.pairs
    pairs_all = pairs_step
    if world > 1:
        tt = torch.tensor([float(pairs_step)], dtype=torch.float64, device="cuda")
        dist.all_reduce(tt, op=dist.ReduceOp.SUM)
        pairs_all = float(tt.item())
    sampler = ClockSampler(device) if with_clocks else None
    if sampler:
        sampler.__enter__()
    total_ms, info = timed_loop(torch, dist, world, leg, leg.step_device, args.steps, args.warmup, flush)
    dev_launches, kernel_ms = leg.launches, list(leg.kernel_ms)
    leg.launches, leg.kernel_ms = 0, []
    ms_step = total_ms / args.steps
    k_ms = sum(kernel_ms) / len(kernel_ms)
    # measured pipe peak with the same clocks the kernels see (register-only FFMA2 / DFMA loops, lsp_pipe_peak)
    pipe_ops, _ = pkg.lsp_pipe_peak(1 if dtype == "f32" else 2, device)
    out = {
        "dtype": dtype,
        "value": pairs_all * args.steps / (total_ms * 1e-3),
        "ms_per_step": ms_step,
        "kernel": info["kernel"], "n_split": info["n_split"], "fast_math": fast,
        "kernel_ms_per_step": k_ms,
        "gpu_launches": dev_launches,
        "roofline": roofline(info["kernel"], dtype, fast, pairs_step, k_ms, pipe_ops, args.workload),
    }
    if with_e2e:
        e2e_ms, _ = timed_loop(torch, dist, world, leg, leg.step_e2e, args.steps, args.warmup, flush)
        h2d, d2h = leg.e2e_bytes()
        out["e2e"] = {"value": pairs_all * args.steps / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                      "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms / args.steps}
    if sampler:
        sampler.__exit__()
    if sampler:
        out["clocks"] = sampler.summary()
    leg.plan.destroy()
    return out, w


def c4_overlap(args, pkg, torch, device, flush):
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
    h_page = torch.empty((w.n_obj, w.n_freq), dtype=torch.float32)
    h_page.fill_(0.0)                                  # touch the pages once, outside the timed region
    pageable = {}
    for mode in ("staged", "plain"):
        os.environ["LSP_PAGEABLE"] = mode
        pl = pkg.Plan(w.f_min, w.f_max, w.n_freq, "f32", kernel=args.kernel, device=device, n_copy_streams=n_streams,
                      chunk_bytes=chunk_bytes)
        pageable[mode] = timeit(lambda: pl.periodogram_batched(d_off, d_t, d_y, host_out=h_page, h_offsets=h_off), reps=2)
        pl.destroy()
    os.environ.pop("LSP_PAGEABLE", None)
    gb = w.n_obj * row / 1e9
    return {"T_compute_ms": tc, "T_d2h_ms": td, "T_pipelined_ms": tp, "d2h_GBps": gb / (td * 1e-3),
            "T_pageable_staged_ms": pageable["staged"], "T_pageable_plain_ms": pageable["plain"],
            "hidden_fraction": (tc + td - tp) / min(tc, td), "T_over_max": tp / max(tc, td),
            "fully_overlapped": bool(tp <= 1.05 * max(tc, td) + td / max(1, -(-w.n_obj // objs_per_chunk))),
            "chunk_bytes": chunk_bytes, "n_copy_streams": n_streams, "bytes": w.n_obj * row}


def run_c5(args, pkg, torch, device, flush):
    """BASELINE.json configs[4]: single object, N_t x N_f sweep in FP32 and FP64; pairs/s and roofline fraction per
    point (device-resident, full periodogram; kernel time from CUDA events on the launching stream)."""
    from workloads import make_config, C5_NT, C5_NF
    dev = torch.device("cuda", device)
    rows = []
    for dtype in ("f32", "f64"):
        pipe_ops, _ = pkg.lsp_pipe_peak(1 if dtype == "f32" else 2, device)
        tdt = torch.float32 if dtype == "f32" else torch.float64
        for i, nt in enumerate(C5_NT):
            for j, nf in enumerate(C5_NF):
                w = make_config(5, dtype=dtype, n_t=nt, n_freq=nf, point=i * len(C5_NF) + j)
                plan = pkg.Plan(w.f_min, w.f_max, w.n_freq, dtype, kernel=args.kernel, fast_math=args.fast_math and dtype == "f32",
                                device=device)
                plan.set_timing(True)
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
                    kms += plan.last_kernel_ms()
                info = plan.last_call_info()
                rf = roofline(info["kernel"], dtype, args.fast_math and dtype == "f32", w.pairs, kms / steps, pipe_ops)
                rows.append({"dtype": dtype, "n_t": nt, "n_freq": nf, "pairs": w.pairs, "kernel": info["kernel"],
                             "n_split": info["n_split"], "ms_per_step": tot / steps, "kernel_ms": kms / steps,
                             "pairs_per_s": w.pairs * steps / (tot * 1e-3), "bound": rf["bound"], "roofline_frac": rf["frac"],
                             "frac_executed": rf.get("frac_executed")})
                plan.destroy()
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
    other = None
    variants = {}
    if not args.no_secondary and args.workload == "c2":
        other_dtype = "f64" if args.dtype == "f32" else "f32"
        other, _ = run_leg(args, pkg, torch, dist, rank, world, local_rank, other_dtype, flush, False)
        if args.kernel == "auto" and not args.fast_math:
            # the other FP32 formulations on the same workload (device-resident only): the FFMA2 contraction on the
            # FMA pipe (north_star's "FP32 issue-bound roofline") and the fast_math tensor mode
            variants["fp32_fma_pipe"], _ = run_leg(args, pkg, torch, dist, rank, world, local_rank, "f32", flush, False,
                                                   kernel="factored", fast=False, with_e2e=False)
            variants["fp32_fast_math"], _ = run_leg(args, pkg, torch, dist, rank, world, local_rank, "f32", flush, False,
                                                    kernel="auto", fast=True, with_e2e=False)
            # the paper-shaped kernel (thread = frequency, one sincos per pair): __sincosf-class vs accurate sincos
            # (PAPER.md:L423-433), the comparison north_star asks for
            saved_steps = args.steps
            args.steps = max(3, min(args.steps, 5))
            variants["direct_fp32_sincosf"], _ = run_leg(args, pkg, torch, dist, rank, world, local_rank, "f32", flush, False,
                                                         kernel="direct", fast=True, with_e2e=False)
            variants["direct_fp32_accurate"], _ = run_leg(args, pkg, torch, dist, rank, world, local_rank, "f32", flush, False,
                                                          kernel="direct", fast=False, with_e2e=False)
            variants["direct_fp64"], _ = run_leg(args, pkg, torch, dist, rank, world, local_rank, "f64", flush, False,
                                                 kernel="direct", fast=False, with_e2e=False)
            args.steps = saved_steps
    gls = None
    if not args.no_secondary and args.workload in ("c2", "c3") and rank == 0 and world == 1:
        gls = {}
        for dt in (("f32", "f64") if args.workload == "c2" else ("f32",)):
            g = run_generalized(args, pkg, torch, local_rank, flush, dt)
            std_ms = primary["ms_per_step"] if dt == primary["dtype"] else (other["ms_per_step"] if other else None)
            g["time_vs_standard_same_dtype"] = (g["ms_per_step"] / std_ms) if std_ms else None
            gls[dt] = g
    overlap = None
    if args.workload == "c4" and rank == 0 and world == 1:
        overlap = c4_overlap(args, pkg, torch, local_rank, flush)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(w, args.cpu_seconds)
    if rank == 0:
        line = {
            "metric": METRIC, "value": primary["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": primary["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": primary["dtype"], "data": "synthetic",
            "config": {"workload": describe_workload(args.workload, w), "kernel": primary["kernel"],
                       "fast_math": bool(args.fast_math and args.dtype == "f32"), "n_split": primary["n_split"],
                       "l2": "flushed between steps (256 MiB fill, outside the event pairs)",
                       "parallelism": f"replicas x{world} (one object set per rank, no collective)"},
            "e2e": primary["e2e"], "gpu_launches": primary["gpu_launches"],
            "kernel_ms_per_step": primary["kernel_ms_per_step"],
            "roofline": primary["roofline"], "clocks": primary.get("clocks"),
        }
        if other is not None:
            line[other["dtype"] == "f64" and "fp64" or "fp32"] = {k: other[k] for k in
                                                                 ("value", "ms_per_step", "kernel_ms_per_step", "e2e", "roofline",
                                                                  "gpu_launches", "kernel")}
        for name, v in variants.items():
            line[name] = {k: v[k] for k in ("value", "ms_per_step", "kernel_ms_per_step", "roofline", "gpu_launches", "kernel")}
        if gls:
            line["generalized"] = gls
        if overlap is not None:
            line["d2h_overlap"] = overlap
        if cpu is not None:
            line["cpu_baseline"] = cpu
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
