"""Thin ctypes binding of liblsp_b200.so (include/lsp.h).  Argument marshalling only: every step of the
Lomb-Scargle hot path runs inside the CUDA library; torch is used for device memory and streams.

The module-level functions carry the C ABI's names (lsp_plan_create, lsp_periodogram_batched, lsp_best_period,
lsp_destroy); `Plan` is a small convenience wrapper around them.  If the shared library is missing and cannot
be built, importing this module raises: there is no CPU fallback.
"""
from __future__ import annotations

import ctypes
from typing import Optional

import torch

from . import build as _build

LSP_F32, LSP_F64 = 0, 1
LSP_KERNEL_AUTO, LSP_KERNEL_DIRECT, LSP_KERNEL_FACTORED, LSP_KERNEL_TENSOR = 0, 1, 2, 3
LSP_OK, LSP_ERR_INVALID_ARG, LSP_ERR_CUDA, LSP_ERR_OOM, LSP_ERR_UNSUPPORTED = 0, 1, 2, 3, 4
_STATUS = {0: "LSP_OK", 1: "LSP_ERR_INVALID_ARG", 2: "LSP_ERR_CUDA", 3: "LSP_ERR_OOM", 4: "LSP_ERR_UNSUPPORTED"}
_KERNELS = {"auto": LSP_KERNEL_AUTO, "direct": LSP_KERNEL_DIRECT, "factored": LSP_KERNEL_FACTORED,
            "tensor": LSP_KERNEL_TENSOR}
_KERNEL_NAMES = {v: k for k, v in _KERNELS.items()}

EXPORTS = ("lsp_plan_create", "lsp_periodogram_batched", "lsp_best_period", "lsp_periodogram_batched_host",
           "lsp_periodogram_generalized", "lsp_periodogram_generalized_host", "lsp_best_merge", "lsp_best_period_static",
           "lsp_destroy",
           "lsp_last_error",
           "lsp_last_call_info", "lsp_set_timing", "lsp_last_kernel_ms", "lsp_version")
LSP_FLAG_PAGEABLE_STAGED = 1
LSP_STATIC_SCRATCH_BYTES = 16 << 20      # include/lsp.h: fixed scratch of lsp_best_period_static


class LspConfig(ctypes.Structure):
    """struct lsp_config of include/lsp.h (field order and widths must match)."""
    _fields_ = [
        ("f_min", ctypes.c_double), ("f_max", ctypes.c_double), ("n_freq", ctypes.c_int64),
        ("dtype", ctypes.c_int32), ("fast_math", ctypes.c_int32), ("normalize", ctypes.c_int32),
        ("center", ctypes.c_int32), ("device", ctypes.c_int32), ("n_copy_streams", ctypes.c_int32),
        ("chunk_bytes", ctypes.c_int64), ("max_objects", ctypes.c_int64), ("max_total_obs", ctypes.c_int64),
        ("kernel", ctypes.c_int32), ("flags", ctypes.c_int32),
        ("table_budget_bytes", ctypes.c_int64), ("tensor_roles", ctypes.c_int32), ("tensor_b_stages", ctypes.c_int32),
        ("tensor_products", ctypes.c_int32), ("tensor_pair", ctypes.c_int32),
    ]


class LspError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{_STATUS.get(status, status)}: {message}")
        self.status = status


_lib = None


def load_library(path: Optional[str] = None) -> ctypes.CDLL:
    """dlopen the in-tree liblsp_b200.so (building it with nvcc first if it is missing or stale)."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    lib = ctypes.CDLL(path or _build.build())
    vp, i64, i32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32
    lib.lsp_plan_create.argtypes = [ctypes.POINTER(LspConfig), ctypes.POINTER(vp)]
    lib.lsp_plan_create.restype = ctypes.c_int
    lib.lsp_periodogram_batched.argtypes = [vp, i64, vp, vp, vp, vp, vp, i32, vp, vp, vp, vp]
    lib.lsp_periodogram_batched.restype = ctypes.c_int
    lib.lsp_best_period.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.lsp_best_period.restype = ctypes.c_int
    lib.lsp_periodogram_batched_host.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.lsp_periodogram_batched_host.restype = ctypes.c_int
    lib.lsp_periodogram_generalized.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.lsp_periodogram_generalized.restype = ctypes.c_int
    lib.lsp_periodogram_generalized_host.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.lsp_periodogram_generalized_host.restype = ctypes.c_int
    lib.lsp_best_merge.argtypes = [vp, i64, i32, vp, vp, vp, vp, vp, vp]
    lib.lsp_best_merge.restype = ctypes.c_int
    lib.lsp_best_period_static.argtypes = [ctypes.POINTER(LspConfig), i64, vp, vp, vp, vp, vp, vp, vp]
    lib.lsp_best_period_static.restype = ctypes.c_int
    lib.lsp_destroy.argtypes = [vp]
    lib.lsp_destroy.restype = None
    lib.lsp_last_error.argtypes = [vp]
    lib.lsp_last_error.restype = ctypes.c_char_p
    lib.lsp_last_call_info.argtypes = [vp, ctypes.POINTER(i64), ctypes.POINTER(i64), ctypes.POINTER(i32),
                                       ctypes.POINTER(i32), ctypes.POINTER(i64), ctypes.POINTER(i32), ctypes.POINTER(i32)]
    lib.lsp_last_call_info.restype = None
    lib.lsp_set_timing.argtypes = [vp, i32]
    lib.lsp_set_timing.restype = None
    lib.lsp_last_kernel_ms.argtypes = [vp]
    lib.lsp_last_kernel_ms.restype = ctypes.c_float
    lib.lsp_version.argtypes = []
    lib.lsp_version.restype = ctypes.c_char_p
    if path is None:
        _lib = lib
    return lib


def _check(status: int, plan=None):
    if status != LSP_OK:
        msg = load_library().lsp_last_error(plan).decode(errors="replace")
        raise LspError(status, msg)


def _dptr(x: Optional[torch.Tensor]):
    return None if x is None else ctypes.c_void_p(x.data_ptr())


def _stream_ptr(stream) -> ctypes.c_void_p:
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


# ---- the C ABI's four calls, same names ---------------------------------------------------------------------
def lsp_plan_create(cfg: LspConfig) -> ctypes.c_void_p:
    plan = ctypes.c_void_p()
    _check(load_library().lsp_plan_create(ctypes.byref(cfg), ctypes.byref(plan)))
    return plan


def lsp_periodogram_batched(plan, n_obj: int, d_offsets, h_offsets, d_t, d_y, out_power, out_is_host: bool,
                            d_best_period=None, d_best_power=None, d_best_index=None, stream=None) -> None:
    h_ptr = None if h_offsets is None else ctypes.c_void_p(h_offsets.data_ptr())
    _check(load_library().lsp_periodogram_batched(plan, int(n_obj), _dptr(d_offsets), h_ptr, _dptr(d_t), _dptr(d_y),
                                                  _dptr(out_power), int(bool(out_is_host)), _dptr(d_best_period),
                                                  _dptr(d_best_power), _dptr(d_best_index), _stream_ptr(stream)), plan)


def lsp_best_period(plan, n_obj: int, d_offsets, h_offsets, d_t, d_y, d_best_period, d_best_power, d_best_index,
                    stream=None) -> None:
    h_ptr = None if h_offsets is None else ctypes.c_void_p(h_offsets.data_ptr())
    _check(load_library().lsp_best_period(plan, int(n_obj), _dptr(d_offsets), h_ptr, _dptr(d_t), _dptr(d_y),
                                          _dptr(d_best_period), _dptr(d_best_power), _dptr(d_best_index),
                                          _stream_ptr(stream)), plan)


def lsp_periodogram_batched_host(plan, n_obj: int, h_offsets, h_t, h_y, h_out_power=None, h_best_period=None,
                                 h_best_power=None, h_best_index=None, stream=None) -> None:
    """All-HOST form (include/lsp.h): every tensor is a host tensor; H2D, kernels and D2H run inside the call."""
    _check(load_library().lsp_periodogram_batched_host(plan, int(n_obj), _dptr(h_offsets), _dptr(h_t), _dptr(h_y),
                                                       _dptr(h_out_power), _dptr(h_best_period), _dptr(h_best_power),
                                                       _dptr(h_best_index), _stream_ptr(stream)), plan)


def lsp_periodogram_generalized_host(plan, n_obj: int, h_offsets, h_t, h_y, h_sigma, h_out_power=None, h_best_period=None,
                                     h_best_power=None, h_best_index=None, stream=None) -> None:
    """All-HOST form of the generalised LSP (include/lsp.h): H2D, kernels and D2H (chunk ring + copy streams) inside the call."""
    _check(load_library().lsp_periodogram_generalized_host(plan, int(n_obj), _dptr(h_offsets), _dptr(h_t), _dptr(h_y),
                                                           _dptr(h_sigma), _dptr(h_out_power), _dptr(h_best_period),
                                                           _dptr(h_best_power), _dptr(h_best_index), _stream_ptr(stream)), plan)


def lsp_periodogram_generalized(plan, n_obj: int, d_offsets, h_offsets, d_t, d_y, d_sigma, d_out_power=None,
                                d_best_period=None, d_best_power=None, d_best_index=None, stream=None) -> None:
    """Generalised LSP (floating mean + errors; include/lsp.h): device tensors, asynchronous on `stream`."""
    h_ptr = None if h_offsets is None else ctypes.c_void_p(h_offsets.data_ptr())
    _check(load_library().lsp_periodogram_generalized(plan, int(n_obj), _dptr(d_offsets), h_ptr, _dptr(d_t), _dptr(d_y),
                                                      _dptr(d_sigma), _dptr(d_out_power), _dptr(d_best_period),
                                                      _dptr(d_best_power), _dptr(d_best_index), _stream_ptr(stream)), plan)


def lsp_best_merge(plan, n_obj: int, n_parts: int, d_part_power, d_part_index, d_best_period, d_best_power, d_best_index,
                   stream=None) -> None:
    """Merge the fused-argmax results of n_parts frequency shards (include/lsp.h): device tensors, asynchronous."""
    _check(load_library().lsp_best_merge(plan, int(n_obj), int(n_parts), _dptr(d_part_power), _dptr(d_part_index),
                                         _dptr(d_best_period), _dptr(d_best_power), _dptr(d_best_index),
                                         _stream_ptr(stream)), plan)


def lsp_best_period_static(cfg: LspConfig, n_obj: int, d_offsets, d_t, d_y, d_best_period, d_best_power, d_best_index,
                           stream=None) -> None:
    """Best period per object through the library's allocation-free entry point (include/lsp.h): no plan, scratch in a fixed
    array inside the library (LSP_STATIC_SCRATCH_BYTES), for callers that may not allocate device memory.  All tensors are the
    caller's own CUDA tensors; asynchronous on `stream`; calls that could overlap on one GPU must be ordered by the caller."""
    _check(load_library().lsp_best_period_static(ctypes.byref(cfg), int(n_obj), _dptr(d_offsets), _dptr(d_t), _dptr(d_y),
                                                 _dptr(d_best_period), _dptr(d_best_power), _dptr(d_best_index),
                                                 _stream_ptr(stream)))


def lsp_destroy(plan) -> None:
    load_library().lsp_destroy(plan)


def lsp_version() -> str:
    return load_library().lsp_version().decode()


# ---- convenience wrapper ---------------------------------------------------------------------------------------
class Plan:
    """One frequency grid + precision + output conventions (lsp_plan).  Buffers are torch tensors."""

    def __init__(self, f_min: float, f_max: float, n_freq: int, dtype: str = "f32", *, fast_math: bool = False,
                 normalize: bool = False, center: bool = False, device: int = 0, n_copy_streams: int = 0,
                 chunk_bytes: int = 0, kernel: str = "auto", max_objects: int = 0, max_total_obs: int = 0,
                 pageable_staged: bool = False, table_budget_bytes: int = 0, tensor_roles: int = 0,
                 tensor_b_stages: int = 0, tensor_products: int = 0, tensor_pair: int = 0):
        if dtype not in ("f32", "f64"):
            raise ValueError("dtype must be 'f32' or 'f64'")
        self.cfg = LspConfig(float(f_min), float(f_max), int(n_freq), LSP_F32 if dtype == "f32" else LSP_F64,
                             int(fast_math), int(normalize), int(center), int(device), int(n_copy_streams),
                             int(chunk_bytes), int(max_objects), int(max_total_obs), _KERNELS[kernel],
                             LSP_FLAG_PAGEABLE_STAGED if pageable_staged else 0, int(table_budget_bytes),
                             int(tensor_roles), int(tensor_b_stages), int(tensor_products), int(tensor_pair))
        self.dtype = dtype
        self.torch_dtype = torch.float32 if dtype == "f32" else torch.float64
        self.n_freq = int(n_freq)
        self.device = torch.device("cuda", device)
        self._plan = lsp_plan_create(self.cfg)

    # -- life cycle
    def destroy(self):
        if getattr(self, "_plan", None) is not None:
            lsp_destroy(self._plan)
            self._plan = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    # -- helpers
    def _check_inputs(self, offsets, t, y, h_offsets=None):
        """The C side receives raw pointers and cannot check any of this: a mismatched CSR must become a TypeError here,
        not an out-of-bounds device read there."""
        if offsets.dtype != torch.int64 or not offsets.is_cuda or not offsets.is_contiguous() or offsets.numel() < 1:
            raise TypeError("offsets must be a contiguous CUDA int64 tensor of n_obj + 1 elements")
        for x in (t, y):
            if x.dtype != self.torch_dtype or not x.is_cuda or not x.is_contiguous():
                raise TypeError(f"t and y must be contiguous CUDA tensors of {self.torch_dtype}")
        if t.numel() != y.numel():
            raise TypeError("t and y must have the same number of elements")
        n_obj = int(offsets.numel() - 1)
        if h_offsets is not None:
            if h_offsets.is_cuda or h_offsets.dtype != torch.int64 or not h_offsets.is_contiguous() \
                    or h_offsets.numel() != n_obj + 1:
                raise TypeError("h_offsets must be a contiguous host int64 tensor of n_obj + 1 elements")
            if int(h_offsets[-1]) > t.numel():
                raise TypeError("offsets[n_obj] exceeds the length of t / y")
        return n_obj

    def set_timing(self, on: bool):
        load_library().lsp_set_timing(self._plan, int(on))

    def last_kernel_ms(self) -> float:
        return float(load_library().lsp_last_kernel_ms(self._plan))

    def last_call_info(self) -> dict:
        nl, npairs, nch = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64()
        ku, ns, ts, tp = ctypes.c_int32(), ctypes.c_int32(), ctypes.c_int32(), ctypes.c_int32()
        load_library().lsp_last_call_info(self._plan, ctypes.byref(nl), ctypes.byref(npairs), ctypes.byref(ku),
                                          ctypes.byref(ns), ctypes.byref(nch), ctypes.byref(ts), ctypes.byref(tp))
        return {"launches": nl.value, "pairs": npairs.value, "kernel": _KERNEL_NAMES.get(ku.value, ku.value),
                "n_split": ns.value, "chunks": nch.value, "tensor_shape": ts.value, "tensor_products": tp.value}

    # -- the two calls
    def periodogram_batched(self, offsets, t, y, *, out=None, host_out=None, best: bool = False, h_offsets=None,
                            stream=None):
        """Full periodogram.  Returns (power, best) where power is `out` (device), `host_out` (host) or a new
        device tensor [n_obj, n_freq], and best is None or (period, power, index) device tensors."""
        n_obj = self._check_inputs(offsets, t, y, h_offsets)
        if host_out is not None:
            if host_out.is_cuda or host_out.dtype != self.torch_dtype or host_out.numel() != n_obj * self.n_freq \
                    or not host_out.is_contiguous():
                raise TypeError("host_out must be a contiguous host tensor [n_obj, n_freq] of the plan dtype")
            power, is_host = host_out, True
        else:
            power = out if out is not None else torch.empty((n_obj, self.n_freq), dtype=self.torch_dtype, device=self.device)
            if not power.is_cuda or power.dtype != self.torch_dtype or power.numel() != n_obj * self.n_freq \
                    or not power.is_contiguous():
                raise TypeError("out must be a contiguous CUDA tensor [n_obj, n_freq] of the plan dtype")
            is_host = False
        bp = bw = bi = None
        if best:
            bp = torch.empty(n_obj, dtype=self.torch_dtype, device=self.device)
            bw = torch.empty(n_obj, dtype=self.torch_dtype, device=self.device)
            bi = torch.empty(n_obj, dtype=torch.int64, device=self.device)
        lsp_periodogram_batched(self._plan, n_obj, offsets, h_offsets, t, y, power, is_host, bp, bw, bi, stream)
        return power, ((bp, bw, bi) if best else None)

    def periodogram_batched_host(self, h_offsets, h_t, h_y, *, host_out=None, best_out=None, stream=None):
        """End-to-end call on HOST tensors (pinned for overlap): fills `host_out` [n_obj, n_freq] (or skips the
        periodogram when None) and `best_out` = (period, power, index) host tensors (optional unless host_out
        is None).  Returns after all results are on the host."""
        if h_offsets.is_cuda or h_offsets.dtype != torch.int64 or not h_offsets.is_contiguous() or h_offsets.numel() < 1:
            raise TypeError("h_offsets must be a contiguous host int64 tensor of n_obj + 1 elements")
        n_obj = int(h_offsets.numel() - 1)
        for x in (h_t, h_y):
            if x.is_cuda or x.dtype != self.torch_dtype or not x.is_contiguous():
                raise TypeError(f"h_t and h_y must be contiguous host tensors of {self.torch_dtype}")
        if h_t.numel() != h_y.numel() or int(h_offsets[-1]) > h_t.numel():
            raise TypeError("h_t and h_y must have the same length, at least offsets[n_obj]")
        if host_out is not None and (host_out.is_cuda or host_out.dtype != self.torch_dtype or not host_out.is_contiguous()
                                     or host_out.numel() != n_obj * self.n_freq):
            raise TypeError("host_out must be a contiguous host tensor [n_obj, n_freq] of the plan dtype")
        bp = bw = bi = None
        if best_out is not None:
            bp, bw, bi = best_out
            if bp.is_cuda or bw.is_cuda or bi.is_cuda or bp.dtype != self.torch_dtype or bw.dtype != self.torch_dtype \
                    or bi.dtype != torch.int64 or min(bp.numel(), bw.numel(), bi.numel()) < n_obj:
                raise TypeError("best_out must be host tensors (period, power, index[int64]) of n_obj elements")
        lsp_periodogram_batched_host(self._plan, n_obj, h_offsets, h_t, h_y, host_out, bp, bw, bi, stream)
        return host_out, best_out

    def periodogram_generalized(self, offsets, t, y, sigma, *, out=None, best: bool = False, want_power: bool = True,
                                h_offsets=None, stream=None):
        """Generalised LSP: (power [n_obj, n_freq] or None, best = (period, power, index) or None), device tensors."""
        n_obj = self._check_inputs(offsets, t, y, h_offsets)
        if sigma.dtype != self.torch_dtype or not sigma.is_cuda or not sigma.is_contiguous() or sigma.numel() != y.numel():
            raise TypeError("sigma must be a contiguous CUDA tensor like y")
        power = None
        if want_power:
            power = out if out is not None else torch.empty((n_obj, self.n_freq), dtype=self.torch_dtype, device=self.device)
            if not power.is_cuda or power.dtype != self.torch_dtype or power.numel() != n_obj * self.n_freq or not power.is_contiguous():
                raise TypeError("out must be a contiguous CUDA tensor [n_obj, n_freq] of the plan dtype")
        bp = bw = bi = None
        if best:
            bp = torch.empty(n_obj, dtype=self.torch_dtype, device=self.device)
            bw = torch.empty(n_obj, dtype=self.torch_dtype, device=self.device)
            bi = torch.empty(n_obj, dtype=torch.int64, device=self.device)
        lsp_periodogram_generalized(self._plan, n_obj, offsets, h_offsets, t, y, sigma, power, bp, bw, bi, stream)
        return power, ((bp, bw, bi) if best else None)

    def periodogram_generalized_host(self, h_offsets, h_t, h_y, h_sigma, *, host_out=None, best_out=None, stream=None):
        """Generalised LSP end to end on HOST tensors (pinned for overlap): fills `host_out` [n_obj, n_freq] (or skips the
        periodogram when None) and `best_out` = (period, power, index) host tensors.  Returns after all results are on the host."""
        if h_offsets.is_cuda or h_offsets.dtype != torch.int64 or not h_offsets.is_contiguous() or h_offsets.numel() < 1:
            raise TypeError("h_offsets must be a contiguous host int64 tensor of n_obj + 1 elements")
        n_obj = int(h_offsets.numel() - 1)
        for x in (h_t, h_y, h_sigma):
            if x.is_cuda or x.dtype != self.torch_dtype or not x.is_contiguous():
                raise TypeError(f"h_t, h_y and h_sigma must be contiguous host tensors of {self.torch_dtype}")
        if not (h_t.numel() == h_y.numel() == h_sigma.numel()) or int(h_offsets[-1]) > h_t.numel():
            raise TypeError("h_t, h_y and h_sigma must have the same length, at least offsets[n_obj]")
        if host_out is not None and (host_out.is_cuda or host_out.dtype != self.torch_dtype or not host_out.is_contiguous()
                                     or host_out.numel() != n_obj * self.n_freq):
            raise TypeError("host_out must be a contiguous host tensor [n_obj, n_freq] of the plan dtype")
        bp = bw = bi = None
        if best_out is not None:
            bp, bw, bi = best_out
            if bp.is_cuda or bw.is_cuda or bi.is_cuda or bp.dtype != self.torch_dtype or bw.dtype != self.torch_dtype \
                    or bi.dtype != torch.int64 or min(bp.numel(), bw.numel(), bi.numel()) < n_obj:
                raise TypeError("best_out must be host tensors (period, power, index[int64]) of n_obj elements")
        lsp_periodogram_generalized_host(self._plan, n_obj, h_offsets, h_t, h_y, h_sigma, host_out, bp, bw, bi, stream)
        return host_out, best_out

    def best_merge(self, part_power, part_index, *, stream=None):
        """Merge per-shard (power, GLOBAL index) candidates, tensors [n_parts, n_obj] on this plan's device, into
        (period, power, index) on this plan's (global) grid.  The tie rule and period = 1/f_k live in the library."""
        if part_power.dim() != 2 or part_power.shape != part_index.shape or part_power.dtype != self.torch_dtype \
                or part_index.dtype != torch.int64 or not part_power.is_cuda or not part_index.is_cuda \
                or not part_power.is_contiguous() or not part_index.is_contiguous():
            raise TypeError("part_power [n_parts, n_obj] (plan dtype) and part_index [n_parts, n_obj] (int64): contiguous CUDA tensors")
        n_parts, n_obj = part_power.shape
        out = (torch.empty(n_obj, dtype=self.torch_dtype, device=self.device),
               torch.empty(n_obj, dtype=self.torch_dtype, device=self.device),
               torch.empty(n_obj, dtype=torch.int64, device=self.device))
        lsp_best_merge(self._plan, n_obj, n_parts, part_power, part_index, out[0], out[1], out[2], stream)
        return out

    def best_period(self, offsets, t, y, *, out=None, h_offsets=None, stream=None):
        """Fused best period: (period, power, index) device tensors; the periodogram is never materialised."""
        n_obj = self._check_inputs(offsets, t, y, h_offsets)
        if out is None:
            out = (torch.empty(n_obj, dtype=self.torch_dtype, device=self.device),
                   torch.empty(n_obj, dtype=self.torch_dtype, device=self.device),
                   torch.empty(n_obj, dtype=torch.int64, device=self.device))
        lsp_best_period(self._plan, n_obj, offsets, h_offsets, t, y, out[0], out[1], out[2], stream)
        return out
