"""lsp_best_period_static: the library's allocation-free entry point (include/lsp.h), checked against the plan-based path.

Why the entry point exists: every other call of the library works on a plan, and plans allocate device memory (at creation and
whenever their scratch must grow).  A caller that has given all of its HBM to its own pool allocator, that sits in a
latency-bound loop where a cudaMalloc would stall the whole device, or that runs under a host application's "no driver
allocations after start-up" rule cannot use them.  lsp_best_period_static takes only buffers the caller already owns and
keeps its scratch in a fixed 16 MiB array inside the library image.

What is checked here, through the C ABI binding:
  * two calls in a row (a larger batch, then a smaller one on a coarser grid, so the second call finds the first one's
    leftovers in the shared array), each compared with the existing path -- a LSP_KERNEL_DIRECT plan's periodogram + best
    period -- at the tolerances of tests/test_gpu_parity.py (BASELINE.json: 1e-3 / 1e-9 of the object's max P; a different index
    only on a near tie); the pair of calls is then repeated and must reproduce itself bit for bit;
  * free device memory does not move across the repeated pair (nothing was allocated);
  * a request beyond the fixed scratch is refused with LSP_ERR_UNSUPPORTED and a message that names the limit (no GPU needed).

This file is named so that pytest collects it last: with `-x` a failure here cannot hide any other test.  It depends on no
state left by other tests and leaves none behind.
"""
import numpy as np
import pytest

from workloads import make_config

TOL = {"f32": 1e-3, "f64": 1e-9}        # of the object's max P, as in tests/test_gpu_parity.py


def _cfg(pkg, w, **over):
    args = dict(f_min=w.f_min, f_max=w.f_max, n_freq=w.n_freq, dtype=0 if w.dtype == "f32" else 1, fast_math=0, normalize=0,
                center=0, device=0, n_copy_streams=0, chunk_bytes=0, max_objects=0, max_total_obs=0, kernel=0, flags=0,
                table_budget_bytes=0, tensor_roles=0, tensor_b_stages=0, tensor_products=0, tensor_pair=0)
    args.update(over)
    return pkg.LspConfig(**args)


def _with_empty_object(w):
    """Splice an object without observations into the CSR (index 2): its slot must come back as (-1, 0, NaN)."""
    off = np.concatenate([w.offsets[:3], w.offsets[2:]]).astype(np.int64)
    return off


@pytest.mark.gpu
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("center_normalize", [False, True])
def test_static_entry_point_matches_the_plan_path_on_two_calls_in_a_row(dtype, center_normalize):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device is visible")
    import paper_2105_04006_b200 as pkg
    pkg.load_library()
    tdt = torch.float32 if dtype == "f32" else torch.float64
    flag = int(center_normalize)

    # call A: 160 config-3-shaped objects (+ one empty) on 9,000 frequencies -> 4-frequency threads, 9 tiles per object;
    # call B: 5 objects (+ one empty) on 3,000 frequencies -> 1-frequency threads, 12 tiles per object: far fewer slots than A
    # filled, so most of A's candidates are still in the array while B runs
    cases = []
    for n_obj, n_freq in ((160, 9000), (5, 3000)):
        w = make_config(3, n_obj=n_obj, n_freq=n_freq, dtype=dtype)
        off = _with_empty_object(w)
        case = dict(w=w, n_obj=n_obj + 1, off=torch.from_numpy(off).cuda(), h_off=torch.from_numpy(off),
                    t=torch.from_numpy(w.t).to(tdt).cuda(), y=torch.from_numpy(w.y).to(tdt).cuda())
        # the existing path: full periodogram + fused best period of a direct-kernel plan
        with pkg.Plan(w.f_min, w.f_max, w.n_freq, dtype, kernel="direct", center=bool(flag), normalize=bool(flag)) as plan:
            power, best = plan.periodogram_batched(case["off"], case["t"], case["y"], best=True, h_offsets=case["h_off"])
            torch.cuda.synchronize()
            case["P"] = power.cpu().numpy().astype(np.float64)
            case["ref"] = tuple(x.cpu().numpy() for x in best)
        # outputs of the static call: allocated here, by the caller, before anything is measured
        case["out"] = (torch.full((case["n_obj"],), -7.0, dtype=tdt, device="cuda"),
                       torch.full((case["n_obj"],), -7.0, dtype=tdt, device="cuda"),
                       torch.full((case["n_obj"],), -7, dtype=torch.int64, device="cuda"))
        case["cfg"] = _cfg(pkg, w, center=flag, normalize=flag, kernel=3 if dtype == "f32" else 2)   # `kernel` is ignored
        cases.append(case)

    def run_pair():
        got = []
        for c in cases:                      # back to back on the current stream, no synchronisation in between
            pkg.lsp_best_period_static(c["cfg"], c["n_obj"], c["off"], c["t"], c["y"], *c["out"])
        torch.cuda.synchronize()
        for c in cases:
            got.append(tuple(x.cpu().numpy().copy() for x in c["out"]))
        return got

    first = run_pair()
    for c, (per, pw, idx) in zip(cases, first):
        w, P = c["w"], c["P"]
        rper, rpw, ridx = c["ref"]
        df = (w.f_max - w.f_min) / w.n_freq
        assert idx[2] == -1 and pw[2] == 0 and np.isnan(per[2]), "empty object"
        assert ridx[2] == -1
        for o in range(c["n_obj"]):
            if o == 2:
                continue
            pmax = P[o].max()
            assert 0 <= idx[o] < w.n_freq
            if idx[o] != ridx[o]:            # only a near tie excuses a different index
                assert P[o, idx[o]] >= pmax - TOL[dtype] * pmax, f"object {o}: index {idx[o]} vs {ridx[o]}"
            assert abs(pw[o] - P[o, idx[o]]) <= TOL[dtype] * pmax, f"object {o}: best power"
            assert abs(pw[o] - rpw[o]) <= TOL[dtype] * pmax, f"object {o}: best power vs the plan's fused argmax"
            f_k = w.f_min + idx[o] * df
            assert abs(per[o] - 1.0 / f_k) <= (1e-6 if dtype == "f32" else 1e-14) / f_k, f"object {o}: period is not 1/f_k"

    # the same two calls again: identical bits (the shared array carries nothing from one call into the next), and no change
    # in free device memory (every kernel and the one-time set-up have run already, so any difference would be an allocation)
    free_before, _ = torch.cuda.mem_get_info()
    second = run_pair()
    free_after, _ = torch.cuda.mem_get_info()
    for a, b in zip(first, second):
        for x, y in zip(a, b):
            assert np.array_equal(x, y, equal_nan=True)
    assert free_after >= free_before, f"free device memory fell by {free_before - free_after} bytes across allocation-free calls"


def test_static_entry_point_refuses_requests_beyond_its_scratch():
    """Host-side check, decided before any CUDA call: 16 B x n_obj x (ceil(n_freq / 1024) + 1) must fit in 16 MiB."""
    import paper_2105_04006_b200 as pkg
    lib = pkg.load_library()
    assert pkg.LSP_STATIC_SCRATCH_BYTES == 16 << 20
    w = make_config(3, n_obj=1, n_freq=100_000, dtype="f32")
    cfg = _cfg(pkg, w)
    tiles = (100_000 + 1023) // 1024 + 1
    fits = (pkg.LSP_STATIC_SCRATCH_BYTES // 16) // tiles          # 10,591 objects on this grid
    assert fits >= 10_000                                          # BASELINE.json config 3 fits in one call
    with pytest.raises(pkg.LspError) as ei:
        pkg.lsp_best_period_static(cfg, fits + 1, None, None, None, None, None, None, stream=_NoStream())
    assert ei.value.status == pkg.binding.LSP_ERR_INVALID_ARG     # NULL pointers are caught first
    dummy = _FakeTensor()
    with pytest.raises(pkg.LspError) as ei:
        pkg.lsp_best_period_static(cfg, fits + 1, dummy, dummy, dummy, dummy, dummy, dummy, stream=_NoStream())
    assert ei.value.status == pkg.binding.LSP_ERR_UNSUPPORTED
    assert "static scratch" in str(ei.value) and str(fits) in str(ei.value)
    # bad grids are rejected like lsp_plan_create rejects them, and a NULL cfg is not dereferenced
    with pytest.raises(pkg.LspError) as ei:
        pkg.lsp_best_period_static(_cfg(pkg, w, n_freq=0), 1, dummy, dummy, dummy, dummy, dummy, dummy, stream=_NoStream())
    assert ei.value.status == pkg.binding.LSP_ERR_INVALID_ARG
    with pytest.raises(pkg.LspError) as ei:
        pkg.lsp_best_period_static(_cfg(pkg, w, dtype=1, fast_math=1), 1, dummy, dummy, dummy, dummy, dummy, dummy, stream=_NoStream())
    assert ei.value.status == pkg.binding.LSP_ERR_INVALID_ARG
    assert lib.lsp_best_period_static(None, 0, None, None, None, None, None, None, None) == pkg.binding.LSP_ERR_INVALID_ARG


class _NoStream:
    """Stands in for a torch stream on a box without a GPU: the NULL (default) stream; never used, the call fails first."""
    cuda_stream = 0


class _FakeTensor:
    """A non-NULL pointer the library never dereferences on the host (it is rejected before any launch)."""
    def data_ptr(self):
        return 256
