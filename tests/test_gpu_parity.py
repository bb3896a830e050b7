"""GPU parity: the CUDA path (through the C ABI binding) against the CPU oracle, element by element, on the
same seeded inputs.  Tolerances are BASELINE.json's: FP64 |dP| <= 1e-9 max P, FP32 |dP| <= 1e-3 max P per
object; best period equal to the oracle's unless the oracle's power at the GPU's index is within that
tolerance of the oracle's maximum (reading a7).
"""
import numpy as np
import pytest

from workloads import make_config, Workload

pytestmark = pytest.mark.gpu

TOL = {"f32": 1e-3, "f64": 1e-9}


@pytest.fixture(scope="module")
def lsp():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device is visible")
    import paper_2105_04006_b200 as pkg
    pkg.load_library()
    return pkg


def to_device(w: Workload):
    import torch
    dt = torch.float32 if w.dtype == "f32" else torch.float64
    return (torch.from_numpy(w.offsets).cuda(), torch.from_numpy(w.t).to(dt).cuda(), torch.from_numpy(w.y).to(dt).cuda())


def gpu_full(lsp, w: Workload, *, kernel="auto", fast_math=False, best=True, **kw):
    off, t, y = to_device(w)
    with lsp.Plan(w.f_min, w.f_max, w.n_freq, w.dtype, kernel=kernel, fast_math=fast_math, **kw) as plan:
        power, b = plan.periodogram_batched(off, t, y, best=best, h_offsets=__import__("torch").from_numpy(w.offsets))
        info = plan.last_call_info()
        P = power.cpu().numpy().astype(np.float64)
        bb = None if b is None else tuple(x.cpu().numpy() for x in b)
    return P, bb, info


def gpu_best(lsp, w: Workload, *, kernel="auto", fast_math=False, **kw):
    off, t, y = to_device(w)
    with lsp.Plan(w.f_min, w.f_max, w.n_freq, w.dtype, kernel=kernel, fast_math=fast_math, **kw) as plan:
        b = plan.best_period(off, t, y)
        info = plan.last_call_info()
        return tuple(x.cpu().numpy() for x in b), info


def assert_power_parity(P_gpu, P_ref, dtype, what=""):
    assert P_gpu.shape == P_ref.shape
    assert np.all(np.isfinite(P_gpu)), f"{what}: non-finite power"
    for o in range(P_ref.shape[0]):
        pmax = P_ref[o].max() if P_ref.shape[1] else 0.0
        err = np.max(np.abs(P_gpu[o] - P_ref[o])) if P_ref.shape[1] else 0.0
        assert err <= TOL[dtype] * pmax + 1e-300, f"{what}: object {o}: max|dP| = {err:.3e} > {TOL[dtype]:.0e} * {pmax:.3e}"


def assert_best_parity(best_gpu, P_ref, w: Workload, dtype, oracle, what=""):
    per, pw, idx = best_gpu
    ridx, rpw, rper = oracle.best(w.offsets, P_ref, w.f_min, w.f_max, w.n_freq)
    df = (w.f_max - w.f_min) / w.n_freq
    for o in range(w.n_obj):
        if ridx[o] < 0:
            assert idx[o] == -1 and np.isnan(per[o]) and pw[o] == 0
            continue
        pmax = rpw[o]
        assert 0 <= idx[o] < w.n_freq
        if idx[o] != ridx[o]:   # a near tie is the only excuse
            assert P_ref[o, idx[o]] >= pmax - TOL[dtype] * pmax, f"{what}: object {o}: index {idx[o]} vs {ridx[o]}"
        assert abs(pw[o] - P_ref[o, idx[o]]) <= TOL[dtype] * pmax, f"{what}: object {o}: best power"
        f_k = w.f_min + idx[o] * df
        rel = 1e-6 if dtype == "f32" else 1e-14
        assert abs(per[o] - 1.0 / f_k) <= rel / f_k, f"{what}: object {o}: period is not 1/f_k"


def oracle_full(oracle, w: Workload):
    return oracle.periodogram(w.offsets, w.t, w.y, w.f_min, w.f_max, w.n_freq)


# ---- config 1: single object, FP64, full + best -------------------------------------------------------------
@pytest.mark.parametrize("kernel", ["direct", "factored"])
def test_config1_full_and_best_f64(lsp, oracle, kernel):
    w = make_config(1)
    P_ref = oracle_full(oracle, w)
    P, best, info = gpu_full(lsp, w, kernel=kernel)
    assert info["kernel"] == kernel and info["pairs"] == w.pairs
    assert_power_parity(P, P_ref, "f64", f"c1/{kernel}")
    assert_best_parity(best, P_ref, w, "f64", oracle, f"c1/{kernel}")
    assert abs(best[0][0] - 0.3) < 0.002


# ---- config 2 shape: one long object, large f*t, all precisions and kernels -------------------------------
@pytest.mark.parametrize("dtype,fast", [("f64", False), ("f32", False), ("f32", True)])
@pytest.mark.parametrize("kernel", ["direct", "factored", "tensor"])
def test_config2_shape_small(lsp, oracle, dtype, fast, kernel):
    if kernel == "tensor" and dtype == "f64":
        pytest.skip("the tensor-core kernel is FP32-mode only")
    # N_t = 1500 spans several observation chunks with a ragged tail; N_f = 9001 spans several tiles with a ragged tail
    w = make_config(2, dtype=dtype, n_t=1500, n_freq=9001)
    P_ref = oracle_full(oracle, w)
    P, best, info = gpu_full(lsp, w, kernel=kernel, fast_math=fast)
    assert_power_parity(P, P_ref, dtype, f"c2s/{kernel}/{dtype}/fast={fast}")
    assert_best_parity(best, P_ref, w, dtype, oracle)


@pytest.mark.parametrize("dtype,fast", [("f64", False), ("f32", False), ("f32", True)])
def test_config2_full_size_sampled(lsp, oracle, dtype, fast):
    """BASELINE config 2 at full size (N_t = 1e4, N_f = 1e6) in the bench launch configuration; the oracle
    checks a seeded sample of frequencies plus a window around the peak, and the bounds hold everywhere."""
    w = make_config(2, dtype=dtype)
    P, best, info = gpu_full(lsp, w, fast_math=fast)
    assert info["kernel"] == ("tensor" if dtype == "f32" else "factored")
    rng = np.random.default_rng(22)
    ks = np.unique(np.concatenate([rng.integers(0, w.n_freq, 600), np.arange(0, 64), np.arange(w.n_freq - 64, w.n_freq),
                                   np.clip(np.arange(-100, 101) + int(best[2][0]), 0, w.n_freq - 1)])).astype(np.int64)
    P_ref = oracle.periodogram(w.offsets, w.t, w.y, w.f_min, w.f_max, w.n_freq, k_list=ks)
    yy = w.y.astype(np.float64)
    half_sum = 0.5 * float(yy @ yy)
    pmax = max(P_ref.max(), P[0].max())
    assert np.max(np.abs(P[0, ks] - P_ref[0])) <= TOL[dtype] * pmax
    assert P.min() >= -TOL[dtype] * pmax and P.max() <= half_sum * (1 + TOL[dtype])
    # the GPU's global argmax is inside the window the oracle evaluated
    assert abs(P_ref[0].max() - best[1][0]) <= TOL[dtype] * pmax
    true_f = 1.0 / w.meta["true_period_days"]
    assert abs(1.0 / best[0][0] - true_f) < 5 * (w.f_max - w.f_min) / w.n_freq + 1.0 / 3650.0


# ---- config 3 shape: batch of short night-clustered objects, best period fused ----------------------------
@pytest.mark.parametrize("kernel,fast", [("factored", False), ("factored", True), ("direct", True),
                                         ("tensor", False), ("tensor", True)])
def test_config3_shape_best_only(lsp, oracle, kernel, fast):
    w = make_config(3, n_obj=24, n_freq=20_011)
    P_ref = oracle_full(oracle, w)
    best, info = gpu_best(lsp, w, kernel=kernel, fast_math=fast)
    assert_best_parity(best, P_ref, w, "f32", oracle, f"c3s/{kernel}")
    P, best2, _ = gpu_full(lsp, w, kernel=kernel, fast_math=fast)
    assert_power_parity(P, P_ref, "f32", f"c3s/{kernel}")
    # fused best-only and full+best agree bit for bit
    for a, b in zip(best, best2):
        assert np.array_equal(a, b, equal_nan=True)


def test_config3_full_size_sampled_objects(lsp, oracle):
    """BASELINE config 3 at full size (10,000 objects, N_f = 1e5), best-period output only; the oracle checks
    a seeded sample of whole objects (so best-period parity is testable)."""
    w = make_config(3)
    best, info = gpu_best(lsp, w, fast_math=True)
    assert info["kernel"] == "tensor" and info["n_split"] == 1
    rng = np.random.default_rng(33)
    pick = np.sort(rng.choice(w.n_obj, 12, replace=False))
    sub = w.take_objects(pick)
    P_ref = oracle_full(oracle, sub)
    assert_best_parity(tuple(x[pick] for x in best), P_ref, sub, "f32", oracle, "c3 full")
    assert np.all(best[2] >= 0) and np.all(best[2] < w.n_freq) and np.all(np.isfinite(best[0]))
    # peak at half the rotation period for most objects
    f_best = 1.0 / best[0].astype(np.float64)
    f_true = 2.0 / (w.meta["rotation_period_h"] / 24.0)
    assert np.mean(np.abs(f_best - f_true) < 0.01) > 0.6


# ---- config 4 shape: full periodograms to pinned host memory through the chunk ring -----------------------
def test_config4_shape_host_output_streams(lsp, oracle):
    import torch
    w = make_config(4, n_obj=37, n_freq=30_007)
    P_ref = oracle_full(oracle, w)
    off, t, y = to_device(w)
    host = torch.empty((w.n_obj, w.n_freq), dtype=torch.float32).pin_memory()
    host.fill_(float("nan"))
    # 5 objects per chunk -> 8 chunks over 3 streams / 4 slots, last chunk ragged
    with lsp.Plan(w.f_min, w.f_max, w.n_freq, "f32", fast_math=True, n_copy_streams=3,
                  chunk_bytes=5 * w.n_freq * 4) as plan:
        _, best = plan.periodogram_batched(off, t, y, host_out=host, best=True)
        info = plan.last_call_info()
        dev, best_dev = plan.periodogram_batched(off, t, y, best=True)
        torch.cuda.synchronize()
    assert info["chunks"] == 8
    P = host.numpy().astype(np.float64)
    assert_power_parity(P, P_ref, "f32", "c4s host")
    # same kernels; a chunk may be scheduled with a different observation split than the whole batch, so the
    # summation order (not the result) can differ
    assert np.max(np.abs(host.numpy() - dev.cpu().numpy())) <= 1e-5 * P_ref.max()
    assert_best_parity(tuple(x.cpu().numpy() for x in best), P_ref, w, "f32", oracle)
    # pageable destination: plain cudaMemcpyAsync (default) and the paper's staging scheme
    import os
    for mode in ("plain", "staged"):
        os.environ["LSP_PAGEABLE"] = mode
        try:
            pageable = torch.full((w.n_obj, w.n_freq), float("nan"), dtype=torch.float32)
            with lsp.Plan(w.f_min, w.f_max, w.n_freq, "f32", fast_math=True, chunk_bytes=1 << 20) as plan:
                plan.periodogram_batched(off, t, y, host_out=pageable)
        finally:
            os.environ.pop("LSP_PAGEABLE", None)
        assert np.max(np.abs(pageable.numpy() - host.numpy())) <= 1e-5 * P_ref.max(), mode


# ---- config 5 shape: large N_t / small N_f -> observation split path ----------------------------------------
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("kernel", ["factored", "direct", "tensor"])
def test_config5_split_path(lsp, oracle, dtype, kernel):
    if kernel == "tensor" and dtype == "f64":
        pytest.skip("the tensor-core kernel is FP32-mode only")
    w = make_config(5, dtype=dtype, n_t=16384, n_freq=6000, point=7)
    rng = np.random.default_rng(55)
    P, best, info = gpu_full(lsp, w, kernel=kernel, fast_math=(dtype == "f32"))
    assert info["n_split"] > 1, "this shape must take the split-N_t path"
    ks = np.unique(np.concatenate([rng.integers(0, w.n_freq, 400), [0, w.n_freq - 1],
                                   np.clip(np.arange(-30, 31) + int(best[2][0]), 0, w.n_freq - 1)])).astype(np.int64)
    P_ref = oracle.periodogram(w.offsets, w.t, w.y, w.f_min, w.f_max, w.n_freq, k_list=ks)
    pmax = P_ref.max()
    assert np.max(np.abs(P[0, ks] - P_ref[0])) <= TOL[dtype] * pmax
    assert abs(best[1][0] - pmax) <= TOL[dtype] * pmax


# ---- edge cases ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("kernel", ["direct", "factored", "tensor"])
def test_edge_empty_and_tiny_objects(lsp, oracle, dtype, kernel):
    if kernel == "tensor" and dtype == "f64":
        pytest.skip("the tensor-core kernel is FP32-mode only")
    rng = np.random.default_rng(9)
    lens = [0, 1, 2, 3, 17, 0, 130]
    off = np.zeros(len(lens) + 1, dtype=np.int64)
    off[1:] = np.cumsum(lens)
    t = np.concatenate([np.sort(rng.uniform(0, 30, n)) for n in lens])
    y = rng.normal(0, 1, t.size)
    np_t = np.float32 if dtype == "f32" else np.float64
    w = Workload("edge", off, t.astype(np_t), y.astype(np_t), 0.05, 3.0, 2500, dtype)
    P_ref = oracle_full(oracle, w)
    P, best, _ = gpu_full(lsp, w, kernel=kernel)
    assert np.all(np.isfinite(P))
    assert np.all(P[0] == 0) and np.all(P[5] == 0)
    # N_t = 1 and N_t = 2 hit the singular branch at isolated frequencies: finite + bounded only (reading a6)
    for o in (1, 2):
        yy = w.y[off[o]:off[o + 1]].astype(np.float64)
        slack = 2e-2 if dtype == "f32" else 1e-6   # near-singular frequencies amplify rounding (reading a6)
        assert P[o].min() >= 0 and P[o].max() <= 0.5 * (yy @ yy) * (1 + slack) + 1e-30
    keep = [3, 4, 6]
    assert_power_parity(P[keep], P_ref[keep], dtype, f"edge/{kernel}")
    assert best[2][0] == -1 and np.isnan(best[0][0]) and best[1][0] == 0
    assert best[2][5] == -1
    sub = w.take_objects(keep)
    assert_best_parity(tuple(x[keep] for x in best), P_ref[keep], sub, dtype, oracle)


@pytest.mark.parametrize("n_freq", [1, 255, 4096, 4097])
def test_edge_ragged_grid_sizes(lsp, oracle, n_freq):
    w = make_config(1, n_freq=n_freq, dtype="f32")
    P_ref = oracle_full(oracle, w)
    for kernel in ("direct", "factored", "tensor"):
        P, best, _ = gpu_full(lsp, w, kernel=kernel)
        assert_power_parity(P, P_ref, "f32", f"nf={n_freq}/{kernel}")
        assert_best_parity(best, P_ref, w, "f32", oracle)


def test_edge_zero_objects_and_errors(lsp):
    import torch
    with lsp.Plan(0.1, 2.0, 100, "f32") as plan:
        off = torch.zeros(1, dtype=torch.int64, device="cuda")
        t = torch.zeros(0, dtype=torch.float32, device="cuda")
        power, best = plan.periodogram_batched(off, t, t, best=True)
        assert power.shape == (0, 100) and best[0].numel() == 0
        bad = torch.tensor([0, 5, 3], dtype=torch.int64)
        with pytest.raises(lsp.LspError) as ei:
            plan.best_period(bad.cuda(), torch.zeros(5, device="cuda"), torch.zeros(5, device="cuda"), h_offsets=bad)
        assert ei.value.status == 1
    for kw in (dict(f_min=0.0), dict(f_min=-1.0), dict(f_max=0.05), dict(n_freq=0), dict(dtype="f64", fast_math=True)):
        args = dict(f_min=0.1, f_max=2.0, n_freq=10, dtype="f32")
        args.update(kw)
        with pytest.raises(lsp.LspError) as ei:
            lsp.Plan(**args)
        assert ei.value.status == 1


def test_normalize_and_center_options(lsp, oracle):
    w = make_config(3, n_obj=5, n_freq=5000)
    shifted = Workload(w.name, w.offsets, w.t, (w.y + np.float32(3.25)).astype(np.float32), w.f_min, w.f_max, w.n_freq, "f32")
    # center=1 on shifted data == plain call on data centred by numpy in FP64 (to FP32 tolerance)
    yc = shifted.y.astype(np.float64).copy()
    for o in range(w.n_obj):
        s = slice(w.offsets[o], w.offsets[o + 1])
        yc[s] -= yc[s].mean()
    P_ref = oracle.periodogram(w.offsets, w.t, yc, w.f_min, w.f_max, w.n_freq)
    P, _, _ = gpu_full(lsp, shifted, center=True, best=False)
    assert_power_parity(P, P_ref, "f32", "center")
    Pn, _, _ = gpu_full(lsp, shifted, center=True, normalize=True, best=False)
    for o in range(w.n_obj):
        s = slice(w.offsets[o], w.offsets[o + 1])
        ref = P_ref[o] / (0.5 * (yc[s] @ yc[s]))
        assert np.max(np.abs(Pn[o] - ref)) <= 1e-3 * ref.max()
        assert Pn[o].max() <= 1.0 + 1e-3


def test_deterministic_and_no_h_offsets(lsp):
    import torch
    w = make_config(3, n_obj=40, n_freq=8000)
    off, t, y = to_device(w)
    with lsp.Plan(w.f_min, w.f_max, w.n_freq, "f32", fast_math=True) as plan:
        a, ba = plan.periodogram_batched(off, t, y, best=True)                      # offsets read back by the library
        b, bb = plan.periodogram_batched(off, t, y, best=True, h_offsets=torch.from_numpy(w.offsets))
        torch.cuda.synchronize()
        assert torch.equal(a, b) and all(torch.equal(x, z) for x, z in zip(ba, bb))
    s = torch.cuda.Stream()
    with torch.cuda.stream(s), lsp.Plan(w.f_min, w.f_max, w.n_freq, "f32", fast_math=True) as plan:
        c, _ = plan.periodogram_batched(off, t, y, stream=s)
        s.synchronize()
        assert torch.equal(a, c)


# ---- generalised LSP (floating mean + errors) against oracle/gls_oracle.c ---------------------
def _with_errors(w: Workload, seed: int):
    """Seeded per-point errors for a workload (heteroscedastic, 0.5x-2x a base sigma) and an offset the floating mean must
    absorb; drawn in FP64, rounded once to the workload's dtype like t and y."""
    rng = np.random.Generator(np.random.PCG64(seed))
    base = 0.05 if w.name.startswith(("c3", "c4")) else 0.2
    sigma = (base * rng.uniform(0.5, 2.0, w.n_obs)).astype(w.t.dtype)
    y = (w.y.astype(np.float64) + 7.25).astype(w.t.dtype)
    return y, sigma


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("kernel", ["auto", "direct", "factored", "tensor"])
def test_generalized_batch_parity(lsp, oracle, dtype, kernel):
    import torch
    if kernel == "tensor" and dtype == "f64":
        pytest.skip("the tensor-core kernel is FP32-mode only")
    w = make_config(3, n_obj=5, n_freq=6000, dtype=dtype)
    y, sigma = _with_errors(w, 77)
    P_ref = oracle.periodogram_generalized(w.offsets, w.t, y, sigma, w.f_min, w.f_max, w.n_freq)
    off, t, _ = to_device(w)
    with lsp.Plan(w.f_min, w.f_max, w.n_freq, dtype, kernel=kernel) as plan:
        P, best = plan.periodogram_generalized(off, t, torch.from_numpy(y).cuda(), torch.from_numpy(sigma).cuda(), best=True,
                                               h_offsets=torch.from_numpy(w.offsets))
        info = plan.last_call_info()
        P = P.cpu().numpy().astype(np.float64)
        best = tuple(x.cpu().numpy() for x in best)
        # the plan's own grid is restored: a standard call afterwards still matches the standard oracle
        P_std, _ = plan.periodogram_batched(off, t, to_device(w)[2])
        assert_power_parity(P_std.cpu().numpy().astype(np.float64), oracle_full(oracle, w), dtype, "standard call after generalised")
    assert np.all(P >= -TOL[dtype]) and np.all(P <= 1.0 + TOL[dtype])
    assert_power_parity(P, P_ref, dtype, f"generalised {kernel}")
    assert_best_parity(best, P_ref, w, dtype, oracle, f"generalised {kernel}")


def test_generalized_single_object_and_edge_cases(lsp, oracle):
    import torch
    w = make_config(2, n_t=3000, n_freq=20000, dtype="f64")
    y, sigma = _with_errors(w, 5)
    # add an empty object and a single-point object: P = 0 rows
    off = np.array([0, w.n_obs, w.n_obs, w.n_obs + 1], dtype=np.int64)
    t = np.concatenate([w.t, w.t[:1]])
    y = np.concatenate([y, y[:1]])
    sigma = np.concatenate([sigma, sigma[:1]])
    P_ref = oracle.periodogram_generalized(off, t, y, sigma, w.f_min, w.f_max, w.n_freq)
    with lsp.Plan(w.f_min, w.f_max, w.n_freq, "f64") as plan:
        P, best = plan.periodogram_generalized(torch.from_numpy(off).cuda(), torch.from_numpy(t).cuda(), torch.from_numpy(y).cuda(),
                                               torch.from_numpy(sigma).cuda(), best=True)
        P = P.cpu().numpy()
        _, _, idx = (x.cpu().numpy() for x in best)
    assert np.max(np.abs(P[0] - P_ref[0])) <= TOL["f64"] * P_ref[0].max()
    assert np.all(P[1] == 0.0) and np.all(P[2] == 0.0) and idx[1] == -1
    assert idx[0] == int(np.argmax(P_ref[0]))


# ---- full-size config 4 and config 5 corners, in the launch configurations bench.py times -----------------------
def test_config4_full_size_sampled(lsp, oracle):
    """BASELINE config 4 at full size (2,000 objects, N_f = 5e5, 4.0 GB of periodograms to pinned host over the copy streams with
    the library's default chunking); the oracle checks sampled (object, frequency) values and whole-row properties."""
    import torch
    w = make_config(4)
    off, t, y = to_device(w)
    host = torch.empty((w.n_obj, w.n_freq), dtype=torch.float32).pin_memory()
    with lsp.Plan(w.f_min, w.f_max, w.n_freq, "f32") as plan:
        plan.periodogram_batched(off, t, y, host_out=host, h_offsets=torch.from_numpy(w.offsets))
        info = plan.last_call_info()
    assert info["kernel"] == "tensor" and info["chunks"] == -(-w.n_obj // ((64 << 20) // (w.n_freq * 4)))
    P = host.numpy()
    rng = np.random.default_rng(44)
    pick = np.sort(rng.choice(w.n_obj, 6, replace=False))
    pick = np.unique(np.concatenate([pick, [0, w.n_obj - 1]]))          # first and last chunk too
    ks = np.unique(np.concatenate([rng.integers(0, w.n_freq, 400), [0, 1, w.n_freq - 2, w.n_freq - 1]])).astype(np.int64)
    sub = w.take_objects(pick)
    P_ref = oracle.periodogram(sub.offsets, sub.t, sub.y, w.f_min, w.f_max, w.n_freq, k_list=ks)
    for i, o in enumerate(pick):
        row = P[o].astype(np.float64)
        yy = sub.y[sub.offsets[i]:sub.offsets[i + 1]].astype(np.float64)
        pmax = max(P_ref[i].max(), float(row.max()))
        assert np.max(np.abs(row[ks] - P_ref[i])) <= TOL["f32"] * pmax, f"object {o}"
        assert row.min() >= -TOL["f32"] * pmax and row.max() <= 0.5 * float(yy @ yy) * (1 + TOL["f32"])
    assert np.isfinite(P[::97]).all()


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("n_t,n_freq,point", [(1024, 100_000, 0), (65536, 4_000_000, 11)])
def test_config5_corner_points_sampled(lsp, oracle, dtype, n_t, n_freq, point):
    """The smallest and the largest point of BASELINE config 5's sweep at full size; sampled frequencies + the peak window."""
    w = make_config(5, dtype=dtype, n_t=n_t, n_freq=n_freq, point=point)
    P, best, info = gpu_full(lsp, w)
    rng = np.random.default_rng(5 + point)
    ks = np.unique(np.concatenate([rng.integers(0, n_freq, 96 if n_t > 10000 else 600), [0, n_freq - 1],
                                   np.clip(np.arange(-8, 9) + int(best[2][0]), 0, n_freq - 1)])).astype(np.int64)
    P_ref = oracle.periodogram(w.offsets, w.t, w.y, w.f_min, w.f_max, w.n_freq, k_list=ks)
    pmax = max(P_ref.max(), P[0].max())
    assert np.max(np.abs(P[0, ks] - P_ref[0])) <= TOL[dtype] * pmax
    assert abs(P_ref[0].max() - best[1][0]) <= TOL[dtype] * pmax
    yy = w.y.astype(np.float64)
    assert P.min() >= -TOL[dtype] * pmax and P.max() <= 0.5 * float(yy @ yy) * (1 + TOL[dtype])


# ---- randomized shapes: tile geometry, ring wrap-around and generator-group parity corner cases ------------------
@pytest.mark.parametrize("seed", range(8))
def test_random_shapes_all_kernels(lsp, oracle, seed):
    """Seeded random CSR batches whose object lengths straddle the 16-observation stage size (0, 1, 15, 16, 17, 33, ...) and
    grids whose sizes hit different tile widths (NL), exact multiples of a tile and ragged last tiles; every kernel
    against the oracle, full periodogram + fused best period."""
    rng = np.random.Generator(np.random.PCG64(9000 + seed))
    n_obj = int(rng.integers(1, 10))
    lens = rng.choice([0, 1, 2, 15, 16, 17, 31, 32, 33, 47, 100, 257], size=n_obj)
    if lens.sum() == 0:
        lens[0] = 16
    n_freq = int(rng.choice([1024, 1100, 2048, 4096, 5000, 8192, 16384, 16385, 30000]))
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    t = np.concatenate([np.sort(rng.uniform(0.0, 400.0, n)) for n in lens]) if lens.sum() else np.zeros(0)
    y = rng.normal(0.0, 1.0, t.size) + np.sin(2 * np.pi * 1.37 * t)
    f_min, f_max = 0.03, float(rng.uniform(2.0, 9.0))
    for dtype, kernels in (("f32", ("tensor", "factored", "direct")), ("f64", ("factored",))):
        w = Workload(f"rand{seed}", off, t.astype(np.float32 if dtype == "f32" else np.float64),
                     y.astype(np.float32 if dtype == "f32" else np.float64), f_min, f_max, n_freq, dtype=dtype)
        P_ref = oracle_full(oracle, w)
        for kernel in kernels:
            P, best, info = gpu_full(lsp, w, kernel=kernel)
            for o in range(n_obj):
                if lens[o] == 0:
                    assert np.all(P[o] == 0.0)
                elif lens[o] >= 3:       # N_t <= 2 sits on the vanishing-denominator branch (reading a6): finite and bounded only
                    pmax = P_ref[o].max()
                    assert np.max(np.abs(P[o] - P_ref[o])) <= TOL[dtype] * pmax, f"seed {seed} {dtype} {kernel} object {o} (N_t={lens[o]}, N_f={n_freq})"
                else:
                    yy = w.y[off[o]:off[o + 1]].astype(np.float64)
                    # near sin w(t2 - t1) = 0 the 2 x 2 system is ill-conditioned: bounded, not tolerance-accurate
                    assert np.all(np.isfinite(P[o])) and P[o].min() >= -1e-3 * float(yy @ yy) and P[o].max() <= float(yy @ yy) + 1e-30
            big = [o for o in range(n_obj) if lens[o] >= 3]
            if big:
                sub = w.take_objects(big)
                assert_best_parity(tuple(x[big] for x in best), P_ref[big], sub, dtype, oracle, f"seed {seed} {kernel}")
