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


def plan_kw(kw):
    """tensor_roles in the tests: 1 / 2 = that warp-role shape on single CTAs (tensor_pair = 1: never pair), 3 = CTA pairs
    forced (tensor_pair = 2); 0 or absent = the scheduler's own choice."""
    kw = dict(kw)
    roles = kw.pop("tensor_roles", 0)
    if roles in (1, 2):
        kw.update(tensor_roles=roles, tensor_pair=1)
    elif roles == 3:
        kw.update(tensor_pair=2)
    return kw


def gpu_full(lsp, w: Workload, *, kernel="auto", fast_math=False, best=True, **kw):
    kw = plan_kw(kw)
    off, t, y = to_device(w)
    with lsp.Plan(w.f_min, w.f_max, w.n_freq, w.dtype, kernel=kernel, fast_math=fast_math, **kw) as plan:
        power, b = plan.periodogram_batched(off, t, y, best=best, h_offsets=__import__("torch").from_numpy(w.offsets))
        info = plan.last_call_info()
        P = power.cpu().numpy().astype(np.float64)
        bb = None if b is None else tuple(x.cpu().numpy() for x in b)
    return P, bb, info


def gpu_best(lsp, w: Workload, *, kernel="auto", fast_math=False, **kw):
    kw = plan_kw(kw)
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


# Kernel variants every shape test runs, (kernel, shape, tensor_products): the tensor kernel in ALL THREE launch shapes (1 =
# short-item warp roles, 2 = long-item warp roles, 3 = long-item roles on CTA pairs / cta_group::2; see plan_kw) and BOTH accurate
# precision modes (lsp_config.tensor_products: 3 = the default, 2 = the opt-in), so each template instantiation the scheduler can reach gets
# full-grid element-wise checks.  Shape 3 needs a grid of at least two tiles (> 14,336 frequencies): the shape tests give the
# pair variants a larger grid where their own is a single tile.
KERNEL_VARIANTS = [("direct", 0, 0), ("factored", 0, 0), ("tensor", 1, 2), ("tensor", 2, 2), ("tensor", 1, 3), ("tensor", 2, 3),
                   ("tensor", 3, 2), ("tensor", 3, 3)]
MIN_NT_TWO_PRODUCTS = 32      # a call holding a shorter object runs with three products (lsp.h, lsp_last_call_info)


def variant_id(v):
    return v[0] if v[1] == 0 else f"tensor-shape{v[1]}-products{v[2]}"


def assert_two_point_pin(P_row, t2, y2, w: Workload, dtype, what=""):
    """Pin p7: any two points are fit exactly, so P(f) = (y1^2 + y2^2)/2 wherever sin w(t2 - t1) != 0.
    Checked at the frequencies with |sin| > 0.1, with the tolerance scaled by the 2 x 2 system's conditioning 1/sin^2."""
    f = w.f_min + np.arange(w.n_freq) * (w.f_max - w.f_min) / w.n_freq
    sn = np.sin(2 * np.pi * f * (float(t2[1]) - float(t2[0])))
    ok = np.abs(sn) > 0.1
    assert ok.sum() > 0.5 * w.n_freq
    want = 0.5 * float(np.dot(y2.astype(np.float64), y2.astype(np.float64)))
    err = np.abs(P_row[ok] - want) * sn[ok] ** 2
    assert err.max() <= TOL[dtype] * want, f"{what}: N_t = 2 closed form: {err.max():.3e} > {TOL[dtype]:.0e} * {want:.3e}"


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
@pytest.mark.parametrize("variant", KERNEL_VARIANTS, ids=variant_id)
def test_config2_shape_small(lsp, oracle, dtype, fast, variant):
    kernel, roles, products = variant
    if kernel == "tensor" and (dtype == "f64" or (fast and products == 3)):
        pytest.skip("the tensor-core kernel is FP32-mode only; fast_math has one product")
    # N_t = 1500 spans several observation chunks with a ragged tail; N_f = 9001 spans several tiles with a ragged tail
    # (CTA pairs: 30,011 = three tensor tiles, i.e. one full pair and one pair with a phantom second tile, ragged)
    w = make_config(2, dtype=dtype, n_t=1500, n_freq=30_011 if roles == 3 else 9001)
    P_ref = oracle_full(oracle, w)
    P, best, info = gpu_full(lsp, w, kernel=kernel, fast_math=fast, tensor_roles=roles, tensor_products=products)
    assert info["tensor_shape"] == roles and info["tensor_products"] == (0 if kernel != "tensor" else 1 if fast else products)
    assert_power_parity(P, P_ref, dtype, f"c2s/{kernel}/{dtype}/fast={fast}")
    assert_best_parity(best, P_ref, w, dtype, oracle)


@pytest.mark.parametrize("pair", [1, 0], ids=["single-cta", "auto"])
@pytest.mark.parametrize("n_freq,fast", [(100_000, False), (99_999, False), (100_002, True)])
def test_long_single_object_full_grid_long_item_shape(lsp, oracle, n_freq, fast, pair):
    """The long-item role shape through the scheduler's OWN choice (no override): one object of N_t = 20,000 on a grid of
    seven tiles is split by observations into items of >= 48 stages (config 2's launch configuration on a smaller grid);
    the last split of every tile to arrive finishes the tile in-kernel.  Full grid against the oracle, N_f % 4 in {0, 3, 2}."""
    w = make_config(2, dtype="f32", n_t=20_000, n_freq=n_freq)
    P_ref = oracle_full(oracle, w)
    P, best, info = gpu_full(lsp, w, fast_math=fast, tensor_pair=pair)
    # left to itself the scheduler puts these long items on CTA pairs (shape 3); tensor_pair = 1 keeps single CTAs (shape 2)
    assert info["kernel"] == "tensor" and info["tensor_shape"] == (2 if pair == 1 else 3) and info["n_split"] > 1
    assert_power_parity(P, P_ref, "f32", f"long single nf={n_freq}")
    assert_best_parity(best, P_ref, w, "f32", oracle)


@pytest.mark.parametrize("pair", [1, 0], ids=["single-cta", "auto"])
def test_long_items_unsplit_batch_long_item_shape(lsp, oracle, pair):
    """The long-item shape's NON-split epilogue (power + vector stores + fused argmax in the kernel) by the scheduler's own
    choice: 1,300 objects of N_t = 1,024 on a 16,384-point grid give >= 8 x 148 items of 64 stages each, split 1.  Full
    periodogram + best period; the oracle checks a seeded sample of 16 WHOLE objects element by element."""
    rng = np.random.Generator(np.random.PCG64(4242))
    n_obj, n_t, n_freq = 1300, 1024, 16384
    off = np.arange(n_obj + 1, dtype=np.int64) * n_t
    t = np.sort(rng.uniform(0.0, 3650.0, (n_obj, n_t)), axis=1)
    per = rng.uniform(0.1, 2.0, n_obj)
    y = 0.5 * np.sin(2 * np.pi * t / per[:, None] + rng.uniform(0, 2 * np.pi, (n_obj, 1))) + rng.normal(0, 0.2, (n_obj, n_t))
    y -= y.mean(axis=1, keepdims=True)
    w = Workload("long-batch", off, t.reshape(-1).astype(np.float32), y.reshape(-1).astype(np.float32), 0.05, 12.0, n_freq, "f32")
    P, best, info = gpu_full(lsp, w, tensor_pair=pair)
    assert info["kernel"] == "tensor" and info["tensor_shape"] == (2 if pair == 1 else 3) and info["n_split"] == 1
    pick = np.sort(rng.choice(n_obj, 16, replace=False))
    pick[0], pick[-1] = 0, n_obj - 1
    sub = w.take_objects(pick)
    P_ref = oracle_full(oracle, sub)
    assert_power_parity(P[pick], P_ref, "f32", "long batch")
    assert_best_parity(tuple(x[pick] for x in best), P_ref, sub, "f32", oracle, "long batch")
    best_only, _ = gpu_best(lsp, w, tensor_pair=pair)
    for a, b in zip(best, best_only):
        assert np.array_equal(a, b, equal_nan=True)


_C2_ORACLE = {}


def c2_full_oracle(oracle, dtype):
    """The oracle on the FULL config-2 grid (1e10 pairs: about half a minute on 16 host cores), once per input precision."""
    if dtype not in _C2_ORACLE:
        w = make_config(2, dtype=dtype)
        _C2_ORACLE[dtype] = oracle_full(oracle, w)
    return _C2_ORACLE[dtype]


@pytest.mark.parametrize("dtype,fast,products", [("f64", False, 0), ("f32", False, 0), ("f32", False, 2), ("f32", True, 0)])
def test_config2_full_size_full_grid(lsp, oracle, dtype, fast, products):
    """BASELINE config 2 at full size (N_t = 1e4, N_f = 1e6) in the bench launch configuration, EVERY grid frequency against
    the oracle (SURVEY.md 8(d) "Oracle timing": full grid for C1 and C2), plus best period and the bounds of pin p3."""
    w = make_config(2, dtype=dtype)
    P_ref = c2_full_oracle(oracle, dtype)
    P, best, info = gpu_full(lsp, w, fast_math=fast, tensor_products=products)
    assert info["kernel"] == ("tensor" if dtype == "f32" else "factored")
    if dtype == "f32":
        assert info["tensor_shape"] == 3           # long-item roles on CTA pairs: the launch shape bench.py times on this config
        assert info["tensor_products"] == (1 if fast else products or 3)     # default = three products, as bench.py times it
    assert_power_parity(P, P_ref, dtype, f"c2 full {dtype} fast={fast}")
    assert_best_parity(best, P_ref, w, dtype, oracle, "c2 full")
    yy = w.y.astype(np.float64)
    pmax = P_ref.max()
    assert P.min() >= -TOL[dtype] * pmax and P.max() <= 0.5 * float(yy @ yy) * (1 + TOL[dtype])
    true_f = 1.0 / w.meta["true_period_days"]
    assert abs(1.0 / best[0][0] - true_f) < 5 * (w.f_max - w.f_min) / w.n_freq + 1.0 / 3650.0


# ---- config 3 shape: batch of short night-clustered objects, best period fused ----------------------------
@pytest.mark.parametrize("kernel,fast,roles,products", [("factored", False, 0, 0), ("factored", True, 0, 0), ("direct", True, 0, 0),
                                                        ("tensor", False, 1, 2), ("tensor", True, 1, 0), ("tensor", False, 2, 2),
                                                        ("tensor", True, 2, 0), ("tensor", False, 1, 3), ("tensor", False, 2, 3),
                                                        ("tensor", False, 3, 2), ("tensor", False, 3, 3), ("tensor", True, 3, 0)])
def test_config3_shape_best_only(lsp, oracle, kernel, fast, roles, products):
    w = make_config(3, n_obj=24, n_freq=20_011)
    P_ref = oracle_full(oracle, w)
    best, info = gpu_best(lsp, w, kernel=kernel, fast_math=fast, tensor_roles=roles, tensor_products=products)
    assert info["tensor_shape"] == roles and info["tensor_products"] == (0 if kernel != "tensor" else 1 if fast else products)
    assert_best_parity(best, P_ref, w, "f32", oracle, f"c3s/{kernel}")
    P, best2, _ = gpu_full(lsp, w, kernel=kernel, fast_math=fast, tensor_roles=roles, tensor_products=products)
    assert_power_parity(P, P_ref, "f32", f"c3s/{kernel}")
    # fused best-only and full+best agree bit for bit
    for a, b in zip(best, best2):
        assert np.array_equal(a, b, equal_nan=True)


@pytest.mark.parametrize("fast", [False, True])
def test_config3_full_size_sampled_objects(lsp, oracle, fast):
    """BASELINE config 3 at full size (10,000 objects, N_f = 1e5), best-period output only, in the accurate mode bench.py times
    (and in fast_math); the oracle checks a seeded sample of 64 WHOLE objects (so best-period parity is testable)."""
    w = make_config(3)
    best, info = gpu_best(lsp, w, fast_math=fast)
    assert info["kernel"] == "tensor" and info["n_split"] == 1 and info["tensor_shape"] == 1
    rng = np.random.default_rng(33)
    pick = np.sort(rng.choice(w.n_obj, 64, replace=False))
    pick[0], pick[-1] = 0, w.n_obj - 1
    sub = w.take_objects(pick)
    P_ref = oracle_full(oracle, sub)
    assert_best_parity(tuple(x[pick] for x in best), P_ref, sub, "f32", oracle, "c3 full")
    assert np.all(best[2] >= 0) and np.all(best[2] < w.n_freq) and np.all(np.isfinite(best[0]))
    # peak at half the rotation period for most objects
    f_best = 1.0 / best[0].astype(np.float64)
    f_true = 2.0 / (w.meta["rotation_period_h"] / 24.0)
    assert np.mean(np.abs(f_best - f_true) < 0.01) > 0.6


def test_tensor_products_error_levels_on_noise_only_objects(lsp, oracle):
    """The two precision modes of the accurate tensor path on the data that is hardest for them: pure-noise objects (no signal
    to lift max P above the noise floor), N_t from the 32-observation floor of the two-product mode up to 400.  Two products
    (generated operand = one FP16) must stay within half the tolerance, three products within a twentieth; a launch that holds
    a shorter object must fall back to three products by itself."""
    rng = np.random.Generator(np.random.PCG64(777))
    lens = np.concatenate([[32, 33, 40, 48, 64], rng.integers(32, 401, 59)])
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    t = np.concatenate([np.sort(rng.uniform(0.0, 365.0, n)) for n in lens]).astype(np.float32)
    y = np.concatenate([(lambda v: v - v.mean())(rng.normal(0.0, 1.0, n)) for n in lens]).astype(np.float32)
    w = Workload("noise", off, t, y, 0.02, 12.0, 60_000, "f32")
    P_ref = oracle_full(oracle, w)
    worst = {}
    for products in (2, 3):
        P, best, info = gpu_full(lsp, w, kernel="tensor", tensor_products=products)
        assert info["tensor_products"] == products
        worst[products] = max(np.max(np.abs(P[o] - P_ref[o])) / P_ref[o].max() for o in range(w.n_obj))
        assert_best_parity(best, P_ref, w, "f32", oracle, f"noise/products={products}")
    assert worst[2] <= 0.5 * TOL["f32"] and worst[3] <= 0.05 * TOL["f32"], worst
    short = w.take_objects(np.arange(8))
    short.offsets[-1] = short.offsets[-2] + 12    # last object: 12 observations
    short = Workload("noise-short", short.offsets, short.t[:short.offsets[-1]], short.y[:short.offsets[-1]], w.f_min, w.f_max, 9000, "f32")
    P, _, info = gpu_full(lsp, short, kernel="tensor", tensor_products=2)
    assert info["tensor_products"] == 3
    assert_power_parity(P, oracle_full(oracle, short), "f32", "noise-short")


# ---- ill-conditioned cadences: a few short nights (PAPER.md:L238-246 ZTF/LSST-like records; reading a6's aliasing zone) ---------
FEW_NIGHT_CADENCES = [(6, 0.05), (12, 0.05), (30, 0.1), (3650, 0.3)]      # (nights, nightly window in days)
DEFAULT_VARIANTS = [("direct", 0), ("factored", 0), ("tensor", 1), ("tensor", 2), ("tensor", 3)]      # (kernel, tensor shape)


@pytest.mark.parametrize("signal", [False, True], ids=["noise-only", "signal"])
@pytest.mark.parametrize("cadence", FEW_NIGHT_CADENCES, ids=lambda c: f"{c[0]}nights-{c[1]}d")
def test_few_night_cadences_at_library_defaults(lsp, oracle, cadence, signal):
    """Objects of 32-60 observations taken on a handful of nights inside a short nightly window: the 2 x 2 system of step 5 is
    badly conditioned over wide bands around every integer cycles/day, so rounding of the contraction's operands is amplified.
    Every kernel family at LIBRARY DEFAULTS (the tensor path in all three launch shapes: three FP16 products) must hold the FP32
    tolerance element by element on the whole 100,000-point grid of config 3, noise-only and with a signal.  The two-product
    opt-in is held to the tolerance only on config 3's own cadence (3,650 nights x 0.3 d) and must at least stay finite and
    bounded elsewhere (DESIGN.md 6.3 tabulates what it reaches)."""
    from workloads import few_night_batch
    n_nights, window = cadence
    w = few_night_batch(n_nights, window, signal=signal)
    assert w.n_obj == 30 and 32 <= np.diff(w.offsets).min() and np.diff(w.offsets).max() <= 60
    P_ref = oracle_full(oracle, w)
    for kernel, roles in DEFAULT_VARIANTS:
        P, best, info = gpu_full(lsp, w, kernel=kernel, tensor_roles=roles)
        assert info["tensor_shape"] == roles and info["tensor_products"] == (3 if kernel == "tensor" else 0)
        assert_power_parity(P, P_ref, "f32", f"few-night {cadence} signal={signal} {kernel}/{roles}")
        assert_best_parity(best, P_ref, w, "f32", oracle, f"few-night {cadence} {kernel}/{roles}")
    P, best, info = gpu_full(lsp, w, kernel="tensor", tensor_products=2)
    assert info["tensor_products"] == 2
    if cadence == (3650, 0.3):
        assert_power_parity(P, P_ref, "f32", f"few-night {cadence} two products")
    else:
        yy = np.array([float(w.y[a:b].astype(np.float64) @ w.y[a:b].astype(np.float64)) for a, b in zip(w.offsets[:-1], w.offsets[1:])])
        assert np.all(np.isfinite(P)) and np.all(P.max(axis=1) <= 0.5 * yy * 1.05) and np.all(P.min(axis=1) >= -0.05 * 0.5 * yy)


@pytest.mark.parametrize("products", [0, 2])
def test_mixed_length_batch_cut_and_chunked_equal_whole(lsp, products):
    """A batch that mixes objects shorter than the two-product floor (N_t < 32) with longer ones: the product count is decided per
    CALL, so table-budget sub-ranges and the chunks of the host-output path (one schedule each) must give the bits of the uncut
    device call, at the default and with the two-product opt-in (which this batch turns into three products everywhere)."""
    import torch
    rng = np.random.Generator(np.random.PCG64(4242))
    lens = np.concatenate([[12, 40, 200], rng.integers(33, 300, 40), [7, 31, 32, 150]])
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    t = np.concatenate([np.sort(rng.integers(0, 3650, n) + rng.uniform(0.0, 0.3, n)) for n in lens]).astype(np.float32)
    y = np.concatenate([(lambda v: v - v.mean())(rng.normal(0.0, 1.0, n) + np.sin(2 * np.pi * 3.1 * rng.uniform(0, 1) * np.arange(n)))
                        for n in lens]).astype(np.float32)
    w = Workload("mixed", off, t, y, 0.12, 24.0, 20_000, "f32")
    d_off, d_t, d_y = to_device(w)
    h_off = torch.from_numpy(w.offsets)
    with lsp.Plan(w.f_min, w.f_max, w.n_freq, "f32", kernel="tensor", tensor_products=products) as plan:
        ref, bref = plan.periodogram_batched(d_off, d_t, d_y, best=True, h_offsets=h_off)
        assert plan.last_call_info()["tensor_products"] == 3
        n_ref = plan.last_call_info()["launches"]
    for h in (h_off, None):
        with lsp.Plan(w.f_min, w.f_max, w.n_freq, "f32", kernel="tensor", tensor_products=products, table_budget_bytes=1 << 20,
                      chunk_bytes=6 * w.n_freq * 4, n_copy_streams=2) as plan:
            cut, bcut = plan.periodogram_batched(d_off, d_t, d_y, best=True, h_offsets=h)
            assert plan.last_call_info()["launches"] > n_ref and plan.last_call_info()["tensor_products"] == 3
            host = torch.full((w.n_obj, w.n_freq), float("nan"), dtype=torch.float32).pin_memory()
            plan.periodogram_batched(d_off, d_t, d_y, host_out=host, h_offsets=h)     # 8 chunks of 6 objects, the last one ragged
            assert plan.last_call_info()["chunks"] == 8 and plan.last_call_info()["tensor_products"] == 3
        assert torch.equal(ref, cut) and all(torch.equal(a, b) for a, b in zip(bref, bcut))
        assert torch.equal(ref.cpu(), host)


# ---- the end-to-end entry point: lsp_periodogram_batched_host (PAPER.md:L85-91 call shape; the call bench.py's e2e goes through) ---
@pytest.mark.parametrize("pinned", [True, False], ids=["pinned", "pageable"])
@pytest.mark.parametrize("dtype,kernel", [("f32", "auto"), ("f32", "factored"), ("f64", "auto")])
def test_batched_host_entry_point_against_the_oracle(lsp, oracle, dtype, kernel, pinned):
    """Inputs and outputs on the HOST (pinned or pageable): H2D, kernels and D2H inside the call.  Full periodogram + best period
    in several chunks (5 objects per chunk, ragged last one), then best-only (no periodogram anywhere): against the oracle at the
    tolerances, and bit for bit against the device-resident calls on the same plan."""
    import torch
    w = make_config(3, n_obj=23, n_freq=12_007, dtype=dtype)
    P_ref = oracle_full(oracle, w)
    tdt = torch.float32 if dtype == "f32" else torch.float64
    pin = (lambda x: x.pin_memory()) if pinned else (lambda x: x)
    h_off = torch.from_numpy(w.offsets)
    h_t, h_y = pin(torch.from_numpy(w.t)), pin(torch.from_numpy(w.y))
    host = pin(torch.full((w.n_obj, w.n_freq), float("nan"), dtype=tdt))
    hb = tuple(pin(torch.empty(w.n_obj, dtype=d)) for d in (tdt, tdt, torch.int64))
    hb2 = tuple(pin(torch.empty(w.n_obj, dtype=d)) for d in (tdt, tdt, torch.int64))
    with lsp.Plan(w.f_min, w.f_max, w.n_freq, dtype, kernel=kernel, n_copy_streams=2, chunk_bytes=5 * w.n_freq * host.element_size()) as plan:
        plan.periodogram_batched_host(h_off, h_t, h_y, host_out=host, best_out=hb)
        info = plan.last_call_info()
        plan.periodogram_batched_host(h_off, h_t, h_y, best_out=hb2)                  # best period only
        info2 = plan.last_call_info()
        dev, db = plan.periodogram_batched(h_off.cuda(), h_t.cuda(), h_y.cuda(), best=True, h_offsets=h_off)
        torch.cuda.synchronize()
    assert info["chunks"] == 5 and info2["chunks"] == 0
    assert_power_parity(host.numpy().astype(np.float64), P_ref, dtype, f"batched_host {dtype}/{kernel}")
    assert_best_parity(tuple(x.numpy() for x in hb), P_ref, w, dtype, oracle, "batched_host full+best")
    assert_best_parity(tuple(x.numpy() for x in hb2), P_ref, w, dtype, oracle, "batched_host best-only")
    if info["kernel"] == "tensor":
        # the tensor path's schedule does not depend on how many objects a launch holds: chunked, best-only and device-resident
        # calls give the same bits
        assert np.array_equal(host.numpy(), dev.cpu().numpy())
        for a, b, c in zip(hb, hb2, db):
            assert np.array_equal(a.numpy(), b.numpy(), equal_nan=True) and np.array_equal(a.numpy(), c.cpu().numpy(), equal_nan=True)
    else:
        # FMA-pipe kernels: a 5-object chunk is scheduled for its own size and may split the observations differently from the
        # 23-object launch, i.e. the same sums in another order -- equal to rounding, far inside the tolerance
        pmax = P_ref.max(axis=1, keepdims=True)
        assert np.max(np.abs(host.numpy().astype(np.float64) - dev.cpu().numpy().astype(np.float64)) / pmax) <= 1e-2 * TOL[dtype]
        assert_best_parity(tuple(x.cpu().numpy() for x in db), P_ref, w, dtype, oracle, "device best")


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
    # the same through CTA pairs (three tiles: a phantom fourth), accurate mode, chunks of 7 objects
    host2 = torch.full((w.n_obj, w.n_freq), float("nan"), dtype=torch.float32).pin_memory()
    with lsp.Plan(w.f_min, w.f_max, w.n_freq, "f32", tensor_pair=2, n_copy_streams=2, chunk_bytes=7 * w.n_freq * 4) as plan:
        _, best2 = plan.periodogram_batched(off, t, y, host_out=host2, best=True)
        info2 = plan.last_call_info()
        torch.cuda.synchronize()
    assert info2["tensor_shape"] == 3 and info2["chunks"] == 6
    assert_power_parity(host2.numpy().astype(np.float64), P_ref, "f32", "c4s host pairs")
    assert_best_parity(tuple(x.cpu().numpy() for x in best2), P_ref, w, "f32", oracle)
    # pageable destination: plain cudaMemcpyAsync (default) and the paper's staging scheme (LSP_FLAG_PAGEABLE_STAGED)
    for staged in (False, True):
        pageable = torch.full((w.n_obj, w.n_freq), float("nan"), dtype=torch.float32)
        with lsp.Plan(w.f_min, w.f_max, w.n_freq, "f32", fast_math=True, chunk_bytes=1 << 20, pageable_staged=staged) as plan:
            plan.periodogram_batched(off, t, y, host_out=pageable)
        assert np.max(np.abs(pageable.numpy() - host.numpy())) <= 1e-5 * P_ref.max(), staged


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
@pytest.mark.parametrize("variant", KERNEL_VARIANTS, ids=variant_id)
def test_edge_empty_and_tiny_objects(lsp, oracle, dtype, variant):
    kernel, roles, products = variant
    if kernel == "tensor" and dtype == "f64":
        pytest.skip("the tensor-core kernel is FP32-mode only")
    rng = np.random.default_rng(9)
    lens = [0, 1, 2, 3, 17, 0, 130]
    off = np.zeros(len(lens) + 1, dtype=np.int64)
    off[1:] = np.cumsum(lens)
    t = np.concatenate([np.sort(rng.uniform(0, 30, n)) for n in lens])
    y = rng.normal(0, 1, t.size)
    np_t = np.float32 if dtype == "f32" else np.float64
    w = Workload("edge", off, t.astype(np_t), y.astype(np_t), 0.05, 3.0, 20_000 if roles == 3 else 2500, dtype)
    P_ref = oracle_full(oracle, w)
    P, best, info = gpu_full(lsp, w, kernel=kernel, tensor_roles=roles, tensor_products=products)
    if kernel == "tensor":       # objects of a few observations: the launch runs with three products whatever the plan says
        assert info["tensor_products"] == 3
    assert np.all(np.isfinite(P))
    assert np.all(P[0] == 0) and np.all(P[5] == 0)
    # N_t = 1 and N_t = 2 hit the singular branch at isolated frequencies: there, finite + bounded only (reading a6) ...
    f_grid = w.f_min + np.arange(w.n_freq) * ((w.f_max - w.f_min) / w.n_freq)
    for o in (1, 2):
        yy = w.y[off[o]:off[o + 1]].astype(np.float64)
        # N_t = 1: P = y^2 / 2 at every frequency.  N_t = 2: the 2 x 2 system degenerates where sin w(t2 - t1) = 0 and rounding is
        # amplified by 1/sin^2 near those points (reading a6): away from them (|sin| >= 0.02, whatever the grid density) the power
        # is held to its exact bound (1/2) sum y^2 with the same small slack for every variant; at them, finite and capped only
        slack = 2e-2 if dtype == "f32" else 1e-6
        ok = np.ones(w.n_freq, dtype=bool)
        if o == 2:
            tt = w.t[off[o]:off[o + 1]].astype(np.float64)
            ok = np.abs(np.sin(2.0 * np.pi * f_grid * (tt[1] - tt[0]))) >= 0.02
            assert ok.sum() > 0.9 * w.n_freq
        assert P[o].min() >= 0 and P[o][ok].max() <= 0.5 * (yy @ yy) * (1 + slack) + 1e-30
        assert P[o].max() <= 1.2 * (yy @ yy) + 1e-30
    # ... and away from them N_t = 2 has a closed form (pin p7)
    assert_two_point_pin(P[2], w.t[off[2]:off[3]], w.y[off[2]:off[3]], w, dtype, f"edge/{kernel}")
    keep = [3, 4, 6]
    assert_power_parity(P[keep], P_ref[keep], dtype, f"edge/{kernel}")
    assert best[2][0] == -1 and np.isnan(best[0][0]) and best[1][0] == 0
    assert best[2][5] == -1
    sub = w.take_objects(keep)
    assert_best_parity(tuple(x[keep] for x in best), P_ref[keep], sub, dtype, oracle)


@pytest.mark.parametrize("n_freq", [1, 255, 4096, 4097, 28_672, 28_673, 43_009])
def test_edge_ragged_grid_sizes(lsp, oracle, n_freq):
    """Grid sizes around the tile sizes: one point, a ragged single tile, exact tiles, one over; for the CTA-pair shape exactly
    two tiles of 14,336, one over (three tiles: a phantom fourth), and three full tiles + 1."""
    w = make_config(1, n_freq=n_freq, dtype="f32")
    P_ref = oracle_full(oracle, w)
    for kernel, roles, products in KERNEL_VARIANTS:
        if (roles == 3) != (n_freq > 14_336):
            continue
        P, best, info = gpu_full(lsp, w, kernel=kernel, tensor_roles=roles, tensor_products=products)
        assert info["tensor_products"] == products and (roles != 3 or info["tensor_shape"] == 3)
        assert_power_parity(P, P_ref, "f32", f"nf={n_freq}/{kernel}/{products}")
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


@pytest.mark.parametrize("roles,n_freq", [(0, 5000), (3, 20_000)], ids=["auto", "cta-pairs"])
def test_normalize_and_center_options(lsp, oracle, roles, n_freq):
    w = make_config(3, n_obj=5, n_freq=n_freq)
    shifted = Workload(w.name, w.offsets, w.t, (w.y + np.float32(3.25)).astype(np.float32), w.f_min, w.f_max, w.n_freq, "f32")
    # center=1 on shifted data == plain call on data centred by numpy in FP64 (to FP32 tolerance)
    yc = shifted.y.astype(np.float64).copy()
    for o in range(w.n_obj):
        s = slice(w.offsets[o], w.offsets[o + 1])
        yc[s] -= yc[s].mean()
    P_ref = oracle.periodogram(w.offsets, w.t, yc, w.f_min, w.f_max, w.n_freq)
    P, _, info = gpu_full(lsp, shifted, center=True, best=False, tensor_roles=roles)
    assert roles != 3 or info["tensor_shape"] == 3
    assert_power_parity(P, P_ref, "f32", "center")
    Pn, _, _ = gpu_full(lsp, shifted, center=True, normalize=True, best=False, tensor_roles=roles)
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


@pytest.mark.parametrize("fast", [False, True])
def test_generalized_fused_epilogue_unsplit_batch(lsp, oracle, fast):
    """The generalised mode's fused tensor-kernel epilogue (n_split = 1: the w pass leaves (C, S) per element, the weighted
    pass evaluates ZK09's power in its own epilogue): a config-3-shaped batch large enough to run unsplit, full periodogram +
    best period; the oracle checks a seeded sample of whole objects, empty and tiny objects included."""
    import torch
    w = make_config(3, n_obj=1300, n_freq=9001)
    off = w.offsets.copy()
    y, sigma = _with_errors(w, 78)
    # make object 3 empty and object 4 a single point (P = 0 rows)
    keep = np.ones(w.n_obs, dtype=bool)
    keep[off[3]:off[4]] = False
    keep[off[4] + 1:off[5]] = False
    lens = np.diff(off)
    lens[3], lens[4] = 0, 1
    off2 = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    t2, y2, s2 = w.t[keep], y[keep], sigma[keep]
    with lsp.Plan(w.f_min, w.f_max, w.n_freq, "f32", fast_math=fast) as plan:
        P, best = plan.periodogram_generalized(torch.from_numpy(off2).cuda(), torch.from_numpy(t2).cuda(), torch.from_numpy(y2).cuda(),
                                               torch.from_numpy(s2).cuda(), best=True, h_offsets=torch.from_numpy(off2))
        info = plan.last_call_info()
        best_only = plan.periodogram_generalized(torch.from_numpy(off2).cuda(), torch.from_numpy(t2).cuda(), torch.from_numpy(y2).cuda(),
                                                 torch.from_numpy(s2).cuda(), best=True, want_power=False)[1]
        P = P.cpu().numpy().astype(np.float64)
        best = tuple(x.cpu().numpy() for x in best)
        best_only = tuple(x.cpu().numpy() for x in best_only)
    assert info["kernel"] == "tensor" and info["n_split"] == 1
    for a_, b_ in zip(best, best_only):
        assert np.array_equal(a_, b_, equal_nan=True)
    rng = np.random.default_rng(8)
    pick = np.unique(np.concatenate([rng.choice(1300, 20, replace=False), [0, 3, 4, 1299]]))
    sub_off = np.concatenate([[0], np.cumsum(lens[pick])]).astype(np.int64)
    sel = np.concatenate([np.arange(off2[o], off2[o + 1]) for o in pick])
    P_ref = oracle.periodogram_generalized(sub_off, t2[sel], y2[sel], s2[sel], w.f_min, w.f_max, w.n_freq)
    assert np.all(P[3] == 0.0) and np.all(P[4] == 0.0) and best[2][3] == -1
    assert np.all(np.isfinite(P)) and P.min() >= -TOL["f32"] and P.max() <= 1.0 + TOL["f32"]
    big = [i for i, o in enumerate(pick) if lens[o] >= 3]
    assert_power_parity(P[pick][big], P_ref[big], "f32", "generalised fused")
    sub = Workload("gls", np.concatenate([[0], np.cumsum(lens[pick][big])]).astype(np.int64), None, None, w.f_min, w.f_max, w.n_freq, "f32")
    assert_best_parity(tuple(x[pick][big] for x in best), P_ref[big], sub, "f32", oracle, "generalised fused")


@pytest.mark.parametrize("dtype,kernel", [("f32", "auto"), ("f32", "factored"), ("f64", "auto")])
def test_generalized_host_output_through_the_chunk_ring(lsp, oracle, dtype, kernel):
    """lsp_periodogram_generalized_host: inputs and outputs on the host, full periodograms back through the chunk ring and the
    copy streams in several rounds (5 objects per chunk, ragged last round), best periods by their own small copies; equal to
    the device-output call bit for bit and to the oracle within tolerance; best-only form as well."""
    import torch
    w = make_config(3, n_obj=23, n_freq=12_007, dtype=dtype)
    y, sigma = _with_errors(w, 91)
    P_ref = oracle.periodogram_generalized(w.offsets, w.t, y, sigma, w.f_min, w.f_max, w.n_freq)
    tdt = torch.float32 if dtype == "f32" else torch.float64
    h_off = torch.from_numpy(w.offsets)
    h_t, h_y, h_s = (torch.from_numpy(x).pin_memory() for x in (w.t, y, sigma))
    host = torch.full((w.n_obj, w.n_freq), float("nan"), dtype=tdt).pin_memory()
    hb = (torch.empty(w.n_obj, dtype=tdt).pin_memory(), torch.empty(w.n_obj, dtype=tdt).pin_memory(),
          torch.empty(w.n_obj, dtype=torch.int64).pin_memory())
    with lsp.Plan(w.f_min, w.f_max, w.n_freq, dtype, kernel=kernel, n_copy_streams=2, chunk_bytes=5 * w.n_freq * host.element_size()) as plan:
        plan.periodogram_generalized_host(h_off, h_t, h_y, h_s, host_out=host, best_out=hb)
        info = plan.last_call_info()
        dev, db = plan.periodogram_generalized(h_off.cuda(), h_t.cuda(), h_y.cuda(), h_s.cuda(), best=True, h_offsets=h_off)
        hb2 = tuple(torch.empty_like(x) for x in hb)
        plan.periodogram_generalized_host(h_off, h_t, h_y, h_s, best_out=hb2)
        torch.cuda.synchronize()
    assert info["chunks"] == 5
    P = host.numpy().astype(np.float64)
    assert_power_parity(P, P_ref, dtype, f"generalised host {dtype}/{kernel}")
    assert np.array_equal(host.numpy(), dev.cpu().numpy())
    best = tuple(x.numpy() for x in hb)
    assert_best_parity(best, P_ref, w, dtype, oracle, "generalised host")
    for a, b, c in zip(hb, db, hb2):
        assert np.array_equal(a.numpy(), b.cpu().numpy(), equal_nan=True) and np.array_equal(a.numpy(), c.numpy(), equal_nan=True)


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
    pick = np.sort(rng.choice(w.n_obj, 64, replace=False))
    pick = np.unique(np.concatenate([pick, [0, w.n_obj - 1]]))          # first and last chunk too
    sub = w.take_objects(pick)
    P_ref = oracle_full(oracle, sub)               # 64+ WHOLE objects on the full 5e5-point grid
    assert_power_parity(P[pick].astype(np.float64), P_ref, "f32", "c4 full")
    for i, o in enumerate(pick):
        yy = sub.y[sub.offsets[i]:sub.offsets[i + 1]].astype(np.float64)
        assert P[o].max() <= 0.5 * float(yy @ yy) * (1 + TOL["f32"])
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
    # the denominator is the ORACLE's maximum over a window that holds its peak: the injected signal's own frequency
    k_true = int(round((1.0 / w.meta["true_period_days"] - w.f_min) / ((w.f_max - w.f_min) / n_freq)))
    kw = np.clip(np.arange(-8, 9) + k_true, 0, n_freq - 1).astype(np.int64)
    pmax = max(P_ref.max(), oracle.periodogram(w.offsets, w.t, w.y, w.f_min, w.f_max, w.n_freq, k_list=np.unique(kw)).max())
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
    lens0, off0, t0, y0 = lens, off, t, y
    # (dtype, kernel variants, shift): the two-product tensor mode only runs when every object has >= 32 observations, so its
    # variants get the same draw with 32 more observations on every non-empty object (48 = 3 stages exactly, 49, 63, ...)
    for dtype, kernels, shift in (("f32", (("tensor", 1, 3), ("tensor", 2, 3), ("tensor", 3, 3), ("factored", 0, 0), ("direct", 0, 0)), 0),
                                  ("f32", (("tensor", 1, 2), ("tensor", 2, 2), ("tensor", 3, 2)), MIN_NT_TWO_PRODUCTS),
                                  ("f64", (("factored", 0, 0),), 0)):
        if shift:
            lens = np.where(lens0 > 0, lens0 + shift, 0)
            off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
            rng2 = np.random.Generator(np.random.PCG64(19000 + seed))
            t = np.concatenate([np.sort(rng2.uniform(0.0, 400.0, n)) for n in lens])
            y = rng2.normal(0.0, 1.0, t.size) + np.sin(2 * np.pi * 1.37 * t)
        else:
            lens, off, t, y = lens0, off0, t0, y0
        w = Workload(f"rand{seed}", off, t.astype(np.float32 if dtype == "f32" else np.float64),
                     y.astype(np.float32 if dtype == "f32" else np.float64), f_min, f_max, n_freq, dtype=dtype)
        P_ref = oracle_full(oracle, w)
        for kernel, roles, products in kernels:
            if roles == 3 and n_freq <= 14_336:
                continue                 # a single tile: nothing to pair
            P, best, info = gpu_full(lsp, w, kernel=kernel, tensor_roles=roles, tensor_products=products)
            assert info["tensor_shape"] == roles and info["tensor_products"] == products
            for o in range(n_obj):
                if lens[o] == 0:
                    assert np.all(P[o] == 0.0)
                elif lens[o] >= 3:       # N_t <= 2 sits on the vanishing-denominator branch (reading a6): finite and bounded only
                    pmax = P_ref[o].max()
                    assert np.max(np.abs(P[o] - P_ref[o])) <= TOL[dtype] * pmax, f"seed {seed} {dtype} {kernel} object {o} (N_t={lens[o]}, N_f={n_freq})"
                else:
                    yy = w.y[off[o]:off[o + 1]].astype(np.float64)
                    # near sin w(t2 - t1) = 0 the 2 x 2 system is ill-conditioned: bounded there, closed form (pin p7) elsewhere
                    assert np.all(np.isfinite(P[o])) and P[o].min() >= -1e-3 * float(yy @ yy) and P[o].max() <= float(yy @ yy) + 1e-30
                    if lens[o] == 2:
                        assert_two_point_pin(P[o], w.t[off[o]:off[o + 1]], w.y[off[o]:off[o + 1]], w, dtype, f"seed {seed} {kernel}")
            big = [o for o in range(n_obj) if lens[o] >= 3]
            if big:
                sub = w.take_objects(big)
                assert_best_parity(tuple(x[big] for x in best), P_ref[big], sub, dtype, oracle, f"seed {seed} {kernel}")


# ---- object ranges under a small operand-table budget; shards through the real library ------------------------------------
def test_table_budget_cut_equals_uncut(lsp):
    """A config-3-shaped batch with the tensor path's B-operand table capped at 1 MiB runs in object ranges; the result must
    equal the uncut call bit for bit (an object's sums never span launches), device and host output."""
    import torch
    w = make_config(3, n_obj=60, n_freq=20_000)
    off, t, y = to_device(w)
    h_off = torch.from_numpy(w.offsets)
    with lsp.Plan(w.f_min, w.f_max, w.n_freq, "f32", kernel="tensor") as plan:
        ref, bref = plan.periodogram_batched(off, t, y, best=True, h_offsets=h_off)
        n_ref = plan.last_call_info()["launches"]
    for h in (h_off, None):
        with lsp.Plan(w.f_min, w.f_max, w.n_freq, "f32", kernel="tensor", table_budget_bytes=1 << 20) as plan:
            cut, bcut = plan.periodogram_batched(off, t, y, best=True, h_offsets=h)
            assert plan.last_call_info()["launches"] > n_ref
            host = torch.empty((w.n_obj, w.n_freq), dtype=torch.float32).pin_memory()
            plan.periodogram_batched(off, t, y, host_out=host, h_offsets=h)      # one chunk, cut inside the chunk
        assert torch.equal(ref, cut) and all(torch.equal(a, b) for a, b in zip(bref, bcut))
        assert torch.equal(ref.cpu(), host)


def test_object_shards_through_the_library_equal_unsharded(lsp):
    """a config-3 batch cut by `sharding.partition_objects` (balanced by sum N_t); each shard runs
    lsp_best_period on its own CSR slice (here: one after the other on one GPU); the concatenation is bit-identical to the
    unsharded call."""
    import torch
    from paper_2105_04006_b200 import sharding
    w = make_config(3, n_obj=300, n_freq=30_000)
    whole, _ = gpu_best(lsp, w)
    for world in (2, 3):
        parts = []
        for o0, o1 in sharding.partition_objects(w.offsets, world):
            off, t, y = sharding.slice_csr(w.offsets, w.t, w.y, o0, o1)
            sub = Workload("shard", off.copy(), t, y, w.f_min, w.f_max, w.n_freq, "f32")
            parts.append(gpu_best(lsp, sub)[0])
        for i in range(3):
            assert np.array_equal(np.concatenate([p[i] for p in parts]), whole[i], equal_nan=True)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_frequency_shards_merge_equals_unsharded(lsp, dtype):
    """A single object cut by `sharding.partition_frequencies`; each shard's fused argmax + lsp_best_merge (the library's own
    tie rule and period) must equal the unsharded fused argmax: same index, same power, same period."""
    import torch
    from paper_2105_04006_b200 import sharding
    w = make_config(2, dtype=dtype, n_t=3000, n_freq=120_000)
    whole, _ = gpu_best(lsp, w)
    tdt = torch.float32 if dtype == "f32" else torch.float64
    for world in (2, 3):
        pp, pk = [], []
        for k0, k1, fa, fb in sharding.partition_frequencies(w.f_min, w.f_max, w.n_freq, world):
            sub = Workload("fshard", w.offsets, w.t, w.y, fa, fb, k1 - k0, dtype)
            (per, pw, idx), _ = gpu_best(lsp, sub)
            pp.append(pw)
            pk.append(np.where(idx >= 0, idx + k0, -1))
        with lsp.Plan(w.f_min, w.f_max, w.n_freq, dtype) as plan:
            per, pw, idx = plan.best_merge(torch.from_numpy(np.stack(pp)).to(tdt).cuda(), torch.from_numpy(np.stack(pk)).cuda())
            per, pw, idx = per.cpu().numpy(), pw.cpu().numpy(), idx.cpu().numpy()
        # the slice grids reproduce the global grid to FP64 rounding (phases move by ~1e-11 cycles at f t = 1.8e5)
        assert idx[0] == whole[2][0]
        assert abs(pw[0] - whole[1][0]) <= TOL[dtype] * whole[1][0]
        assert per[0] == whole[0][0]
    # planted ties / NaN / no-candidate columns: lowest global index wins exact ties, NaN and -1 never win
    with lsp.Plan(w.f_min, w.f_max, w.n_freq, dtype) as plan:
        P = torch.tensor([[7.0, float("nan"), 0.0, 2.0], [7.0, 1.0, 0.0, 3.0]], dtype=tdt).cuda()
        K = torch.tensor([[40, 3, -1, 10], [5, 9, -1, 11]], dtype=torch.int64).cuda()
        per, pw, idx = (x.cpu().numpy() for x in plan.best_merge(P, K))
    assert idx.tolist() == [5, 9, -1, 11] and pw.tolist() == [7.0, 1.0, 0.0, 3.0] and np.isnan(per[2])
    df = (w.f_max - w.f_min) / w.n_freq
    assert abs(per[0] - 1.0 / (w.f_min + 5 * df)) <= 1e-6 / (w.f_min + 5 * df)


def test_two_devices_in_one_process(lsp, oracle):
    """Plans on two devices of one process are independent (the dynamic shared-memory opt-in is per device)."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    w = make_config(2, dtype="f32", n_t=1500, n_freq=9001)
    P_ref = oracle_full(oracle, w)
    for dev in (0, 1):
        with torch.cuda.device(dev):
            for kernel in ("tensor", "factored"):
                off, t, y = (x.to(f"cuda:{dev}") for x in to_device(w))
                with lsp.Plan(w.f_min, w.f_max, w.n_freq, "f32", kernel=kernel, device=dev) as plan:
                    P, _ = plan.periodogram_batched(off, t, y)
                    assert_power_parity(P.cpu().numpy().astype(np.float64), P_ref, "f32", f"device {dev} {kernel}")
