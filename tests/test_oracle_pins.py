"""Pins for the CPU oracle (oracle/lsp_oracle.c) against what the paper and the mathematics fix.

The paper prints no periodogram values, so the oracle is pinned by identities that
hold for Eq. 1-2 and by a brute-force least-squares fit, each chosen so that a
plausible mistake (dropped 1/2, wrong sign of tau, sin/cos swapped, transposed output, off-by-one grid)
fails at least one of them.  None of these tests retypes the oracle's formula.
"""
import numpy as np
import pytest

from workloads import make_config

TWO_PI = 2.0 * np.pi


def _rand_series(rng, n_t, span=10.0):
    t = np.sort(rng.uniform(0.0, span, n_t))
    y = rng.normal(0.0, 1.0, n_t)
    return t, y


def _csr(*series):
    off = np.zeros(len(series) + 1, dtype=np.int64)
    off[1:] = np.cumsum([len(s[0]) for s in series])
    t = np.concatenate([s[0] for s in series]) if series else np.zeros(0)
    y = np.concatenate([s[1] for s in series]) if series else np.zeros(0)
    return off, t, y


# ---- p1: chi^2 reduction of a brute-force least-squares sinusoid fit (BASELINE.json north_star) -----------
@pytest.mark.parametrize("n_t", [3, 4, 7, 20])
def test_p1_chi2_reduction_lstsq(oracle, n_t):
    """P(f) = 1/2 [ sum y^2 - min_{a,b} sum (y - a cos wt - b sin wt)^2 ]  (Lomb 1976 / Scargle 1982:
    Eq. 2 is the chi^2 reduction of the best-fitting sinusoid at w; PAPER.md:L13 'least-squares')."""
    rng = np.random.default_rng(100 + n_t)
    t, y = _rand_series(rng, n_t)
    y = y + 0.3                       # NOT centred: the identity holds for any y
    f_min, f_max, n_freq = 0.2, 3.0, 37
    off, tt, yy = _csr((t, y))
    P = oracle.periodogram(off, tt, yy, f_min, f_max, n_freq)[0]
    f = f_min + np.arange(n_freq) * (f_max - f_min) / n_freq
    ref = np.empty(n_freq)
    for k in range(n_freq):
        A = np.stack([np.cos(TWO_PI * f[k] * t), np.sin(TWO_PI * f[k] * t)], axis=1)
        coef, *_ = np.linalg.lstsq(A, y, rcond=None)
        resid = y - A @ coef
        ref[k] = 0.5 * (np.dot(y, y) - np.dot(resid, resid))
    assert np.max(np.abs(P - ref)) <= 1e-12 * np.max(ref)


# ---- p2: tau-free quadratic form, an algebraically independent route -----------------------------------
def test_p2_tau_free_quadratic_form_config1(oracle):
    """P = 1/2 b^T M^-1 b with b = (sum y cos wt, sum y sin wt), M = [[CC, CS], [CS, SS]] (un-rotated sums):
    the normal-equation form of the same fit; checks Eq. 1's tau really diagonalises M."""
    w = make_config(1, n_freq=2000)
    P = oracle.periodogram(w.offsets, w.t, w.y, w.f_min, w.f_max, w.n_freq)[0]
    f = w.f_min + np.arange(w.n_freq) * (w.f_max - w.f_min) / w.n_freq
    th = TWO_PI * np.outer(f, w.t)
    c, s = np.cos(th), np.sin(th)
    xc, xs = c @ w.y, s @ w.y
    CC, SS, CS = (c * c).sum(1), (s * s).sum(1), (c * s).sum(1)
    ref = 0.5 * (SS * xc**2 + CC * xs**2 - 2 * CS * xc * xs) / (CC * SS - CS**2)
    assert np.max(np.abs(P - ref)) <= 1e-12 * np.max(ref)


# ---- p3: bounds ------------------------------------------------------------------------------------------
def test_p3_bounds(oracle):
    """0 <= P(f) <= 1/2 sum y^2 (a chi^2 reduction cannot be negative nor exceed the total)."""
    w = make_config(3, n_obj=6, n_freq=3000, dtype="f64")
    P = oracle.periodogram(w.offsets, w.t, w.y, w.f_min, w.f_max, w.n_freq)
    for o in range(w.n_obj):
        yy = w.y[w.offsets[o]:w.offsets[o + 1]]
        assert P[o].min() >= 0.0
        assert P[o].max() <= 0.5 * np.dot(yy, yy) * (1 + 1e-12)


# ---- p4 / p5: invariances (BASELINE.json north_star) -----------------------------------------------------
def test_p4_time_shift_invariance(oracle):
    """P(t + c) = P(t): tau absorbs the shift (Scargle 1982; the reason Eq. 1 exists)."""
    rng = np.random.default_rng(4)
    t, y = _rand_series(rng, 60)
    off, tt, yy = _csr((t, y))
    P0 = oracle.periodogram(off, tt, yy, 0.1, 5.0, 500)[0]
    P1 = oracle.periodogram(off, tt + 123.456, yy, 0.1, 5.0, 500)[0]
    assert np.max(np.abs(P0 - P1)) <= 1e-11 * P0.max()
    # and it is NOT invariant without tau: guards against a test that cannot fail
    assert P0.max() > 0


def test_p5_scaling(oracle):
    """P(a y) = a^2 P(y), exactly for a power of two; argmax unchanged."""
    rng = np.random.default_rng(5)
    t, y = _rand_series(rng, 45)
    off, tt, yy = _csr((t, y))
    P0 = oracle.periodogram(off, tt, yy, 0.1, 5.0, 400)[0]
    P4 = oracle.periodogram(off, tt, 4.0 * yy, 0.1, 5.0, 400)[0]
    assert np.array_equal(P4, 16.0 * P0)
    P3 = oracle.periodogram(off, tt, 3.0 * yy, 0.1, 5.0, 400)[0]
    assert np.max(np.abs(P3 - 9.0 * P0)) <= 1e-13 * P3.max()
    assert np.argmax(P3) == np.argmax(P0)


# ---- p6: noiseless on-grid sinusoid (BASELINE.json north_star) -------------------------------------------
@pytest.mark.parametrize("m,phi", [(0, 0.3), (137, 1.1), (499, 2.9)])
def test_p6_noiseless_sinusoid_exact_recovery(oracle, m, phi):
    """y = A sin(2 pi f_m t + phi) with f_m ON the grid is fit exactly: P(f_m) = 1/2 sum y^2, k* = m, and
    the reported period is 1/f_m (PAPER.md:L87 with cyclic f, reading a1).  Pins the grid (half-open,
    f_k = f_min + k df), the index and the period convention; an off-by-one grid fails it."""
    rng = np.random.default_rng(6)
    f_min, f_max, n_freq = 0.5, 8.0, 500
    df = (f_max - f_min) / n_freq
    f_m = f_min + m * df
    t = np.sort(rng.uniform(0.0, 40.0, 80))
    y = 0.7 * np.sin(TWO_PI * f_m * t + phi)
    off, tt, yy = _csr((t, y))
    P = oracle.periodogram(off, tt, yy, f_min, f_max, n_freq)
    assert abs(P[0, m] - 0.5 * np.dot(y, y)) <= 1e-12 * np.dot(y, y)
    idx, bp, per = oracle.best(off, P, f_min, f_max, n_freq)
    assert idx[0] == m
    assert bp[0] == P[0, m]
    assert abs(per[0] - 1.0 / f_m) <= 1e-15 / f_m * 4
    # grid: last sampled frequency is f_max - df, never f_max
    g = oracle.grid(f_min, f_max, n_freq)
    assert g[0] == f_min and abs(g[-1] - (f_max - df)) < 1e-12 and g.size == n_freq


# ---- p7: N_t = 2 ------------------------------------------------------------------------------------------
def test_p7_two_points_fit_exactly(oracle):
    """Two points are fit exactly by a cos + b sin whenever sin w(t2 - t1) != 0: P = (y1^2 + y2^2)/2."""
    t = np.array([0.37, 1.91])
    y = np.array([0.8, -1.7])
    off, tt, yy = _csr((t, y))
    P = oracle.periodogram(off, tt, yy, 0.11, 0.3, 19)[0]   # w dt stays away from multiples of pi
    assert np.max(np.abs(P - 0.5 * (y @ y))) <= 1e-12


# ---- p8: even sampling reduces to the textbook (Schuster) DFT periodogram -------------------------------
def test_p8_even_sampling_dft(oracle):
    """t_j = j dt, f_m = m/(N dt), 0 < m < N/2  =>  tau = 0 (mod quarter period), CC = SS = N/2 and
    P = |sum y_j exp(-i w t_j)|^2 / N, computed here with numpy's FFT (a library routine)."""
    rng = np.random.default_rng(8)
    N, dt = 64, 0.25
    t = np.arange(N) * dt
    y = rng.normal(0, 1, N)
    f1 = 1.0 / (N * dt)
    # grid f_min = f1, N_f = N/2 - 1 points spaced f1: m = 1 .. N/2 - 1
    n_freq = N // 2 - 1
    off, tt, yy = _csr((t, y))
    P = oracle.periodogram(off, tt, yy, f1, f1 * (N // 2), n_freq)[0]
    Y = np.fft.fft(y)
    ref = np.abs(Y[1:N // 2]) ** 2 / N
    assert np.max(np.abs(P - ref)) <= 1e-12 * ref.max()


# ---- p10: the paper's own accuracy check, by library call ------------------------------------------------
def test_p10_scipy_lombscargle(oracle):
    """PAPER.md:L293/L327 validate against scipy.signal.lombscargle (angular frequencies, un-normalised)."""
    sig = pytest.importorskip("scipy.signal")
    w = make_config(1, n_freq=1500)
    P = oracle.periodogram(w.offsets, w.t, w.y, w.f_min, w.f_max, w.n_freq)[0]
    f = oracle.grid(w.f_min, w.f_max, w.n_freq)
    ref = sig.lombscargle(w.t, w.y, TWO_PI * f)
    assert np.max(np.abs(P - ref)) <= 1e-11 * ref.max()


# ---- self-bound: FP64 oracle against its all-long-double twin --------------------------------------------
def test_long_double_self_bound_large_phase(oracle):
    """The FP64 oracle's own rounding error at config-2-sized phases (f t up to 1.8e5 cycles) stays two
    orders inside the FP64 GPU tolerance 1e-9 max P."""
    w = make_config(2, n_t=400, n_freq=1_000_000)
    ks = np.unique(np.linspace(0, w.n_freq - 1, 300).astype(np.int64))
    P = oracle.periodogram(w.offsets, w.t, w.y, w.f_min, w.f_max, w.n_freq, k_list=ks)[0]
    PL = oracle.periodogram(w.offsets, w.t, w.y, w.f_min, w.f_max, w.n_freq, k_list=ks, long_double=True)[0]
    assert np.max(np.abs(P - PL)) <= 1e-11 * PL.max()


# ---- batch layout / best-period conventions ---------------------------------------------------------------
def test_batch_rows_equal_single_object_calls(oracle):
    """Row o of a CSR batch equals the periodogram of object o alone (guards CSR offsets / transposition),
    and k_list picks grid indices."""
    w = make_config(3, n_obj=5, n_freq=257, dtype="f64")
    P = oracle.periodogram(w.offsets, w.t, w.y, w.f_min, w.f_max, w.n_freq)
    assert P.shape == (5, 257)
    for o in range(w.n_obj):
        one = w.take_objects([o])
        Po = oracle.periodogram(one.offsets, one.t, one.y, w.f_min, w.f_max, w.n_freq)[0]
        assert np.array_equal(P[o], Po)
    ks = np.array([0, 5, 256, 17], dtype=np.int64)
    Pk = oracle.periodogram(w.offsets, w.t, w.y, w.f_min, w.f_max, w.n_freq, k_list=ks)
    assert np.array_equal(Pk, P[:, ks])


def test_best_tie_break_nan_and_empty(oracle):
    """Lowest index wins exact ties; NaN never wins; N_t = 0 gives index -1, period NaN (readings a6, a7)."""
    off = np.array([0, 3, 3, 5], dtype=np.int64)           # object 1 is empty
    power = np.array([[1.0, 7.0, 7.0, np.nan, 2.0],
                      [0.0, 0.0, 0.0, 0.0, 0.0],
                      [np.nan, 3.0, 1.0, 3.0, 0.5]])
    idx, bp, per = oracle.best(off, power, 1.0, 6.0, 5)
    assert idx.tolist() == [1, -1, 1]
    assert bp.tolist() == [7.0, 0.0, 3.0]
    assert per[0] == 1.0 / 2.0 and np.isnan(per[1]) and per[2] == 0.5


def test_empty_object_power_is_zero(oracle):
    rng = np.random.default_rng(11)
    a = _rand_series(rng, 5)
    e = (np.zeros(0), np.zeros(0))
    off, tt, yy = _csr(a, e)
    P = oracle.periodogram(off, tt, yy, 0.1, 1.0, 10)
    assert np.all(P[1] == 0.0) and np.all(P[0] > 0.0)


def test_config1_best_period_sanity(oracle):
    """Config 1 (BASELINE.json): the injected 0.3 d period is recovered (sanity, not parity)."""
    w = make_config(1)
    P = oracle.periodogram(w.offsets, w.t, w.y, w.f_min, w.f_max, w.n_freq)
    idx, bp, per = oracle.best(w.offsets, P, w.f_min, w.f_max, w.n_freq)
    assert abs(per[0] - 0.3) < 0.002


def test_config3_peak_is_half_rotation_period(oracle):
    """Config 3's signal is sin(4 pi t / P): the LS period is P/2 (reading a8)."""
    w = make_config(3, n_obj=3, n_freq=100_000, dtype="f64")
    hits = 0
    for o in range(3):
        one = w.take_objects([o])
        f_true = 2.0 / (one.meta["rotation_period_h"][0] / 24.0)
        k0 = int(round((f_true - w.f_min) / ((w.f_max - w.f_min) / w.n_freq)))
        ks = np.arange(max(0, k0 - 40), min(w.n_freq, k0 + 41), dtype=np.int64)
        P = oracle.periodogram(one.offsets, one.t, one.y, w.f_min, w.f_max, w.n_freq, k_list=ks)[0]
        yy = one.y
        hits += P.max() > 0.25 * 0.5 * (yy @ yy)
    assert hits == 3


# ---- p11: the low-order bits of the phase at config-2 magnitudes, against exact rational arithmetic -------------
def test_p11_phase_reduction_against_exact_rationals(oracle):
    """At config 2's scale f*t reaches ~1.8e5 cycles: the fractional part keeps only ~35 of the product's 53 bits unless the
    rounding error of f*t is carried along (the oracle's compensation term).  Here the phase of every (f_k, t_j) is reduced
    with exact rationals -- Fraction(f) * Fraction(t) mod 1, every double is a dyadic rational -- and the power follows from
    the tau-free normal equations  P = 1/2 b^T M^-1 b  (b = sum y (cos, sin), M = sum (cos, sin)(cos, sin)^T), a route that
    shares neither the reduction nor Eq. 1's tau with the oracle.  Dropping or mis-signing the compensation term moves the
    phase by ulp(1.8e5)/2 ~ 1.5e-11 cycles and P by ~1e-10 of max P; the bound is 1e-12."""
    from fractions import Fraction
    rng = np.random.default_rng(1105)
    f_min, f_max, n_freq = 0.05, 50.0, 1_000_000                       # config 2's grid
    ks = np.sort(rng.choice(np.arange(900_000, n_freq), 20, replace=False))      # f ~ 45-50 c/d
    t = np.sort(rng.uniform(3000.0, 3650.0, 40))                        # f * t ~ 1.4e5 .. 1.8e5 cycles
    y = rng.normal(0.0, 1.0, t.size)
    y -= y.mean()
    off = np.array([0, t.size], dtype=np.int64)
    P = oracle.periodogram(off, t, y, f_min, f_max, n_freq, k_list=ks)[0]
    f = oracle.grid(f_min, f_max, n_freq, k_list=ks)
    ref = np.empty_like(P)
    for i, fk in enumerate(f):
        ff = Fraction(float(fk))
        r = np.array([float(((ff * Fraction(float(tj))) % 1)) for tj in t])          # exact product, exact mod, one rounding
        c, s = np.cos(TWO_PI * r), np.sin(TWO_PI * r)
        b = np.array([y @ c, y @ s])
        M = np.array([[c @ c, c @ s], [c @ s, s @ s]])
        ref[i] = 0.5 * b @ np.linalg.solve(M, b)
    assert np.max(np.abs(P - ref)) <= 1e-12 * ref.max()
    # the pin bites: the same evaluation with the naively reduced double product is off by far more than the bound
    naive = np.empty_like(P)
    for i, fk in enumerate(f):
        r = np.mod(fk * t, 1.0)
        c, s = np.cos(TWO_PI * r), np.sin(TWO_PI * r)
        b = np.array([y @ c, y @ s])
        M = np.array([[c @ c, c @ s], [c @ s, s @ s]])
        naive[i] = 0.5 * b @ np.linalg.solve(M, b)
    assert np.max(np.abs(naive - ref)) > 1e-11 * ref.max()


# ---- the object-parallel branch of the batch driver (n_obj >= 2 x threads), reachable on any box with one thread -------
def test_object_parallel_branch_equals_single_object_calls(oracle):
    """lsp_oracle_periodogram loops over objects in parallel when n_obj >= 2 x threads, else over frequencies.  On a many-core
    box small CPU batches only ever take the second loop; with n_threads = 1 a 5-object batch takes the first.  Both must
    return, row for row, what single-object calls return (those take the frequency loop)."""
    rng = np.random.default_rng(77)
    series = [_rand_series(rng, n) for n in (5, 0, 31, 2, 64)]
    off, t, y = _csr(*series)
    f_min, f_max, n_freq = 0.1, 4.0, 301
    ks = np.array([0, 7, 150, 300])
    _, default_threads = oracle.periodogram(off[:2], t[:5], y[:5], f_min, f_max, n_freq, return_threads=True)
    try:
        P1, used = oracle.periodogram(off, t, y, f_min, f_max, n_freq, n_threads=1, return_threads=True)
        Pk = oracle.periodogram(off, t, y, f_min, f_max, n_freq, k_list=ks, n_threads=1)
    finally:
        oracle.periodogram(off[:2], t[:5], y[:5], f_min, f_max, n_freq, n_threads=default_threads)     # give the threads back
    assert used == 1 and P1.shape == (5, n_freq)
    for o, (to, yo) in enumerate(series):
        single = oracle.periodogram(np.array([0, len(to)], dtype=np.int64), to, yo, f_min, f_max, n_freq)[0]
        assert np.array_equal(P1[o], single)
        assert np.array_equal(Pk[o], single[ks])
    assert np.all(P1[1] == 0.0)
