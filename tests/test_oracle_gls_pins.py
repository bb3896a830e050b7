"""Pins of the generalised-LSP oracle (oracle/gls_oracle.c, ZK09 = PAPER.md:L520) against things
other than itself: a numpy least-squares fit of the same model, ZK09's closed form typed here independently, the
invariances the floating mean and the weights must have, exact recovery, the classic oracle, and scipy's implementation."""
import numpy as np
import pytest


def _data(seed, n, t_span=30.0):
    rng = np.random.Generator(np.random.PCG64(seed))
    t = np.sort(rng.uniform(0.0, t_span, n))
    sigma = rng.uniform(0.05, 0.4, n)
    y = 3.7 + 0.8 * np.sin(2 * np.pi * t / 1.7 + 0.4) + sigma * rng.normal(size=n)
    return t, y, sigma


def _freqs(f_min, f_max, n_freq):
    return f_min + (f_max - f_min) / n_freq * np.arange(n_freq)


@pytest.mark.parametrize("n_t", [4, 9, 40])
def test_g1_weighted_lstsq_chi2_reduction(oracle, n_t):
    t, y, sigma = _data(11 + n_t, n_t)
    f_min, f_max, n_freq = 0.05, 3.0, 37
    P = oracle.periodogram_generalized([0, n_t], t, y, sigma, f_min, f_max, n_freq)[0]
    w = sigma ** -2.0
    w /= w.sum()
    chi0 = np.sum(w * (y - np.sum(w * y)) ** 2)
    for k, f in enumerate(_freqs(f_min, f_max, n_freq)):
        A = np.stack([np.cos(2 * np.pi * f * t), np.sin(2 * np.pi * f * t), np.ones(n_t)], axis=1) * np.sqrt(w)[:, None]
        r = np.linalg.lstsq(A, y * np.sqrt(w), rcond=None)[0]
        chi = np.sum((y * np.sqrt(w) - A @ r) ** 2)
        assert P[k] == pytest.approx((chi0 - chi) / chi0, abs=2e-12)


def test_g2_zechmeister_kuerster_closed_form(oracle):
    # ZK09 Eq. 5 (tau-free form): p = (SS YC^2 + CC YS^2 - 2 CS YC YS) / (YY D), D = CC SS - CS^2, hatted sums.
    t, y, sigma = _data(5, 60)
    f_min, f_max, n_freq = 0.02, 4.0, 400
    P = oracle.periodogram_generalized([0, 60], t, y, sigma, f_min, f_max, n_freq)[0]
    w = sigma ** -2.0
    w /= w.sum()
    f = _freqs(f_min, f_max, n_freq)[:, None]
    c, s = np.cos(2 * np.pi * f * t), np.sin(2 * np.pi * f * t)
    Y, C, S = np.sum(w * y), (w * c).sum(1), (w * s).sum(1)
    YY = np.sum(w * y * y) - Y * Y
    YC, YS = (w * y * c).sum(1) - Y * C, (w * y * s).sum(1) - Y * S
    CC, SS, CS = (w * c * c).sum(1) - C * C, (w * s * s).sum(1) - S * S, (w * c * s).sum(1) - C * S
    ref = (SS * YC ** 2 + CC * YS ** 2 - 2 * CS * YC * YS) / (YY * (CC * SS - CS ** 2))
    assert np.max(np.abs(P - ref)) <= 1e-12
    assert P.min() >= -1e-15 and P.max() <= 1.0 + 1e-15


def test_g3_floating_mean_and_weight_scale_invariance(oracle):
    t, y, sigma = _data(7, 50)
    args = (0.05, 5.0, 300)
    P = oracle.periodogram_generalized([0, 50], t, y, sigma, *args)[0]
    assert np.max(np.abs(oracle.periodogram_generalized([0, 50], t, y + 123.456, sigma, *args)[0] - P)) <= 1e-11
    assert np.max(np.abs(oracle.periodogram_generalized([0, 50], t, y, 8.0 * sigma, *args)[0] - P)) <= 1e-13
    assert np.max(np.abs(oracle.periodogram_generalized([0, 50], t, 4.0 * y, sigma, *args)[0] - P)) <= 1e-13
    assert np.max(np.abs(oracle.periodogram_generalized([0, 50], t + 1000.0, y, sigma, *args)[0] - P)) <= 1e-10


@pytest.mark.parametrize("m", [3, 150])
def test_g4_noiseless_sinusoid_plus_offset_is_fit_exactly(oracle, m):
    rng = np.random.Generator(np.random.PCG64(99))
    n, f_min, f_max, n_freq = 35, 0.1, 6.1, 200
    f_m = f_min + m * (f_max - f_min) / n_freq
    t = np.sort(rng.uniform(0, 20, n))
    y = -2.5 + 1.3 * np.sin(2 * np.pi * f_m * t + 0.9)
    P = oracle.periodogram_generalized([0, n], t, y, rng.uniform(0.1, 1.0, n), f_min, f_max, n_freq)[0]
    assert P[m] == pytest.approx(1.0, abs=1e-13) and int(np.argmax(P)) == m


def test_g5_reduces_to_classic_when_cos_sin_means_vanish(oracle):
    # even sampling over whole periods, equal errors, zero-mean y: C = S = 0 and the floating mean changes nothing, so
    # P_GLS = P_classic(Eq. 2) / (1/2 sum y^2) ... with w = 1/N:  chi0^2 = sum y^2 / N.
    n = 64
    t = np.arange(n) * 0.25
    rng = np.random.Generator(np.random.PCG64(3))
    y = rng.normal(size=n)
    y -= y.mean()
    fk = np.arange(1, 20) / (n * 0.25)                      # Fourier frequencies: sum cos = sum sin = 0
    f_min, df = fk[0], fk[1] - fk[0]
    Pg = oracle.periodogram_generalized([0, n], t, y, np.full(n, 0.3), f_min, f_min + df * fk.size, fk.size)[0]
    Pc = oracle.periodogram([0, n], t, y, f_min, f_min + df * fk.size, fk.size)[0]
    assert np.max(np.abs(Pg - Pc / (0.5 * np.sum(y * y)))) <= 1e-12


def test_g6_scipy_lombscargle_weights_floating_mean(oracle):
    sig = pytest.importorskip("scipy.signal")
    t, y, sigma = _data(21, 80)
    f_min, f_max, n_freq = 0.05, 4.0, 250
    P = oracle.periodogram_generalized([0, 80], t, y, sigma, f_min, f_max, n_freq)[0]
    try:
        ref = sig.lombscargle(t, y, 2 * np.pi * _freqs(f_min, f_max, n_freq), weights=sigma ** -2.0, floating_mean=True,
                              normalize="normalize", precenter=False)
    except TypeError:
        pytest.skip("this scipy has no weights / floating_mean arguments")
    assert np.max(np.abs(P - ref)) <= 1e-10


def test_g7_batch_rows_and_degenerate_objects(oracle):
    t, y, sigma = _data(1, 30)
    off = np.array([0, 30, 30, 31, 60 - 29])
    tt, yy, ss = np.concatenate([t, t[:1]]), np.concatenate([y, y[:1]]), np.concatenate([sigma, sigma[:1]])
    P = oracle.periodogram_generalized(off[:4], tt, yy, ss, 0.1, 2.0, 50)
    assert np.array_equal(P[0], oracle.periodogram_generalized([0, 30], t, y, sigma, 0.1, 2.0, 50)[0])
    assert np.all(P[1] == 0.0) and np.all(P[2] == 0.0)     # empty object; a single point has chi0^2 = 0
