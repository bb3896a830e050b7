"""BASELINE.json configs 1-5 as seeded synthetic draws.

Everything is drawn in FP64 with numpy.random.Generator(PCG64(seed)), seed = 210504006 + 1000*config
(+ sweep-point index for config 5), in the draw order listed in DESIGN.md.  Times are sorted
ascending per object, magnitudes are centred per object in FP64 ("the mean is normalized
to zero"; done here, outside every timed region).  FP32 runs round t and y ONCE to
float32 (`as_dtype`); the oracle then receives those float32 values widened back to float64, so input
quantisation is part of the input and not an error of either side.

The frequency grid is only described (f_min, f_max, n_freq: half-open, linear in frequency,
PAPER.md:L53); evaluating it is the business of the oracle and of the CUDA path, separately.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace

import numpy as np

BASE_SEED = 210504006

C5_NT = (1024, 4096, 16384, 65536)
C5_NF = (100_000, 1_000_000, 4_000_000)


@dataclass
class Workload:
    name: str
    offsets: np.ndarray          # int64, n_obj+1, offsets[0] = 0 (CSR)
    t: np.ndarray                # concatenated observation times (days)
    y: np.ndarray                # concatenated magnitudes, centred per object
    f_min: float                 # cycles/day
    f_max: float                 # cycles/day, NOT sampled (half-open grid)
    n_freq: int
    dtype: str = "f64"           # "f64" or "f32": element type of t and y
    meta: dict = field(default_factory=dict)

    @property
    def n_obj(self) -> int:
        return int(self.offsets.shape[0] - 1)

    @property
    def n_obs(self) -> int:
        return int(self.offsets[-1])

    @property
    def pairs(self) -> int:
        """(t, f) pair evaluations of one pass over the workload."""
        return self.n_obs * int(self.n_freq)

    def with_grid(self, f_min=None, f_max=None, n_freq=None) -> "Workload":
        return replace(
            self,
            f_min=self.f_min if f_min is None else float(f_min),
            f_max=self.f_max if f_max is None else float(f_max),
            n_freq=self.n_freq if n_freq is None else int(n_freq),
        )

    def take_objects(self, idx) -> "Workload":
        """A new CSR batch holding the listed objects (whole objects, original order of `idx`)."""
        idx = np.asarray(idx, dtype=np.int64)
        lens = self.offsets[idx + 1] - self.offsets[idx]
        off = np.zeros(idx.size + 1, dtype=np.int64)
        np.cumsum(lens, out=off[1:])
        sel = np.concatenate([np.arange(self.offsets[i], self.offsets[i + 1]) for i in idx]) if idx.size else np.zeros(0, np.int64)
        meta = dict(self.meta)
        for k, v in list(meta.items()):
            if isinstance(v, np.ndarray) and v.shape[:1] == (self.n_obj,):
                meta[k] = v[idx]
        return replace(self, offsets=off, t=self.t[sel], y=self.y[sel], meta=meta)


def config_seed(config: int, point: int = 0) -> int:
    return BASE_SEED + 1000 * int(config) + int(point)


def as_dtype(w: Workload, dtype: str) -> Workload:
    """Round t and y once to `dtype` ("f32" or "f64")."""
    if dtype not in ("f32", "f64"):
        raise ValueError(dtype)
    np_t = np.float32 if dtype == "f32" else np.float64
    return replace(w, t=w.t.astype(np_t), y=w.y.astype(np_t), dtype=dtype)


def _centre(y: np.ndarray) -> np.ndarray:
    return y - y.mean() if y.size else y


def single_object(rng: np.random.Generator, n_t: int, span_days: float, *, period=None, amp=0.5,
                  sigma=0.2, phase=None):
    """Configs 2 and 5: t = sort U(0, span)^n_t; P = U(0.1, 2) d; phi = U(0, 2pi); n = N(0, sigma^2);
    y = amp*sin(2 pi t / P + phi) + n.  Draw order: t, P, phi, n."""
    t = np.sort(rng.uniform(0.0, span_days, n_t))
    if period is None:
        period = rng.uniform(0.1, 2.0)
    if phase is None:
        phase = rng.uniform(0.0, 2.0 * np.pi)
    noise = rng.normal(0.0, sigma, n_t)
    y = amp * np.sin(2.0 * np.pi * t / period + phase) + noise
    return t, _centre(y), float(period), float(phase)


def asteroid_batch(rng: np.random.Generator, n_obj: int, *, nt_lo=50, nt_hi=500, n_nights=3650,
                   intranight=0.3, sigma=0.05):
    """Configs 3 and 4: N_t[i] = integers[nt_lo, nt_hi] (inclusive) for all i first; then per object:
    night = integers[0, n_nights)^N_t, off = U(0, intranight)^N_t, t = sort(night + off);
    A = U(0.05, 0.5); P_h = exp U(ln 2, ln 100) hours; n = N(0, sigma^2); y = A sin(4 pi t / P) + n."""
    n_t = rng.integers(nt_lo, nt_hi + 1, size=n_obj)
    offsets = np.zeros(n_obj + 1, dtype=np.int64)
    np.cumsum(n_t, out=offsets[1:])
    t = np.empty(int(offsets[-1]), dtype=np.float64)
    y = np.empty_like(t)
    amps = np.empty(n_obj)
    periods_h = np.empty(n_obj)
    for i in range(n_obj):
        n = int(n_t[i])
        night = rng.integers(0, n_nights, size=n)
        off = rng.uniform(0.0, intranight, n)
        ti = np.sort(night + off)
        a = rng.uniform(0.05, 0.5)
        p_h = float(np.exp(rng.uniform(np.log(2.0), np.log(100.0))))
        noise = rng.normal(0.0, sigma, n)
        yi = a * np.sin(4.0 * np.pi * ti / (p_h / 24.0)) + noise
        lo, hi = offsets[i], offsets[i + 1]
        t[lo:hi] = ti
        y[lo:hi] = _centre(yi)
        amps[i] = a
        periods_h[i] = p_h
    return offsets, t, y, amps, periods_h


def few_night_batch(n_nights: int, window: float, *, n_obj: int = 30, nt_lo: int = 32, nt_hi: int = 60, signal: bool = False,
                    n_freq: int = 100_000, dtype: str = "f32", seed: int = 0) -> Workload:
    """Ill-conditioned survey cadences (ZTF/LSST-like records of a few short nights): the asteroid_batch
    recipe with short objects (N_t = integers[nt_lo, nt_hi]) on `n_nights` nights and a nightly window of `window` days, on
    config 3's grid.  signal = False: y = N(0, 1) only (nothing lifts max P above the noise floor -- the hardest case for a
    reduced-precision contraction); signal = True: asteroid_batch's sinusoid + N(0, 0.05^2).  Seed: BASE_SEED + 9000 + seed."""
    rng = np.random.Generator(np.random.PCG64(BASE_SEED + 9000 + seed))
    if signal:
        offsets, t, y, _, _ = asteroid_batch(rng, n_obj, nt_lo=nt_lo, nt_hi=nt_hi, n_nights=n_nights, intranight=window)
    else:
        n_t = rng.integers(nt_lo, nt_hi + 1, size=n_obj)
        offsets = np.zeros(n_obj + 1, dtype=np.int64)
        np.cumsum(n_t, out=offsets[1:])
        t = np.empty(int(offsets[-1]), dtype=np.float64)
        y = np.empty_like(t)
        for i in range(n_obj):
            n = int(n_t[i])
            ti = np.sort(rng.integers(0, n_nights, size=n) + rng.uniform(0.0, window, n))
            t[offsets[i]:offsets[i + 1]] = ti
            y[offsets[i]:offsets[i + 1]] = _centre(rng.normal(0.0, 1.0, n))
    w = Workload(f"fewnight_{n_nights}x{window}_{'signal' if signal else 'noise'}", offsets, t, y, 24.0 / 200.0, 24.0, n_freq,
                 meta={"n_nights": n_nights, "window": window})
    return as_dtype(w, dtype)


def make_config(config: int, *, dtype: str = None, n_obj: int = None, n_freq: int = None,
                n_t: int = None, point: int = 0) -> Workload:
    """BASELINE.json config `config` (1..5).  `n_obj`, `n_freq`, `n_t` shrink a config for parity tests
    (same generator, same seed, fewer draws); config 5 takes (n_t, n_freq) of the sweep point and
    `point` = its index in the C5_NT x C5_NF grid (row-major)."""
    rng = np.random.Generator(np.random.PCG64(config_seed(config, point)))
    if config == 1:
        n = 100 if n_t is None else n_t
        t = np.sort(rng.uniform(0.0, 10.0, n))
        noise = rng.normal(0.0, 0.1, n)
        y = _centre(np.sin(2.0 * np.pi * t / 0.3) + noise)
        w = Workload("c1_single_f64", np.array([0, n], dtype=np.int64), t, y, 0.1, 20.0,
                     10_000 if n_freq is None else n_freq, meta={"true_period_days": 0.3})
        default_dtype = "f64"
    elif config in (2, 5):
        n = (10_000 if config == 2 else C5_NT[0]) if n_t is None else n_t
        t, y, period, phase = single_object(rng, n, 3650.0)
        nf = (1_000_000 if config == 2 else C5_NF[0]) if n_freq is None else n_freq
        w = Workload(f"c{config}_single_nt{n}_nf{nf}", np.array([0, n], dtype=np.int64), t, y, 0.05, 50.0,
                     nf, meta={"true_period_days": period, "phase": phase})
        default_dtype = "f64"
    elif config in (3, 4):
        no = (10_000 if config == 3 else 2_000) if n_obj is None else n_obj
        offsets, t, y, amps, periods_h = asteroid_batch(rng, no)
        nf = (100_000 if config == 3 else 500_000) if n_freq is None else n_freq
        # periods of 1-200 hours -> [24/200, 24/1) cycles/day
        w = Workload(f"c{config}_batch_no{no}_nf{nf}", offsets, t, y, 24.0 / 200.0, 24.0, nf,
                     meta={"amp": amps, "rotation_period_h": periods_h})
        default_dtype = "f32"
    else:
        raise ValueError(f"unknown config {config}")
    return as_dtype(w, default_dtype if dtype is None else dtype)
