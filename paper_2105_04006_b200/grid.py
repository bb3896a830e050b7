"""Frequency-grid helper and period post-processing (host-side, no periodogram arithmetic).

PAPER.md:L262 (section 4.3, after Richards et al. 2011): the spacing of a practical grid follows from the observing window,
delta_f = 0.2 pi / T_max in ANGULAR frequency (rad per unit of t) -- 0.1 / T_max in cyclic frequency -- with
T_max = |t_1 - t_Nt| of the object (the maximum over the objects of a batch), and N_f = (f_max - f_min) / delta_f.
The library's API takes cyclic frequencies (reading a1); the paper's printed ranges are angular, so both
conversions are here.  PAPER.md:L289: the Lomb-Scargle period of an asteroid light curve is half its rotation period.
"""
from __future__ import annotations

import math

import numpy as np

TWO_PI = 2.0 * math.pi


def angular_to_cyclic(f_angular: float) -> float:
    """rad per unit of t -> cycles per unit of t (the paper's f = 2 pi / p against the API's f = 1 / p)."""
    return f_angular / TWO_PI


def cyclic_to_angular(f_cyclic: float) -> float:
    return f_cyclic * TWO_PI


def observing_window(offsets, t) -> float:
    """T_max: the longest |t_last - t_first| over the objects of a CSR batch (times sorted or not)."""
    off = np.asarray(offsets, dtype=np.int64)
    t = np.asarray(t)
    best = 0.0
    for o in range(off.size - 1):
        seg = t[off[o]:off[o + 1]]
        if seg.size:
            best = max(best, float(seg.max() - seg.min()))
    return best


def delta_f(t_max: float, *, angular: bool = False) -> float:
    """Grid spacing for an observing window T_max: 0.2 pi / T_max (angular) = 0.1 / T_max (cyclic).  PAPER.md:L262."""
    if not t_max > 0:
        raise ValueError("T_max must be positive")
    return (0.2 * math.pi if angular else 0.1) / t_max


def n_freq_for(f_min: float, f_max: float, df: float) -> int:
    """N_f = (f_max - f_min) / delta_f, to the nearest integer (Table 2 prints 28,194 for 28,194.4 and 28,608 for 28,607.9),
    at least 1.  Works in either unit as long as the three arguments share it."""
    if not (f_max > f_min and df > 0):
        raise ValueError("need f_max > f_min and delta_f > 0")
    return max(1, int(round((f_max - f_min) / df)))


def practical_grid(offsets, t, f_min: float, f_max: float):
    """(f_min, f_max, n_freq) in CYCLIC frequency for a CSR batch: the arguments of `Plan`.  The grid is half-open and
    the library derives its own spacing (f_max - f_min) / n_freq, which differs from 0.1 / T_max only by the rounding of N_f."""
    return float(f_min), float(f_max), n_freq_for(f_min, f_max, delta_f(observing_window(offsets, t)))


def light_curve_period(f, *, angular: bool = False):
    """Period of a frequency: 1 / f (cyclic) or 2 pi / f (angular)."""
    f = np.asarray(f, dtype=np.float64)
    return (TWO_PI if angular else 1.0) / f


def rotation_period(ls_period):
    """An asteroid's rotation period from the Lomb-Scargle (light-curve) period: twice it.  The library itself
    never doubles (reading a8)."""
    return 2.0 * np.asarray(ls_period, dtype=np.float64)
