"""Seeded synthetic light-curve generators shared by the oracle tests and the GPU harness.

This module holds NONE of the Lomb-Scargle arithmetic: it only draws observation times and
magnitudes with the shapes BASELINE.json's five configs name (recipe: DESIGN.md "Input recipe",
SURVEY.md section 8(d)) and describes the frequency grid as three numbers.  Neither `oracle/`
nor the CUDA path is imported from here.
"""
from .configs import (  # noqa: F401
    Workload,
    make_config,
    single_object,
    asteroid_batch,
    few_night_batch,
    config_seed,
    as_dtype,
    C5_NT,
    C5_NF,
)
