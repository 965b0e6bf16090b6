"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA-side tests/bench.

This package holds NONE of the method's arithmetic (no DFT, no convolution): it only
draws the densities rho and the real-space Green's functions K that BASELINE.json's
configs describe, plus the one kernel that is *defined* in Fourier space (-1/k^2).
Neither `oracle/` nor `paper_1211_5244_b200/` is imported from here.
"""
from .generators import (  # noqa: F401
    CONFIGS,
    WorkloadConfig,
    SplitMix64,
    get_config,
    gaussian_density,
    green_kernel_realspace,
    periodic_kernel_spectrum,
    padded_shape,
    signed_displacement,
)
