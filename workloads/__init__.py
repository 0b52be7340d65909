"""Seeded synthetic inputs for the lensed-image hot path (configs C0..C4).

This package holds NONE of the method's arithmetic: it only draws parameters
and builds PSF kernels (harness-side constructions).
It is the one module shared by the CPU oracle's tests and the CUDA path's
tests/bench; neither `oracle/` nor `paper_2606_01547_b200/` imports the other.

The recipe follows BASELINE.json:configs[0..4] (0-based, named C0..C4).
"""
from .configs import (  # noqa: F401
    Workload,
    BatchWorkload,
    SwarmWorkload,
    config_swarm,
    config_c0,
    config_c1,
    config_c2,
    config_c3,
    config_c4,
    conv_sweep_case,
    SEEDS,
)
from .psf import gaussian_psf, mixture3_psf, airymix_psf  # noqa: F401
