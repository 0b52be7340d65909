"""jt -- B200-native lensed-image simulation (hot path of arxiv/paper_2606_01547).

The product is libjt.so (C ABI in include/jt.h, CUDA kernels in csrc/).  This package is a thin
ctypes binding with the same names; PyTorch supplies device memory and streams only.
There is no CPU fallback: calls raise if libjt.so is missing or no sm_100 device is present.
"""
from .binding import (  # noqa: F401
    Grid,
    chi2_batch,
    simulate_batch_chi2,
    lensing_maps,
    ray_shoot_profiles,
    light_profiles,
    light_core_sersic,
    light_shapelets,
    simulate_image_supersampled_psf,
    profile_records,
    DEFLECTOR_TYPES,
    LIGHT_TYPES,
    JtError,
    lib,
    kernel_launches,
    lib_path,
    probe_alu,
    probe_lib_path,
    profile_enable,
    profile_read,
    profile_tiers,
    psf_convolve,
    psf_convolve_plan,
    trace_plan,
    psf_convolve_batch,
    psf_convolve_batch_workspace_bytes,
    psf_convolve_workspace_bytes,
    ray_shoot,
    ray_shoot_noalloc,
    ray_shoot_noalloc_capacity,
    ray_shoot_workspace_bytes,
    simulate_batch,
    simulate_image,
    simulate_image_workspace_bytes,
    source_brightness,
    version,
)
