"""B200 (sm_100a) FP64 radiation-integral evaluator -- thin Python binding.

Argument marshalling only: every step of the hot path runs in the CUDA kernels of
``csrc/rad.cu`` behind the C ABI of ``include/rad.h``.  PyTorch is used for device
memory and streams.  There is no CPU fallback: if the shared library is missing or
no CUDA device is visible, calls raise.

Functions mirror the C entry points one to one:
``rad_classical``, ``rad_semiclassical``, ``rad_ensemble_sum``, ``rad_sections_sum``, ``rad_sections_check``,
``rad_angular_sum``, ``rad_angular_spectrum``, ``rad_number_spectrum``, ``rad_sum_cubes``, ``rad_workspace_bytes``,
``rad_eval_host``, ``rad_ensemble_sum_host``, ``rad_generate_trajectories``, ``rad_plan_kernel``,
``rad_plan_describe``, ``rad_measure_fp64_peak``, ``rad_launch_count``; per-call options (``kernel=``, ``profile=``)
are keyword arguments (``rad_options`` in the header).
"""
from __future__ import annotations

from .binding import (CLASSICAL, FIELDS, KERNEL_AUTO, KERNEL_DIRECT, KERNEL_FUSED, KERNEL_SEPARABLE, SPIN0, SPIN_HALF,
                      WELL_AXIAL_EXP, WELL_COSINE, WELL_HARMONIC_MS, RadError, RadProfile, build_library, library_path,
                      load_library, rad_angular_spectrum, rad_angular_sum, rad_classical, rad_ensemble_sum,
                      rad_ensemble_sum_host, rad_eval_host, rad_formation_length, rad_generate_trajectories,
                      rad_launch_count, rad_measure_fp64_peak, rad_number_spectrum, rad_plan_describe, rad_plan_kernel,
                      rad_sections_check, rad_sections_sum, rad_semiclassical, rad_sum_cubes, rad_workspace_bytes,
                      rad_eval_static, rad_static_scratch_bytes)
from .sharding import rad_ensemble_sum_sharded, rad_eval_grid_sharded, shard_range, shard_sizes

__all__ = [
    "CLASSICAL", "SPIN0", "SPIN_HALF", "FIELDS", "RadError", "build_library", "library_path",
    "load_library", "rad_classical", "rad_semiclassical", "rad_ensemble_sum", "rad_angular_sum",
    "rad_workspace_bytes", "rad_eval_host", "rad_ensemble_sum_host", "rad_measure_fp64_peak",
    "rad_launch_count", "RadProfile", "rad_sum_cubes", "rad_plan_kernel", "rad_sections_sum", "rad_sections_check",
    "rad_number_spectrum", "KERNEL_AUTO", "KERNEL_DIRECT", "KERNEL_SEPARABLE", "KERNEL_FUSED",
    "rad_generate_trajectories", "rad_plan_describe", "rad_angular_spectrum", "rad_formation_length", "WELL_COSINE", "WELL_AXIAL_EXP", "WELL_HARMONIC_MS",
    "rad_ensemble_sum_sharded", "rad_eval_grid_sharded", "shard_range", "shard_sizes",
    "rad_eval_static", "rad_static_scratch_bytes",
]
