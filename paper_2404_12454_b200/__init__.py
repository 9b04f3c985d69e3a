"""B200-native plane-evaluation Gaussian Beamlet Decomposition (arXiv 2404.12454 hot path).

Product code: csrc/ (CUDA kernels + C ABI, built to libgbd.so) and gbd.py (ctypes binding).
It never imports `oracle` (the CPU checker used by tests and bench baselines).
"""
from . import gbd  # noqa: F401
from .gbd import (  # noqa: F401
    GbdError, Detector, Beamlets, beamlets_create, beamlets_custom, propagate_q, eval_field,
    eval_field_host, eval_field_pointwise, hg_modes, eval_field_modes, eval_workspace_bytes, host_workspace_bytes, probe_dfma, run_workload,
    launch_count, load_library, set_profile_events, psf_metrics, psf_metrics_static, STATIC_METRICS_ROWS, airy_sweep, lattice_count, SweepRun, trace_mirrors, TraceSystem, PRECISION_FP64, PRECISION_MIXED, ALGO_DIRECT, ALGO_RECURRENCE, ALGO_SEPARABLE,
)
