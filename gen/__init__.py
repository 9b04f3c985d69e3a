"""Seeded synthetic-input generators shared by the CPU oracle and the CUDA library.

This package holds NONE of the method's arithmetic (no Q^-1 propagation, no
amplitude, no field sum): it only produces the inputs of the hot path -- the
ray-transfer (ABCD) matrices, base-ray data, pupil weights, position jitter and
the detector descriptor -- as float64 numpy arrays, from fixed seeds.  Both
sides are handed identical bytes.  See DESIGN.md "Input recipe".
"""
from .workloads import (  # noqa: F401
    SEED_BASE, Workload, workload, sweep_workloads, ideal_lens_abcd,
    jitter_positions, apodised_random_weights, zernike_opd, zernike_opd_grad,
    ParaboloidSystem, make_inputs, detector_dict, trace_spec, HST_TABLE2,
)
