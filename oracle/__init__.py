"""CPU oracle of the GBD plane-evaluation hot path (TEST INFRASTRUCTURE -- not the product).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It never imports paper_2404_12454_b200 and vice versa.
"""
from .gbd_oracle import (  # noqa: F401
    lattice, waist, propagate, to_detector, field, field_rows, field_pixels, field_points,
    run_workload, psf_metrics, trace_mirrors, field_pointeval, hg_modes, field_modes, num_threads, set_num_threads, NREC,
)
