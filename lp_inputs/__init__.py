"""Seeded synthetic inputs for the LP hot path (grid fields, particles, initial spectra).

Shared by the oracle-side tests and the CUDA-side tests/bench: it produces INPUT BYTES
only and contains none of the method's arithmetic (no gather, push, CFL or upwind
step).  It imports neither oracle/ nor paper_2602_23434_b200/.  The recipe is stated
in DESIGN.md section 4; the five workloads are BASELINE.json's `configs`.
"""
from .configs import LPWorkload, workload, WORKLOAD_NAMES  # noqa: F401
from .fields import make_fields, mean_magnetic_energy      # noqa: F401
from .particles import make_particles, make_spectrum, bin_edges  # noqa: F401
