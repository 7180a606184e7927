"""Seeded synthetic inputs for the tracking hot path (particles + beamlines).

This package is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_1710_07350_b200/``).  It holds none of the method's arithmetic: it
draws particle coordinates from a counter-based generator and writes down the
element lists of the five workloads of BASELINE.json (readings G4-G8, G22-G25 of
SURVEY.md section 8c, restated in DESIGN.md).  Both sides receive the same bytes.
"""
from .rng import uniform01, normal01, SEED_BASE
from .configs import (
    ELECTRON_MC2_EV, C_LIGHT, Workload, make_workload, WORKLOAD_NAMES,
    drift_matrix, thin_quad_matrix, compose, pair_index, second_order_drift, thin_quad_sextupole,
    triple_index, thin_quad_sext_octupole, third_order_drift,
    dense_symplectic_matrix, dense_higher_order, dense_map_element,
)

__all__ = [
    "uniform01", "normal01", "SEED_BASE", "ELECTRON_MC2_EV", "C_LIGHT", "Workload",
    "make_workload", "WORKLOAD_NAMES", "drift_matrix", "thin_quad_matrix", "compose",
    "pair_index", "second_order_drift", "thin_quad_sextupole",
    "triple_index", "thin_quad_sext_octupole", "third_order_drift",
    "dense_symplectic_matrix", "dense_higher_order", "dense_map_element",
]
