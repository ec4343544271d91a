"""Seeded synthetic workloads shaped like the paper's (arXiv:1609.06634 section 4) and like the five
BASELINE.json configs.  This package is the ONLY thing the CUDA path's callers and the oracle's callers share.

It holds: the config table, the model / orientation-grid / CTF-grid generators, and a *synthetic microscope*
(`simulate.py`) that renders noisy particle images.  It imports neither `oracle` nor
`paper_1609_06634_b200`, and neither of them imports it: tests and bench.py generate arrays here and hand the
same arrays to both sides.  Recipe and its readings: DESIGN.md section 4.
"""
from .configs import CONFIGS, WorkloadSpec, get_spec
from .generate import (build_workload, ctf_from_defocus, euler_grid, euler_zyz_to_quat, hopf_fibonacci_grid,
                       make_atom_model, make_density_model, make_ensemble_models, ctf_grid)

__all__ = [
    "CONFIGS", "WorkloadSpec", "get_spec", "build_workload", "ctf_from_defocus", "euler_grid",
    "euler_zyz_to_quat", "hopf_fibonacci_grid", "make_atom_model", "make_density_model",
    "make_ensemble_models", "ctf_grid",
]
