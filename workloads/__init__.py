"""Seeded synthetic input generators (shared by the oracle tests, the GPU tests and bench.py).

This package holds NO arithmetic of the method (no curl, no coefficient averaging, no update):
it only builds the *inputs* of the EM time-marching path -- grids, per-cell material ids, the
material table, dt, port edge lists, waveform tables, probe lists and initial fields -- as plain
NumPy arrays.  Both the CPU oracle (``oracle/``) and the CUDA library consume the same arrays.

The five configurations are the synthetic stand-ins named in BASELINE.json ``configs``; the recipe
follows SURVEY.md section 8(d) and is restated in DESIGN.md.  The paper's own layout (PAPER.md
L130-L138, Fig. 1) is not public, so these inputs stand in for its structure.
"""
from .problem import Problem, EPS0, MU0, C0, material_table, thermal_table, MATERIAL_NAMES, cfl_dt
from .configs import (
    config1_cavity,
    config2_slab,
    config3_interposer,
    config4_package,
    config5_graded,
    config6_paper_mesh,
    random_problem,
    impulse_problem,
    make_config,
)

__all__ = [
    "Problem", "EPS0", "MU0", "C0", "material_table", "thermal_table", "MATERIAL_NAMES", "cfl_dt",
    "config1_cavity", "config2_slab", "config3_interposer", "config4_package",
    "config5_graded", "config6_paper_mesh", "random_problem", "impulse_problem", "make_config",
]
