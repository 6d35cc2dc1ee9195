"""Seeded synthetic inputs for the C-PCM hot path (BASELINE.json configs[0..4]).

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
product path (``paper_1505_07851_b200/``).  It holds none of the method's
arithmetic: no Boys function, no integrals, no A-matrix entries, no solver.  It
only draws geometry, basis-set shaped shells, surface points, P and q from a
seeded ``numpy.random.Generator(PCG64(seed))`` following the recipe stated in
DESIGN.md ("Input recipe") and SURVEY.md section 8(d).
"""
from .generators import (  # noqa: F401
    ANGSTROM,
    Basis,
    Surface,
    Workload,
    make_chain,
    make_basis,
    make_surface,
    make_density,
    make_charges,
    make_workload,
    make_solver_points,
    nuclear_charges,
    cavity_radii,
    CONFIG_ATOMS,
)
