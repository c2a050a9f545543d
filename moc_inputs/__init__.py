"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

This package holds NONE of the method's arithmetic (no track laydown, no ray
walk, no sweep, no source, no eigenvalue update).  It only produces the input
arrays of a planar-MOC problem: a conforming triangle mesh of a rectangle,
per-triangle material ids, multigroup cross sections, a polar quadrature and
the run parameters of the five BASELINE.json configurations.  Both sides read
identical bytes from here; neither the oracle nor the product imports the
other.

Stand-in note: the paper measures on C5G7, ABTR,
Empire and MSRE.  None of those benchmark specifications,
meshes or cross-section sets are reproduced here; the generators only take
their *shapes* (lattice kinds, group counts, element counts) and draw every
number from a seeded numpy Generator.
"""
from .quadrature import tabuchi_yamamoto
from .mesh import (Mesh, validate_mesh, rect_tri_mesh, pin_cell_mesh,
                   square_lattice_mesh, hex_core_mesh, delaunay_mesh)
from .xs import CrossSections, make_xs, homogeneous_xs
from .configs import Problem, make_config, N_CONFIGS, BC_VACUUM, BC_REFLECTIVE

__all__ = [
    "tabuchi_yamamoto", "Mesh", "validate_mesh", "rect_tri_mesh", "pin_cell_mesh",
    "square_lattice_mesh", "hex_core_mesh", "delaunay_mesh", "CrossSections",
    "make_xs", "homogeneous_xs", "Problem", "make_config", "N_CONFIGS",
    "BC_VACUUM", "BC_REFLECTIVE",
]
