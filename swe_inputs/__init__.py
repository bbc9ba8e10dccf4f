"""Seeded synthetic inputs (meshes, bathymetry, initial fields, boundary tags) for the five
BASELINE.json configs.

This package serves BOTH the CPU oracle (``oracle/``) and the CUDA library
(``paper_2307_16758_b200/``).  It holds none of the method's arithmetic: no flux, no gradient,
no limiter, no time step -- only geometry-free array generation (lattices, jitter, lattice noise,
depth = max(0, level - bed)).  Recipes are stated in DESIGN.md ("Input recipe").
"""
from .meshes import grid_mesh, river_mesh, boundary_edges, delaunay_mesh
from .noise import value_noise, gaussian_bumps
from .configs import (config0, config1, config2, config3, simple_wave_case, lake_case,
                      channel_flow_case, permuted, flooded, delaunay_case, CONFIG_BUILDERS)

__all__ = ["grid_mesh", "river_mesh", "boundary_edges", "value_noise", "gaussian_bumps",
           "config0", "config1", "config2", "config3", "simple_wave_case", "lake_case",
           "channel_flow_case", "permuted", "flooded", "delaunay_case", "delaunay_mesh",
           "CONFIG_BUILDERS"]
