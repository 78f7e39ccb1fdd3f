"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is the ONLY code shared by the fp64 oracle (`oracle/`) and the CUDA
library (`paper_1910_11335_b200/`).  It holds no transport arithmetic: it only
builds the *inputs* a DOCTORS user would supply — voxel
mesh, material map, density, multigroup tables, source description — from a
counter-based splitmix64 generator, so both sides see identical arrays.

The phantoms stand in for the paper's water cylinder / abdomen phantom and its
90-group NJOY library, none of which exist in this container.
"""
from .rng import splitmix64_u64, uniform01, normal01
from .configs import (Workload, SourceSpec, make_config, make_xs, CONFIG_NAMES,
                      energy_grid, single_sweep_case, paper_shaped)

__all__ = ["splitmix64_u64", "uniform01", "normal01", "Workload", "SourceSpec",
           "make_config", "make_xs", "CONFIG_NAMES", "energy_grid",
           "single_sweep_case", "paper_shaped"]
