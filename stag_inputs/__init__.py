"""Seeded synthetic inputs for the staggered Dslash / multi-shift CG path.

This module is DATA ONLY: lattice indexing helpers, a counter-based random
number generator, SU(3) link generators, Gaussian sources and the five
workload descriptions of BASELINE.json:configs.  It holds none of the method's
arithmetic (no Dirac operator, no solver) and is the one module that the
oracle (`oracle/`) and the CUDA path (`paper_1010_5433_b200/`) both take their
inputs from.  Recipes are stated in DESIGN.md ("Input recipe").
"""
from .gen import (  # noqa: F401
    volume, half_volume, site_coords, parity_sites,
    links_unit, links_haar, links_smooth, gauge_transform_field,
    apply_gauge_transform, source_gaussian, source_plane_wave, normals,
    su3_project,
)
from .configs import CONFIGS, get_config, make_links, make_source  # noqa: F401
