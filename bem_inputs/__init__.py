"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This package holds *no* arithmetic of the method (no kernels, no quadrature, no
expansions): only mesh generators, the five BASELINE.json configurations and
the density recipes of SURVEY.md §8(d) D1.  Both `oracle/` and
`paper_1905_01341_b200/` are fed from here; neither imports the other.
"""
from .meshes import icosphere, cluster_mesh, deform_radial, lattice_cluster
from .sph import real_sph_harm, real_sph_harm_im
from .configs import make_config, sample_rows, CONFIG_SEED0, N_CONFIGS, random_cube_points

__all__ = [
    "icosphere", "cluster_mesh", "deform_radial", "lattice_cluster",
    "real_sph_harm", "real_sph_harm_im",
    "make_config", "sample_rows", "CONFIG_SEED0", "N_CONFIGS", "random_cube_points",
]
