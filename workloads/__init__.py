"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This package holds *data generators only* (meshes, grids, cotangents, frequency samples). It contains
none of the method's arithmetic (no Fourier transform, no PSF, no gradients) and imports neither
``oracle/`` nor the CUDA package, so both sides can consume the same arrays (SURVEY.md §7 step 1,
§8(d) "Synthetic inputs").
"""
from .meshes import (  # noqa: F401
    icosphere,
    box_mesh,
    tetrahedron_mesh,
    perturb_radial,
    laplacian_smooth,
    pack_spheres,
    vertex_one_ring,
)
from .configs import CONFIGS, Workload, build_workload, sampled_frequencies  # noqa: F401
