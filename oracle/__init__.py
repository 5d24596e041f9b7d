"""fp64 CPU oracle for the deltaMic mesh Fourier transform -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It shares no code with paper_2303_10440_b200 (the CUDA path) and neither imports the
other.  See oracle/mesh_ft_oracle.c for the definitions and citations, oracle/render.py for the
image-formation reference (PSF multiply + inverse rFFT).

Parity status: every function here is pinned by `-m "not gpu"` tests (tests/test_oracle_*.py) except
the behaviour of an inverse real FFT on a half spectrum that is not exactly Hermitian on its
self-conjugate planes (reading R13), where the oracle *defines* the semantics as numpy/pocketfft's
irfftn -- "parity unpinned" for that one convention.  oracle/shape_step.py (the shape-optimisation step of PAPER.md:244-249) is
pinned by tests/test_oracle_shape.py, piece by piece and as a composition (the first step against finite differences of
Phi_1 o render with the closed-form preconditioner of the tetrahedron, and its band branch against the banded render).
"""
from .mesh_ft import (  # noqa: F401
    frequency_grid,
    g_fun,
    g_grad,
    mesh_ft_forward,
    mesh_ft_forward_grid,
    mesh_ft_backward,
    mesh_ft_backward_grid,
    mesh_ft_backward_normalised,
    mesh_ft_backward_weighted,
    mesh_ft_forward_weighted,
    mesh_ft_forward_normalised,
    surface_area_and_gradient,
    num_threads,
)
from .render import (psf_shift_spectrum, render, render_backward, render_backward_psf, spectrum_to_image,  # noqa: F401
                     image_to_spectrum_cotangent)
from .shape_step import (AdamUniformState, ShapeParams, ShapeState, adam_uniform_step, connectivity_laplacian,  # noqa: F401
                         phi1, phi1_grad, precondition, shape_step)
