"""paper_2303_10440_b200 -- B200-native (sm_100a) mesh Fourier transform of deltaMic (arxiv 2303.10440).

Thin ctypes binding over the C-ABI library ``libdeltamic.so`` (declared in ``include/deltamic.h``): argument
marshalling only, every step of the path runs in the library's CUDA kernels.  PyTorch supplies device memory and
streams.  There is no CPU fallback: importing the binding without the built library, or calling it without a CUDA
device, raises.
"""
from ._binding import (  # noqa: F401
    DM_OPT_AREA_NORMALISED,
    DM_OPT_BACKWARD_PATH,
    DM_OPT_FORWARD_PATH,
    DM_OPT_REUSE_SPECTRUM,
    DM_OPT_TAU,
    DM_OPT_TAU_BWD,
    DM_SURFACE,
    DM_VOLUME,
    DeltamicError,
    Plan,
    ShapeParams,
    ShapeState,
    exported_symbols,
    library_path,
    load_library,
    mesh_ft_forward_noalloc,
    DM_NOALLOC_MAX_FACES,
    DM_ERR_TOO_LARGE,
    version,
)

from .autograd import mesh_ft, render  # noqa: F401,E402

__all__ = ["mesh_ft", "render", "mesh_ft_forward_noalloc", "DM_NOALLOC_MAX_FACES", "DM_ERR_TOO_LARGE", "Plan", "ShapeState", "ShapeParams", "DM_VOLUME", "DM_SURFACE", "DeltamicError", "load_library", "library_path", "exported_symbols",
           "version"]
