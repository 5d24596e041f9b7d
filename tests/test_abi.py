"""CPU-side checks of the C-ABI library: it builds, loads, and exports every symbol include/deltamic.h declares.
No compute call is made (there is no GPU here)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2303_10440_b200 import build, load_library
    build_mod = __import__("paper_2303_10440_b200.build", fromlist=["build"])
    build_mod.build()
    return load_library()


def _declared():
    text = open(os.path.join(ROOT, "include", "deltamic.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dm_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported_and_bound(lib):
    import paper_2303_10440_b200 as dm
    declared = _declared()
    assert len(declared) >= 12
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in deltamic.h but not exported"
    assert sorted(dm.exported_symbols()) == declared


def test_host_only_entry_points(lib):
    assert lib.dm_version() >= 100
    assert lib.dm_error_string(0) == b"ok"
    assert b"mesh" in lib.dm_error_string(-2)
    assert lib.dm_error_string(-99) == b"unknown error"
    # argument validation happens before any CUDA call
    h = ctypes.c_void_p()
    assert lib.dm_plan_create(ctypes.byref(h), None, 0, 1, 1, None, None) == -1
    assert lib.dm_plan_create(None, None, 0, 1, 1, None, None) == -1
    assert lib.dm_plan_set_slab(None, 0, 1) == -1
    assert lib.dm_mesh_ft_forward(None, None, None) == -1
    assert lib.dm_plan_launch_count(None) == 0
    lib.dm_plan_destroy(None)


def test_noalloc_entry_point_validates_before_any_cuda_call(lib):
    """dm_mesh_ft_forward_noalloc refuses bad arguments and meshes beyond its fixed scratch on the host, before it touches
    the GPU (the pointers below are never dereferenced)."""
    from paper_2303_10440_b200._binding import _Grid
    import paper_2303_10440_b200 as dm
    g = _Grid((ctypes.c_int32 * 3)(8, 8, 8), (ctypes.c_float * 3)(0.125, 0.125, 0.125), (ctypes.c_float * 3)(0, 0, 0))
    fake = ctypes.c_void_p(256)
    assert lib.dm_mesh_ft_forward_noalloc(None, 0, fake, fake, 1, fake, None) == -1
    assert lib.dm_mesh_ft_forward_noalloc(ctypes.byref(g), 0, None, fake, 1, fake, None) == -1
    assert lib.dm_mesh_ft_forward_noalloc(ctypes.byref(g), 2, fake, fake, 1, fake, None) == -1
    assert lib.dm_mesh_ft_forward_noalloc(ctypes.byref(g), 0, fake, fake, 0, fake, None) == -1
    assert lib.dm_mesh_ft_forward_noalloc(ctypes.byref(g), 0, fake, fake, dm.DM_NOALLOC_MAX_FACES + 1, fake, None) == dm.DM_ERR_TOO_LARGE
    assert b"too large" in lib.dm_error_string(dm.DM_ERR_TOO_LARGE)
    header = open(os.path.join(ROOT, "include", "deltamic.h")).read()
    assert f"#define DM_NOALLOC_MAX_FACES {dm.DM_NOALLOC_MAX_FACES}" in header
    assert "DM_ERR_TOO_LARGE   = -7" in header


def test_product_path_has_no_oracle_or_cpu_fallback():
    """The package never imports oracle/ and refuses to run without CUDA."""
    import torch
    import paper_2303_10440_b200 as dm
    pkg = os.path.join(ROOT, "paper_2303_10440_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in src and "from oracle" not in src and "oracle/" not in src, fn
    if not torch.cuda.is_available():
        with pytest.raises(RuntimeError):
            dm.Plan((8, 8, 8), (1 / 8,) * 3, (0, 0, 0), 0, torch.zeros((4, 3), dtype=torch.int32), 4)
