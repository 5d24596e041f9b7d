"""dm_mesh_ft_forward_noalloc against the plan-based forward (named test_zz_* so that pytest collects it last).

Who needs that entry point: a program that may not allocate device memory while it runs -- its GPU memory is already
committed to one arena (a framework's caching allocator, a fixed per-service budget), or it sits in a loop that cannot
take the device-wide stall of cudaMalloc / cudaFree -- and so cannot create a dm_plan, whose workspace comes from
cudaMalloc.  The entry point takes the caller's buffers and keeps its scratch (triangle records, block sums of the
k = 0 entry) in a fixed 4 MiB array inside libdeltamic.so that all calls on the GPU share.

What is checked, on two calls in a row that share that array (the second on a SMALLER mesh in the other mode, so stale
records of the first call lie behind the ones it writes):
  - each result equals the plan's robust forward (DM_OPT_FORWARD_PATH = 1: the same kernels with cudaMalloc'ed scratch)
    bit for bit, and the plan's default (strip-kernel) forward within the tolerance of the GPU parity tests,
    max|dF| <= 1e-4 |F(0)|;
  - a third call, repeating the first, reproduces the first call's bits (nothing leaks from call to call);
  - a mesh beyond DM_NOALLOC_MAX_FACES is refused with DM_ERR_TOO_LARGE and the output is left untouched.
The test creates its own inputs and plans, so it passes alone in a fresh process (where its first call is also the
first use of the array on the device) as well as after the rest of the suite.
"""
import numpy as np
import pytest

from workloads import build_workload

pytestmark = pytest.mark.gpu

FWD_TOL = 1e-4     # x |F(0)|, the forward bar of tests/test_gpu_parity.py


@pytest.fixture(scope="module")
def dm():
    import torch
    import paper_2303_10440_b200 as dm
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    dm.load_library()
    return dm


def _inputs(w):
    import torch
    v = torch.as_tensor(np.ascontiguousarray(w.vertices, dtype=np.float32), device="cuda")
    f = torch.as_tensor(np.ascontiguousarray(w.faces, dtype=np.int32), device="cuda")
    return v, f


def _plan_forward(dm, w, mode, v, f, robust):
    plan = dm.Plan(w.n, w.spacing, w.origin, mode, f, w.vertices.shape[0])
    if robust:
        plan.set_option(dm.DM_OPT_FORWARD_PATH, 1)
    F = plan.mesh_ft_forward(v).cpu().numpy()
    plan.close()
    return F


def test_noalloc_forward_matches_plan_forward_on_two_calls_in_a_row(dm):
    import torch

    w_big, w_small = build_workload(2), build_workload(1)
    assert w_small.faces.shape[0] < w_big.faces.shape[0] <= dm.DM_NOALLOC_MAX_FACES
    cases = [(w_big, dm.DM_SURFACE), (w_small, dm.DM_VOLUME)]
    inputs = [_inputs(w) for w, _ in cases]
    # the caller owns the outputs; poison them so that an entry the call failed to write shows up
    outs = [torch.full(w.spectrum_shape, float("nan"), dtype=torch.complex64, device="cuda") for w, _ in cases]

    # two calls back to back on one stream, nothing in between
    for (w, mode), (v, f), out in zip(cases, inputs, outs):
        dm.mesh_ft_forward_noalloc(w.n, w.spacing, mode, v, f, out)
    torch.cuda.synchronize()
    got = [o.cpu().numpy() for o in outs]

    for (w, mode), (v, f), F in zip(cases, inputs, got):
        assert np.isfinite(F).all()
        F_robust = _plan_forward(dm, w, mode, v, f, robust=True)
        assert np.array_equal(F.view(np.float32), F_robust.view(np.float32)), "differs from the plan's robust forward"
        F_fast = _plan_forward(dm, w, mode, v, f, robust=False)
        err = np.abs(F - F_fast).max() / abs(F_fast[0, 0, 0])
        assert err <= FWD_TOL, (w.name, mode, err)

    # the first problem again, after the smaller one used the array: same bits as before
    (w, mode), (v, f) = cases[0], inputs[0]
    again = torch.full(w.spectrum_shape, float("nan"), dtype=torch.complex64, device="cuda")
    dm.mesh_ft_forward_noalloc(w.n, w.spacing, mode, v, f, again)
    assert np.array_equal(again.cpu().numpy().view(np.float32), got[0].view(np.float32))


def test_noalloc_forward_refuses_a_mesh_beyond_its_scratch(dm):
    import torch

    n_faces = dm.DM_NOALLOC_MAX_FACES + 1
    v = torch.zeros((3, 3), dtype=torch.float32, device="cuda")
    f = torch.zeros((n_faces, 3), dtype=torch.int32, device="cuda")
    out = torch.full((8, 8, 5), 7.0, dtype=torch.complex64, device="cuda")
    with pytest.raises(dm.DeltamicError) as e:
        dm.mesh_ft_forward_noalloc((8, 8, 8), (0.125,) * 3, dm.DM_VOLUME, v, f, out)
    assert e.value.code == dm.DM_ERR_TOO_LARGE
    assert "too large" in str(e.value)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())
    # exactly at the limit the call is accepted (degenerate triangles: every pair is zero, F(0) = 0)
    f_ok = f[: dm.DM_NOALLOC_MAX_FACES].contiguous()
    dm.mesh_ft_forward_noalloc((8, 8, 8), (0.125,) * 3, dm.DM_VOLUME, v, f_ok, out)
    torch.cuda.synchronize()
    assert bool((out == 0).all())
