"""World-size-2 (and 3) CPU tests of the sharded path's host logic over gloo.

The CUDA kernels cannot run here, so each rank's slab reduction is computed by the oracle restricted to the rank's rows
(tests may call the oracle); what is under test is the slab partition and the one collective of the sharded backward:
the all-reduced partial gradients must equal the whole-grid gradient, and the slabs of F must tile the whole spectrum.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2303_10440_b200.sharding import (allgather_spectrum_slabs, allreduce_vertex_gradient, sharded_mesh_ft_backward,
                                            sharded_mesh_ft_forward, slab_bounds)


def test_slab_bounds_tile_the_grid():
    for n_x in (1, 2, 5, 32, 128, 205):
        for world in (1, 2, 3, 4, 8, 7, 300):
            rows = []
            for r in range(world):
                b, e = slab_bounds(n_x, world, r)
                assert 0 <= b <= e <= n_x
                rows.extend(range(b, e))
            assert rows == list(range(n_x))
            sizes = [slab_bounds(n_x, world, r)[1] - slab_bounds(n_x, world, r)[0] for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        slab_bounds(8, 2, 2)
    with pytest.raises(ValueError):
        slab_bounds(0, 2, 0)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


class _OraclePlan:
    """Stands in for paper_2303_10440_b200.Plan on CPU (same attributes and calls as sharding.py uses): the slab's rows are
    evaluated by the oracle instead of the CUDA kernels.  What is under test is the host logic of the sharded calls."""

    def __init__(self, w, mode):
        self.w, self.mode = w, mode
        self.n = w.n
        self.spectrum_shape = w.spectrum_shape
        self.n_vertices = w.vertices.shape[0]
        self.device = torch.device("cpu")
        self.slab = (0, w.n[0])
        self.calls = []

    def set_slab(self, b, e):
        self.slab = (b, e)
        self.calls.append(("slab", b, e))

    def _idx(self):
        nx, ny, nz = self.w.n
        nzh = nz // 2 + 1
        return np.arange(self.slab[0] * ny * nzh, self.slab[1] * ny * nzh, dtype=np.int64)

    def mesh_ft_forward(self, vertices, out=None):
        import oracle
        idx = self._idx()
        F = oracle.mesh_ft_forward_grid(vertices.numpy(), self.w.faces, self.w.n, self.w.spacing, self.mode, flat_indices=idx)
        out.view(-1)[torch.as_tensor(idx)] = torch.as_tensor(F).to(out.dtype)
        return out

    def mesh_ft_backward(self, vertices, dL_dF):
        import oracle
        idx = self._idx()
        G = dL_dF.reshape(-1).numpy()[idx].astype(np.complex128)
        dv = oracle.mesh_ft_backward_grid(vertices.numpy(), self.w.faces, self.w.n, self.w.spacing, self.mode, G, flat_indices=idx)
        return torch.as_tensor(np.asarray(dv, dtype=np.float32))


def _worker(rank, world, port, out_dir):
    import oracle
    from workloads import build_workload
    from workloads.configs import spectrum_cotangent

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = build_workload(1, grid_override=(8, 8, 8))        # 320 triangles, 8x8x5 stored frequencies
        nx, ny, nz = w.n
        nzh = nz // 2 + 1
        G = spectrum_cotangent(w).astype(np.complex128)
        b, e = slab_bounds(nx, world, rank)
        idx = np.arange(b * ny * nzh, e * ny * nzh, dtype=np.int64)
        for mode in (0, 1):
            part = oracle.mesh_ft_backward_grid(w.vertices, w.faces, w.n, w.spacing, mode, G.reshape(-1)[idx],
                                                flat_indices=idx) if len(idx) else np.zeros_like(w.vertices, dtype=np.float64)
            dv = torch.as_tensor(np.asarray(part, dtype=np.float64))
            allreduce_vertex_gradient(dv)
            Fslab = oracle.mesh_ft_forward_grid(w.vertices, w.faces, w.n, w.spacing, mode, flat_indices=idx)
            # all-gather of the slabs of F (needed only when one rank runs the inverse FFT)
            Fs = torch.zeros(nx * ny * nzh, dtype=torch.complex128)
            Fs[idx] = torch.as_tensor(Fslab)
            Fr = torch.view_as_real(Fs).clone()
            dist.all_reduce(Fr)
            # ... and through the library's own helper (padded slabs, one all_gather_into_tensor)
            Fg = torch.full((nx, ny, nzh), float("nan"), dtype=torch.complex128)
            Fg[b:e] = torch.as_tensor(Fslab).reshape(e - b, ny, nzh)
            allgather_spectrum_slabs(Fg)
            np.save(os.path.join(out_dir, f"Fg_{mode}_{rank}.npy"), Fg.numpy())
            # ... and the two sharded calls themselves, with the oracle standing in for the kernels
            plan = _OraclePlan(w, mode)
            vt = torch.as_tensor(w.vertices)
            Fs2 = sharded_mesh_ft_forward(plan, vt, out=torch.zeros(w.spectrum_shape, dtype=torch.complex64))
            dv2 = sharded_mesh_ft_backward(plan, vt, torch.as_tensor(G.astype(np.complex64)))
            assert plan.slab == (0, nx)                                     # the plan is handed back on the whole grid
            # a second sharded forward reuses the gather buffers kept on the plan (no per-step allocation), same result
            bufs = {k: (s_.data_ptr(), r_.data_ptr()) for k, (s_, r_) in plan._gather_buffers.items()}
            assert len(bufs) == 1
            Fs3 = sharded_mesh_ft_forward(plan, vt, out=torch.full(w.spectrum_shape, float("nan"), dtype=torch.complex64))
            assert {k: (s_.data_ptr(), r_.data_ptr()) for k, (s_, r_) in plan._gather_buffers.items()} == bufs
            assert torch.equal(Fs3, Fs2)
            # a call that raises still hands the plan back on the whole grid (no collective is pending: it fails before it)
            class _Boom(RuntimeError):
                pass

            def _raise(*a, **k):
                raise _Boom()

            if e > b:
                good_fwd, good_bwd = plan.mesh_ft_forward, plan.mesh_ft_backward
                plan.mesh_ft_forward = plan.mesh_ft_backward = _raise
                for call in (lambda: sharded_mesh_ft_forward(plan, vt, out=torch.zeros(w.spectrum_shape, dtype=torch.complex64), gather=False),
                             lambda: sharded_mesh_ft_backward(plan, vt, torch.as_tensor(G.astype(np.complex64)))):
                    try:
                        call()
                        raise AssertionError("the stand-in kernel call should have raised")
                    except _Boom:
                        pass
                    assert plan.slab == (0, nx)
                plan.mesh_ft_forward, plan.mesh_ft_backward = good_fwd, good_bwd
            np.save(os.path.join(out_dir, f"Fs2_{mode}_{rank}.npy"), Fs2.numpy())
            np.save(os.path.join(out_dir, f"dv2_{mode}_{rank}.npy"), dv2.numpy())
            np.save(os.path.join(out_dir, f"dv_{mode}_{rank}.npy"), dv.numpy())
            np.save(os.path.join(out_dir, f"F_{mode}_{rank}.npy"), torch.view_as_complex(Fr).numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_sharded_backward_allreduce_matches_whole_grid(world, tmp_path):
    import oracle
    from workloads import build_workload
    from workloads.configs import spectrum_cotangent

    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    w = build_workload(1, grid_override=(8, 8, 8))
    G = spectrum_cotangent(w).astype(np.complex128)
    for mode in (0, 1):
        ref = oracle.mesh_ft_backward_grid(w.vertices, w.faces, w.n, w.spacing, mode, G)
        Fref = oracle.mesh_ft_forward_grid(w.vertices, w.faces, w.n, w.spacing, mode).reshape(-1)
        for r in range(world):
            dv = np.load(tmp_path / f"dv_{mode}_{r}.npy")
            assert np.linalg.norm(dv - ref) <= 1e-12 * np.linalg.norm(ref)
            F = np.load(tmp_path / f"F_{mode}_{r}.npy")
            assert np.abs(F - Fref).max() <= 1e-12 * abs(Fref[0])
            Fg = np.load(tmp_path / f"Fg_{mode}_{r}.npy").reshape(-1)
            assert np.isfinite(Fg).all() and np.abs(Fg - Fref).max() <= 1e-12 * abs(Fref[0])
            Fs2 = np.load(tmp_path / f"Fs2_{mode}_{r}.npy").reshape(-1)
            assert np.abs(Fs2 - Fref).max() <= 1e-6 * abs(Fref[0])          # complex64 storage
            dv2 = np.load(tmp_path / f"dv2_{mode}_{r}.npy")
            assert np.linalg.norm(dv2 - ref) <= 1e-6 * np.linalg.norm(ref)  # float32 partial gradients
