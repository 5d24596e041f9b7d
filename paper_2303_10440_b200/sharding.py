"""x-slab sharding of the mesh FT over ranks.

Host logic only: which rows of the stored spectrum a rank owns, and the ONE exchange step of the sharded backward
(an all-reduce of the partial dL/dvertices).  The kernels restrict themselves to a slab through
``Plan.set_slab`` (dm_plan_set_slab).  Works with any ``torch.distributed`` backend (NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations


def slab_bounds(n_x: int, world_size: int, rank: int) -> tuple[int, int]:
    """Rows [ix_begin, ix_end) of the stored spectrum owned by ``rank``: contiguous, disjoint, covering [0, n_x),
    sizes differing by at most one (the first ``n_x % world_size`` ranks hold the extra row).  A rank may own an
    empty slab when world_size > n_x."""
    if n_x <= 0 or world_size <= 0 or not (0 <= rank < world_size):
        raise ValueError(f"bad slab request n_x={n_x} world_size={world_size} rank={rank}")
    base, extra = divmod(n_x, world_size)
    begin = rank * base + min(rank, extra)
    return begin, begin + base + (1 if rank < extra else 0)


def allreduce_vertex_gradient(partial_dv, group=None):
    """Sum the per-slab partial dL/dvertices over ranks in place (the backward's only collective: 3 n_V floats)."""
    import torch.distributed as dist

    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(partial_dv, op=dist.ReduceOp.SUM, group=group)
    return partial_dv


def sharded_mesh_ft_backward(plan, vertices, dL_dF, group=None):
    """dL/dvertices with the stored spectrum sharded over the ranks of ``group`` by x-slab: every rank reduces its
    own rows in the CUDA kernels, then one all-reduce sums the partial gradients.  Every rank gets the full result."""
    import torch.distributed as dist

    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    begin, end = slab_bounds(plan.n[0], world, rank)
    if end > begin:
        plan.set_slab(begin, end)
        dv = plan.mesh_ft_backward(vertices, dL_dF)
        plan.set_slab(0, plan.n[0])
    else:  # more ranks than rows: nothing to reduce here
        import torch

        dv = torch.zeros((plan.n_vertices, 3), dtype=torch.float32, device=plan.device)
    return allreduce_vertex_gradient(dv, group)


def allgather_spectrum_slabs(F, group=None):
    """All-gather of the x-slabs of a spectrum tensor F [n_x, n_y, n_z/2+1] (complex or real, CPU or CUDA), in place:
    on entry every rank holds valid rows ``slab_bounds(n_x, world, rank)`` of F, on return every rank holds all rows.
    Needed only when a rank goes on to the inverse FFT.  Slabs differ by at most one row, so they
    are padded to the largest and exchanged with ONE all_gather_into_tensor (<= 68 MB at config 5)."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return F
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    n_x = F.shape[0]
    rows = max(slab_bounds(n_x, world, r)[1] - slab_bounds(n_x, world, r)[0] for r in range(world))
    Fr = torch.view_as_real(F) if F.is_complex() else F
    send = torch.zeros((rows,) + tuple(Fr.shape[1:]), dtype=Fr.dtype, device=Fr.device)
    b, e = slab_bounds(n_x, world, rank)
    send[: e - b] = Fr[b:e]
    recv = torch.empty((world * rows,) + tuple(Fr.shape[1:]), dtype=Fr.dtype, device=Fr.device)
    dist.all_gather_into_tensor(recv, send, group=group)
    for r in range(world):
        rb, re_ = slab_bounds(n_x, world, r)
        if r != rank and re_ > rb:
            Fr[rb:re_] = recv[r * rows: r * rows + (re_ - rb)]
    return F


def sharded_mesh_ft_forward(plan, vertices, out=None, group=None, gather=True):
    """F with the stored spectrum sharded over the ranks of ``group`` by x-slab: every rank evaluates its own rows in the
    CUDA kernels (no communication: the frequencies are independent); with ``gather`` the slabs are then all-gathered so
    that every rank holds the whole spectrum."""
    import torch
    import torch.distributed as dist

    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    begin, end = slab_bounds(plan.n[0], world, rank)
    if out is None:
        out = torch.zeros(plan.spectrum_shape, dtype=torch.complex64, device=plan.device)
    if end > begin:
        plan.set_slab(begin, end)
        plan.mesh_ft_forward(vertices, out=out)
        plan.set_slab(0, plan.n[0])
    return allgather_spectrum_slabs(out, group) if gather else out
