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
        try:
            dv = plan.mesh_ft_backward(vertices, dL_dF)
        finally:   # a failed call must not leave the plan on a partial slab (every later render would be refused)
            plan.set_slab(0, plan.n[0])
    else:  # more ranks than rows: nothing to reduce here
        import torch

        dv = torch.zeros((plan.n_vertices, 3), dtype=torch.float32, device=plan.device)
    return allreduce_vertex_gradient(dv, group)


def allgather_spectrum_slabs(F, group=None, buffers=None):
    """All-gather of the x-slabs of a spectrum tensor F [n_x, n_y, n_z/2+1] (complex or real, CPU or CUDA), in place:
    on entry every rank holds valid rows ``slab_bounds(n_x, world, rank)`` of F, on return every rank holds all rows.
    Needed only when a rank goes on to the inverse FFT.  Slabs differ by at most one row, so they
    are padded to the largest and exchanged with ONE all_gather_into_tensor (<= 68 MB at config 5).
    ``buffers``: a dict the caller keeps between calls; the padded send buffer and the receive buffer (together about twice
    the spectrum) are created in it on first use and reused afterwards, instead of being allocated on every call (inside a
    timed step, at config 5, that is 2 x 68 MB per call).  ``None`` allocates fresh buffers."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return F
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    n_x = F.shape[0]
    rows = max(slab_bounds(n_x, world, r)[1] - slab_bounds(n_x, world, r)[0] for r in range(world))
    Fr = torch.view_as_real(F) if F.is_complex() else F
    key = (tuple(Fr.shape), Fr.dtype, Fr.device, world)
    if buffers is not None and key in buffers:
        send, recv = buffers[key]
    else:
        send = torch.zeros((rows,) + tuple(Fr.shape[1:]), dtype=Fr.dtype, device=Fr.device)   # padding rows stay zero
        recv = torch.empty((world * rows,) + tuple(Fr.shape[1:]), dtype=Fr.dtype, device=Fr.device)
        if buffers is not None:
            buffers[key] = (send, recv)
    b, e = slab_bounds(n_x, world, rank)
    send[: e - b] = Fr[b:e]
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
        try:
            plan.mesh_ft_forward(vertices, out=out)
        finally:   # a failed call must not leave the plan on a partial slab (every later render would be refused)
            plan.set_slab(0, plan.n[0])
    return allgather_spectrum_slabs(out, group, buffers=_plan_gather_buffers(plan)) if gather else out


def _plan_gather_buffers(plan):
    """The dict in which allgather_spectrum_slabs keeps its send / receive buffers for this plan (one pair per spectrum
    shape, dtype, device and world size), so that a loop of sharded forwards allocates them once, not every step."""
    cache = getattr(plan, "_gather_buffers", None)
    if cache is None:
        cache = {}
        try:
            plan._gather_buffers = cache
        except AttributeError:   # a plan type without instance attributes: no caching
            return None
    return cache
