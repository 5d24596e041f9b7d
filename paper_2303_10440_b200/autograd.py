"""torch.autograd front end of the C-ABI calls (the renderer is "a differentiable function" of the mesh and
the PSF; :105, :251-253: both are fitted by gradient descent).

Argument marshalling only: `forward` calls dm_mesh_ft_forward / dm_render, `backward` calls dm_mesh_ft_backward /
dm_render_backward through the Plan; no arithmetic of the method happens here.

    F   = mesh_ft(plan, vertices)                 # complex64 [N_x, N_y, N_z/2+1], differentiable w.r.t. vertices
    img = render(plan, vertices, psf_cov)         # float32 [N_x, N_y, N_z], differentiable w.r.t. vertices and psf_cov

`psf_cov` is a float tensor of 6 numbers (xx, yy, zz, xy, xz, yz; host or device).  Its gradient costs a stream
synchronisation (the six numbers come back through host memory, include/deltamic.h); it is only computed when
`psf_cov.requires_grad`.

A plan is mutable, and `backward` runs on whatever state the plan has by then.  `forward` therefore records the plan's
`state_epoch()` and `backward` raises when it has moved (a slab, band, weight or option change in between -- or, under
DM_OPT_REUSE_SPECTRUM, another forward on the same plan): the gradient would silently be that of another function.  Both
functions are once-differentiable: the C ABI has no second derivatives, so a double backward raises instead of returning
numbers that ignore the dependence of the gradient on its inputs.
"""
from __future__ import annotations

import torch
from torch.autograd.function import once_differentiable


def _check_epoch(ctx, what):
    now = ctx.plan.state_epoch()
    if now != ctx.epoch:
        raise RuntimeError(
            f"{what}: the plan changed between forward and backward (state epoch {ctx.epoch} -> {now}: set_slab, "
            "set_narrow_band, set_face_weights or set_option was called, or with DM_OPT_REUSE_SPECTRUM another forward ran "
            "on this plan); the gradient would belong to a different function.  Run forward again after changing the plan.")


class _MeshFT(torch.autograd.Function):
    @staticmethod
    def forward(ctx, plan, vertices):
        v = vertices.detach().contiguous()
        ctx.plan = plan
        ctx.save_for_backward(v)
        out = plan.mesh_ft_forward(v)
        ctx.epoch = plan.state_epoch()
        return out

    @staticmethod
    @once_differentiable
    def backward(ctx, dL_dF):
        (v,) = ctx.saved_tensors
        _check_epoch(ctx, "mesh_ft backward")
        # PyTorch's gradient of a real loss w.r.t. a complex tensor is dL/dRe F + i dL/dIm F: the convention of the C ABI (R14)
        g = dL_dF.to(torch.complex64).contiguous()
        return None, ctx.plan.mesh_ft_backward(v, g)


class _Render(torch.autograd.Function):
    @staticmethod
    def forward(ctx, plan, vertices, psf_cov):
        v = vertices.detach().contiguous()
        cov = [float(x) for x in psf_cov.detach().cpu().reshape(-1)]
        ctx.plan, ctx.cov = plan, cov
        ctx.cov_meta = (psf_cov.dtype, psf_cov.device, tuple(psf_cov.shape))   # not the tensor: nothing to keep alive
        ctx.save_for_backward(v)
        out = plan.render(v, cov)
        ctx.epoch = plan.state_epoch()
        return out

    @staticmethod
    @once_differentiable
    def backward(ctx, dL_dimage):
        (v,) = ctx.saved_tensors
        _check_epoch(ctx, "render backward")
        g = dL_dimage.to(torch.float32).contiguous()
        need_cov = ctx.needs_input_grad[2]
        if need_cov:
            dv, dcov = ctx.plan.render_backward(v, ctx.cov, g, with_psf_grad=True)
            dtype, device, shape = ctx.cov_meta
            dcov = torch.tensor(dcov, dtype=dtype, device=device).reshape(shape)
        else:
            dv, dcov = ctx.plan.render_backward(v, ctx.cov, g), None
        return None, (dv if ctx.needs_input_grad[1] else None), dcov


def mesh_ft(plan, vertices):
    """Differentiable dm_mesh_ft_forward: complex64 spectrum of the mesh on the plan's stored frequency grid."""
    return _MeshFT.apply(plan, vertices)


def render(plan, vertices, psf_cov):
    """Differentiable dm_render: the image of the mesh under the Gaussian PSF of covariance ``psf_cov`` (6 numbers)."""
    if not isinstance(psf_cov, torch.Tensor):
        psf_cov = torch.as_tensor(psf_cov, dtype=torch.float32)
    return _Render.apply(plan, vertices, psf_cov)
