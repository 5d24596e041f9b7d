"""Host-side contract of the torch.autograd front end (paper_2303_10440_b200/autograd.py), checked on CPU with a stand-in
plan: the two Functions only marshal, so what can be tested without a GPU is their bookkeeping -- a backward after the plan
changed raises instead of returning the gradient of another function, a double backward raises, and the PSF tensor is not
kept alive by the graph.  (The numbers are covered by the -m gpu tests; the stand-in below computes nothing of the method.)"""
import gc
import weakref

import pytest
import torch

from paper_2303_10440_b200 import autograd as ag


class _FakePlan:
    """Duck-typed Plan: linear toy maps on CPU tensors plus the state_epoch protocol of _binding.Plan."""

    def __init__(self):
        self.config, self.forwards, self.reuse = 0, 0, False

    def state_epoch(self):
        return (self.config, self.forwards if self.reuse else None)

    def mesh_ft_forward(self, v):
        self.forwards += 1
        return (2.0 * v).sum(dim=1).to(torch.complex64)

    def mesh_ft_backward(self, v, g):
        return 2.0 * g.real.to(torch.float32)[:, None].expand(-1, 3).contiguous()

    def render(self, v, cov):
        self.forwards += 1
        return 3.0 * v[:, 0] * sum(cov)

    def render_backward(self, v, cov, g, with_psf_grad=False):
        dv = torch.zeros_like(v)
        dv[:, 0] = 3.0 * g * sum(cov)
        return (dv, [float((3.0 * v[:, 0] * g).sum())] * 6) if with_psf_grad else dv


def test_backward_raises_when_the_plan_changed_since_forward():
    plan = _FakePlan()
    v = torch.randn(5, 3, requires_grad=True)
    F = ag.mesh_ft(plan, v)
    (g,) = torch.autograd.grad(F.real.sum(), v, retain_graph=True)       # unchanged plan: fine
    assert torch.allclose(g, torch.full_like(g, 2.0))
    plan.config += 1                                                      # e.g. set_narrow_band between the two passes
    with pytest.raises(RuntimeError, match="plan changed between forward and backward"):
        torch.autograd.grad(F.real.sum(), v)
    # another forward on the same plan is harmless by default ...
    cov = torch.tensor([1.0, 2.0, 3.0, 0.0, 0.0, 0.0], requires_grad=True)
    img = ag.render(plan, v, cov)
    ag.render(plan, v.detach(), cov.detach())
    gv, gc_ = torch.autograd.grad(img.sum(), (v, cov))
    assert gc_.shape == cov.shape and gc_.dtype == cov.dtype
    # ... but not when the backward takes its spectrum from the last render (DM_OPT_REUSE_SPECTRUM)
    plan.reuse = True
    img = ag.render(plan, v, cov)
    ag.render(plan, v.detach(), cov.detach())
    with pytest.raises(RuntimeError, match="plan changed between forward and backward"):
        img.sum().backward()


def test_double_backward_raises():
    plan = _FakePlan()
    v = torch.randn(4, 3, requires_grad=True)
    img = ag.render(plan, v, torch.ones(6))
    (g,) = torch.autograd.grad((img ** 2).sum(), v, create_graph=True)
    with pytest.raises(RuntimeError, match="once_differentiable"):
        g.sum().backward()


def test_psf_tensor_is_not_kept_alive_by_the_graph():
    plan = _FakePlan()
    v = torch.randn(4, 3, requires_grad=True)
    cov = torch.ones(6)
    ref = weakref.ref(cov)
    img = ag.render(plan, v, cov)
    del cov
    gc.collect()
    assert ref() is None
    img.sum().backward()
    assert v.grad is not None


def test_plan_state_epoch_moves_with_every_setter():
    """The real Plan's bookkeeping, without a device: the setters bump the epoch before they reach the library."""
    import paper_2303_10440_b200._binding as b
    src = open(b.__file__).read()
    for name in ("set_slab", "set_face_weights", "update_face_weights", "set_narrow_band", "set_option"):
        body = src[src.index(f"    def {name}("):]
        body = body[:body.index("\n    def ", 1)]
        assert "self._config_epoch += 1" in body, name
        assert body.index("self._config_epoch += 1") < body.index("_check("), name
    for name in ("mesh_ft_forward", "render"):
        body = src[src.index(f"    def {name}("):]
        body = body[:body.index("\n    def ", 1)]
        assert "self._forward_epoch += 1" in body, name
