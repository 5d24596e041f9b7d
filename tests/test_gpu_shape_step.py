"""GPU parity of the shape-optimisation step (eq. 17; NEXT 4 of SURVEY.md section 8(f)) against
oracle/shape_step.py: the (I + lambda L)^-2 preconditioner on its own (device conjugate gradients against dense solves),
three consecutive steps on a <= 200-vertex mesh, and ten steps at config 4 whose loss must fall."""
import numpy as np
import pytest

import oracle
from workloads import build_workload

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dm():
    import torch
    import paper_2303_10440_b200 as dm
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    dm.load_library()
    return dm


def _rel(a, b):
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


@pytest.mark.parametrize("cfg,sub", [(1, None), (2, 2), (3, 1)])
def test_preconditioner_against_dense_solves(dm, cfg, sub):
    """One sphere (162 vertices), a perturbed sphere and an aggregate of 8 components (8 zero modes of L)."""
    import torch
    w = build_workload(cfg, subdiv_override=sub, grid_override=(8, 8, 8))
    plan = dm.Plan(w.n, w.spacing, w.origin, w.mode, torch.as_tensor(w.faces, device="cuda"), w.vertices.shape[0])
    g = np.random.default_rng(5).standard_normal(w.vertices.shape).astype(np.float32)
    L = oracle.connectivity_laplacian(w.faces, len(w.vertices))
    for lam in (50.0, 3.0, 0.0):
        st = plan.shape_state(lambda_=lam)
        out = st.precondition(torch.as_tensor(g, device="cuda")).cpu().numpy()
        ref = oracle.precondition(g.astype(np.float64), L, lam)
        err = _rel(out, ref)
        print(f"cfg{cfg} n_V={len(w.vertices)} lambda={lam}: preconditioner rel L2 error {err:.2e}")
        assert err <= 1e-5
        out2 = st.precondition(torch.as_tensor(g, device="cuda")).cpu().numpy()
        assert np.array_equal(out, out2)                     # fixed-order reductions: bitwise reproducible
        it = st.last_cg_iterations()
        print(f"   CG iterations of the two solves: {it}")
        assert all(0 <= i <= 300 for i in it) and (lam > 0 or it == (1, 1) or it == (0, 0) or max(it) <= 1)
        # the multi-launch form of the same solve (used when a mesh does not fit one resident grid): same bits
        st2 = plan.shape_state(lambda_=lam, solver=1)
        out3 = st2.precondition(torch.as_tensor(g, device="cuda")).cpu().numpy()
        assert st2.last_cg_iterations() == (-1, -1)
        assert np.array_equal(out, out3)
        # both forms report the residual they stopped at, and that they converged
        for s_ in (st, st2):
            rel, ok = s_.last_cg_residuals()
            assert ok and all(0.0 <= r <= 1e-7 for r in rel), rel
        assert st.last_cg_residuals() == st2.last_cg_residuals()
        if lam == 50.0:
            # a solve cut short is reported, not hidden: two iterations cannot reach 1e-7 at lambda = 50
            st3 = plan.shape_state(lambda_=lam, cg_max_iter=2)
            st3.precondition(torch.as_tensor(g, device="cuda"))
            rel3, ok3 = st3.last_cg_residuals()
            assert not ok3 and max(rel3) > 1e-7 and st3.last_cg_iterations() == (2, 2)
            st3.close()
        st2.close()
        st.close()
    plan.close()


@pytest.mark.parametrize("banded", [False, True])
@pytest.mark.parametrize("mode", [0, 1])
def test_three_shape_steps_against_the_oracle(dm, mode, banded):
    """``banded``: the step on the narrow band, against the oracle's band branch (pinned by finite
    differences of the banded render in tests/test_oracle_shape.py)."""
    import torch
    w = build_workload(1, grid_override=(24, 24, 24))                 # 162 vertices, 320 triangles
    wt = build_workload(2, subdiv_override=2, grid_override=(24, 24, 24))   # target: a perturbed sphere of radius 0.35
    cov = (np.array([1.2, 1.2, 2.0]) * np.array(w.spacing)) ** 2
    cov = np.array([cov[0], cov[1], cov[2], 0.0, 0.0, 0.0])
    target = oracle.render(wt.vertices, wt.faces, w.n, w.spacing, w.origin, cov, mode)
    plan = dm.Plan(w.n, w.spacing, w.origin, mode, torch.as_tensor(w.faces, device="cuda"), w.vertices.shape[0])
    band = None
    if banded:
        cutoff = 0.05
        k = oracle.frequency_grid(w.n, w.spacing)
        h = np.exp(-0.5 * (cov[0] * k[..., 0] ** 2 + cov[1] * k[..., 1] ** 2 + cov[2] * k[..., 2] ** 2))
        assert np.abs(h / cutoff - 1.0).min() > 1e-3        # no frequency sits on the edge of the band: fp32 and fp64 agree on it
        band = h > cutoff
        assert 0.02 < band.mean() < 0.5
        plan.set_narrow_band(cov, cutoff)
    lr = 2e-3
    st = plan.shape_state(lr=lr)
    ost = oracle.ShapeState()
    prm = oracle.ShapeParams(lr=lr)
    vd = torch.as_tensor(w.vertices, device="cuda").clone()
    td = torch.as_tensor(target.astype(np.float32), device="cuda")
    v_o = w.vertices.astype(np.float64)
    for step in range(3):
        v_before = vd.cpu().numpy().astype(np.float64)
        loss = st.step(vd, td, cov, return_loss=True)
        v_new_o, loss_o = oracle.shape_step(v_o.astype(np.float32), w.faces, w.n, w.spacing, w.origin, cov, mode,
                                            target.astype(np.float32), ost, prm, band=band)
        v_gpu = vd.cpu().numpy().astype(np.float64)
        e_v = _rel(v_gpu, v_new_o)
        e_d = _rel(v_gpu - v_before, v_new_o - v_o.astype(np.float32).astype(np.float64))
        e_l = abs(loss - loss_o) / abs(loss_o)
        print(f"mode {mode} banded {banded} step {step}: vertices rel {e_v:.2e}, displacement rel {e_d:.2e}, Phi_1 rel {e_l:.2e}")
        assert e_v <= 1e-4
        assert e_d <= 5e-3
        assert e_l <= 1e-3
        assert np.abs(v_gpu - v_before).max() <= lr * 1.0001 + 1e-7      # AdamUniform: no coordinate moves more than lr
        v_o = v_new_o
    plan.close()


def test_cfg4_ten_shape_steps_decrease_phi1(dm):
    import torch
    w = build_workload(4)
    wt = build_workload(4, seed_offset=100)
    plan = dm.Plan(w.n, w.spacing, w.origin, w.mode, torch.as_tensor(w.faces, device="cuda"), w.vertices.shape[0])
    target = plan.render(torch.as_tensor(wt.vertices, device="cuda"), w.psf_cov).clone()
    plan.set_narrow_band(w.psf_cov, 0.01)                      # the shape step runs on the narrow band
    st = plan.shape_state(lr=2e-4)
    vd = torch.as_tensor(w.vertices, device="cuda").clone()
    losses = [st.step(vd, target, w.psf_cov, return_loss=True) for _ in range(10)]
    print("cfg4 shape steps, Phi_1:", " ".join(f"{x:.4e}" for x in losses))
    assert np.isfinite(losses).all() and torch.isfinite(vd).all()
    assert losses[-1] < losses[0] and sum(b < a for a, b in zip(losses, losses[1:])) >= 8
    st.close()
    plan.close()


def test_shape_fit_recovers_a_sphere_radius(dm):
    """A miniature of the paper's reconstruction experiment on synthetic data: a sphere of radius 0.22
    fitted, by repeated dm_shape_step calls, to the rendered image of a sphere of radius 0.30 -- the mean radius must move
    most of the way, the mesh must stay round (the preconditioner keeps the update smooth) and Phi_1 must fall."""
    import torch
    from workloads import icosphere
    v0, f = icosphere(2, 0.22)
    vt, _ = icosphere(2, 0.30)
    w = build_workload(1)                                  # grid and PSF of config 1 (32^3, sigma 1,1,2 voxels)
    plan = dm.Plan(w.n, w.spacing, w.origin, 0, torch.as_tensor(f.astype(np.int32), device="cuda"), v0.shape[0])
    target = plan.render(torch.as_tensor(vt.astype(np.float32), device="cuda"), w.psf_cov).clone()
    vd = torch.as_tensor(v0.astype(np.float32), device="cuda").clone()
    st = plan.shape_state(lr=2e-3)
    losses = []
    for it in range(80):
        losses.append(st.step(vd, target, w.psf_cov, return_loss=(it % 10 == 0 or it == 79)))
    r = torch.linalg.norm(vd, dim=1)
    losses = [x for x in losses if x is not None]
    print(f"sphere fit: mean radius 0.22 -> {float(r.mean()):.4f} (target 0.30), spread {float(r.std()):.2e}, "
          f"Phi_1 {losses[0]:.3e} -> {losses[-1]:.3e}")
    assert float(r.mean()) > 0.28 and float(r.std()) < 5e-3
    assert losses[-1] < 0.1 * losses[0]
    st.close()
    plan.close()


def test_psf_fit_with_adam_through_the_autograd_front_end(dm):
    """A miniature of the paper's PSF step (phi_0 = ||u - m||^2, Adam [32] on Sigma): the three variances
    of the PSF fitted to an image rendered with other variances, with torch.optim.Adam driving dm.render's gradient
    w.r.t. the six PSF numbers."""
    import torch
    w = build_workload(1)
    plan = dm.Plan(w.n, w.spacing, w.origin, 0, torch.as_tensor(w.faces, device="cuda"), w.vertices.shape[0])
    v = torch.as_tensor(w.vertices, device="cuda")
    h = np.array(w.spacing)
    cov_true = np.array([(1.6 * h[0]) ** 2, (1.2 * h[1]) ** 2, (2.4 * h[2]) ** 2, 0.0, 0.0, 0.0])
    target = plan.render(v, cov_true).clone()
    s = torch.tensor([1.0, 1.0, 1.0], dtype=torch.float64, requires_grad=True)      # sigma in voxels: cov = (s h)^2
    opt = torch.optim.Adam([s], lr=0.05)
    ht = torch.as_tensor(h)
    first = last = None
    for it in range(120):
        opt.zero_grad()
        cov = torch.cat([(s * ht) ** 2, torch.zeros(3, dtype=torch.float64)]).to(torch.float32)
        loss = ((dm.render(plan, v, cov) - target) ** 2).sum()
        loss.backward()
        opt.step()
        last = float(loss.detach())
        first = last if first is None else first
    got = s.detach().numpy()
    print(f"PSF fit: sigma (voxels) 1,1,1 -> {got.round(3)} (target 1.6, 1.2, 2.4), phi_0 {first:.3e} -> {last:.3e}")
    assert np.abs(got - np.array([1.6, 1.2, 2.4])).max() < 0.1 and last < 1e-2 * first
    plan.close()
