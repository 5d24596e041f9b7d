"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (default plan options).

The oracle cannot run configs 3-5 in full, so parity is taken on the sampled set S of stored
frequencies (all |n_a| <= 4, the three axes, random entries on each Nyquist plane, uniform random entries):
  forward   max over S of |F_gpu - F_oracle| <= 1e-4 |F(0)|, the GPU spectrum computed on the WHOLE grid;
  backward  the GPU backward runs on the whole grid with a cotangent that is N(0,1)+iN(0,1) on S and zero elsewhere
            (the backward is linear in G), compared with the oracle's gradient summed over S: relative L2 <= 1e-3;
plus properties that hold at any size (Hermitian symmetry inside the stored grid, fast kernels against the robust
kernels over the whole grid, run-to-run reproducibility).
"""
import numpy as np
import pytest

import oracle
from workloads import build_workload, sampled_frequencies

pytestmark = pytest.mark.gpu

FWD_TOL = 1e-4
GRAD_TOL = 1e-3


@pytest.fixture(scope="module")
def dm():
    import torch
    import paper_2303_10440_b200 as dm
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    dm.load_library()
    return dm


def _setup(dm, cfg):
    import torch
    w = build_workload(cfg)
    plan = dm.Plan(w.n, w.spacing, w.origin, w.mode, torch.as_tensor(w.faces, device="cuda"), w.vertices.shape[0])
    return w, plan, torch.as_tensor(w.vertices, device="cuda")


def _rel_l2(a, b):
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


@pytest.mark.parametrize("cfg", [2, 3, 4, 5])
def test_forward_sampled_frequencies(dm, cfg, report):
    w, plan, vd = _setup(dm, cfg)
    F = plan.mesh_ft_forward(vd).cpu().numpy()
    assert np.isfinite(F.view(np.float32)).all()
    idx = sampled_frequencies(w, n_random=2048 if cfg < 5 else 1024)
    ref = oracle.mesh_ft_forward_grid(w.vertices, w.faces, w.n, w.spacing, w.mode, flat_indices=idx)
    f0 = abs(oracle.mesh_ft_forward_grid(w.vertices, w.faces, w.n, w.spacing, w.mode, flat_indices=np.array([0]))[0])
    err = np.abs(F.reshape(-1)[idx] - ref).max() / f0
    report(f"cfg{cfg} forward: max|dF|/|F(0)| = {err:.2e} over {len(idx)} sampled frequencies")
    assert err <= FWD_TOL, err
    # F(-kx,-ky,0) = conj F(kx,ky,0) inside the stored grid (any size; pin P3)
    nx, ny = w.n[0], w.n[1]
    P = F[:, :, 0]
    Pm = np.conj(P[(-np.arange(nx)) % nx][:, (-np.arange(ny)) % ny])
    interior = np.ones((nx, ny), bool)
    interior[nx // 2, :] = False   # Nyquist rows have no stored partner
    interior[:, ny // 2] = False
    assert np.abs(P - Pm)[interior].max() <= 2 * FWD_TOL * f0
    plan.close()


@pytest.mark.parametrize("cfg", [2, 3, 4, 5])
def test_backward_sampled_frequencies(dm, cfg, report):
    import torch
    w, plan, vd = _setup(dm, cfg)
    idx = sampled_frequencies(w, n_random=768 if cfg < 5 else 384, n_nyquist=32)
    rng = np.random.default_rng(2000 + cfg)
    Gs = (rng.standard_normal(len(idx)) + 1j * rng.standard_normal(len(idx))).astype(np.complex64)
    G = np.zeros(w.n_k, dtype=np.complex64)
    G[idx] = Gs
    Gd = torch.as_tensor(G.reshape(w.spectrum_shape), device="cuda")
    dv = plan.mesh_ft_backward(vd, Gd).cpu().numpy()
    assert np.isfinite(dv).all()
    ref = oracle.mesh_ft_backward_grid(w.vertices, w.faces, w.n, w.spacing, w.mode, Gs.astype(np.complex128),
                                       flat_indices=idx)
    err = _rel_l2(dv, ref)
    report(f"cfg{cfg} backward: rel L2 = {err:.2e} over {len(idx)} sampled frequencies")
    assert err <= GRAD_TOL, err
    plan.close()


@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_fast_kernels_match_robust_kernels_whole_grid(dm, cfg, report):
    """Every (triangle, frequency) pair of the full config: the fast kernels against the kernels that send every pair
    through the series / far-pair branches (which the tests of test_gpu_parity.py tie to the oracle).  Config 5 is the only
    one on the SEG = 16 instantiation of the fast backward kernel (72 < n_z/2+1 = 129 <= 144)."""
    import torch
    from workloads.configs import spectrum_cotangent
    w, plan, vd = _setup(dm, cfg)
    Gd = torch.as_tensor(spectrum_cotangent(w), device="cuda")
    F = plan.mesh_ft_forward(vd).clone()
    dv = plan.mesh_ft_backward(vd, Gd).clone()
    dv2 = plan.mesh_ft_backward(vd, Gd)
    assert torch.equal(dv, dv2)                      # atomic-free: bitwise reproducible (reading R22)
    plan.set_option(dm.DM_OPT_FORWARD_PATH, 1)
    plan.set_option(dm.DM_OPT_BACKWARD_PATH, 1)
    Fr = plan.mesh_ft_forward(vd)
    dvr = plan.mesh_ft_backward(vd, Gd)
    f0 = float(Fr[0, 0, 0].abs())
    ferr = float((F - Fr).abs().max()) / f0
    gerr = float(torch.linalg.norm(dv - dvr) / torch.linalg.norm(dvr))
    report(f"cfg{cfg} fast vs robust over the whole grid: forward {ferr:.2e} |F(0)|, gradient rel L2 {gerr:.2e}")
    assert ferr <= 0.5 * FWD_TOL
    assert gerr <= 0.5 * GRAD_TOL
    plan.close()


def test_cfg3_complete_x_rows_against_the_oracle(dm, report):
    """Config 3 (40 960 triangles, 128 x 128 x 64) against the oracle on EVERY stored frequency of complete x-rows -- rows 0..15
    (the low frequencies, where the series branches live), the Nyquist row and the last row (n_x = -1): 18 x 4224 frequencies,
    about a minute of oracle time -- instead of a sample; and the backward with a cotangent that lives on three complete rows
    (the oracle's backward costs about five times its forward per frequency)."""
    import torch
    w, plan, vd = _setup(dm, 3)
    nx, ny, nzh = w.spectrum_shape
    F = plan.mesh_ft_forward(vd).cpu().numpy()
    rows = list(range(16)) + [nx // 2, nx - 1]
    per_row = ny * nzh
    idx = np.concatenate([np.arange(r * per_row, (r + 1) * per_row, dtype=np.int64) for r in rows])
    ref = oracle.mesh_ft_forward_grid(w.vertices, w.faces, w.n, w.spacing, w.mode, flat_indices=idx)
    f0 = abs(ref[0])
    err_rows = np.abs(F.reshape(-1)[idx] - ref).reshape(len(rows), per_row).max(axis=1) / f0
    report(f"cfg3 forward, complete x-rows {rows[0]}..{rows[15]}, {rows[16]}, {rows[17]} ({len(idx)} frequencies): "
           f"max|dF|/|F(0)| = {err_rows.max():.2e} (worst row {rows[int(err_rows.argmax())]})")
    assert err_rows.max() <= FWD_TOL, err_rows
    brows = [0, 1, nx // 2]
    bidx = np.concatenate([np.arange(r * per_row, (r + 1) * per_row, dtype=np.int64) for r in brows])
    rng = np.random.default_rng(3003)
    Gs = (rng.standard_normal(len(bidx)) + 1j * rng.standard_normal(len(bidx))).astype(np.complex64)
    G = np.zeros(w.n_k, dtype=np.complex64)
    G[bidx] = Gs
    dv = plan.mesh_ft_backward(vd, torch.as_tensor(G.reshape(w.spectrum_shape), device="cuda")).cpu().numpy()
    dref = oracle.mesh_ft_backward_grid(w.vertices, w.faces, w.n, w.spacing, w.mode, Gs.astype(np.complex128), flat_indices=bidx)
    gerr = _rel_l2(dv, dref)
    report(f"cfg3 backward, cotangent on the complete x-rows {brows} ({len(bidx)} frequencies): rel L2 = {gerr:.2e}")
    assert gerr <= GRAD_TOL, gerr
    plan.close()


def test_cfg4_gradient_descent_decreases_loss(dm):
    """Config 4's workload: 10 consecutive gradient steps on the vertices with lr 1e-3 on L = sum (u - m)^2, m the
    render of the target mesh (seed + 100, reading R16); the loss must go down monotonically."""
    import torch
    w, plan, vd = _setup(dm, 4)
    wt = build_workload(4, seed_offset=100)
    assert wt.faces.shape == w.faces.shape
    target = plan.render(torch.as_tensor(wt.vertices, device="cuda"), w.psf_cov).clone()
    v = vd.clone()
    losses = []
    for _ in range(10):
        img = plan.render(v, w.psf_cov)
        diff = img - target
        losses.append(float((diff * diff).sum()))
        dv = plan.render_backward(v, w.psf_cov, 2.0 * diff)
        # lr 1e-3 on a gradient normalised by its largest entry (the raw scale depends on the voxel volume)
        v = v - 1e-3 * dv / dv.abs().max()
    print("cfg4 GD losses:", " ".join(f"{x:.4e}" for x in losses))
    assert all(b < a for a, b in zip(losses, losses[1:])), losses
    plan.close()
