"""Randomised GPU parity sweep: random (seeded) meshes, grids, box lengths, origins, modes, narrow bands and per-face
weights against the oracle on the full grid.  This sweep is what exposed the coarse-mesh regime (DESIGN.md section 6:
thresholds that grow with (|k| h)^3); it stays as a regression net for the regimes the five configs do not reach:
20-triangle spheres, two components of very different resolution, nz = 2, anisotropic boxes, meshes partly outside
the box (the fixed-point turns wrap)."""
import numpy as np
import pytest

import oracle
from workloads import icosphere
from workloads.meshes import perturb_radial

pytestmark = pytest.mark.gpu

FWD_TOL, GRAD_TOL = 1e-4, 1e-3


@pytest.mark.parametrize("seed", [1, 7, 11])
def test_random_meshes_grids_and_modes(seed):
    import torch
    import paper_2303_10440_b200 as dm
    dm.load_library()
    rng = np.random.default_rng(seed)
    for case in range(14):
        sub = int(rng.integers(0, 4))
        c = rng.uniform(-0.3, 0.3, 3)
        v, f = icosphere(sub, rng.uniform(0.05, 0.45), c)
        v = perturb_radial(v, c, 0.08, rng)
        if rng.random() < 0.4:   # stretched, sometimes shifted far outside the box
            v = c + (v - c) * rng.uniform(0.2, 1.5, 3) + rng.uniform(-1.5, 1.5, 3) * (rng.random() < 0.3)
        if rng.random() < 0.3:   # a second component of another resolution
            v2, f2 = icosphere(int(rng.integers(0, 3)), rng.uniform(0.05, 0.2), rng.uniform(-0.4, 0.4, 3))
            f = np.vstack([f, f2 + len(v)])
            v = np.vstack([v, v2])
        v, f = v.astype(np.float32), f.astype(np.int32)
        n = (int(rng.integers(3, 40)), int(rng.integers(3, 40)), 2 * int(rng.integers(1, 20)))
        L = rng.uniform(0.7, 2.0, 3)
        spacing = tuple(L / np.array(n))
        origin = tuple(-L / 2 + rng.uniform(0, 1, 3) * np.array(spacing))
        mode = int(rng.integers(0, 2))
        plan = dm.Plan(n, spacing, origin, mode, torch.as_tensor(f, device="cuda"), v.shape[0])
        k = oracle.frequency_grid(n, spacing).reshape(-1, 3)
        w = None
        if mode == 1 and rng.random() < 0.4:          # membrane densities (positive: |F(0)| stays a meaningful scale)
            w = rng.choice([1.0, 0.5, 2.0], size=len(f)).astype(np.float32)
            plan.set_face_weights(torch.as_tensor(w, device="cuda"))
        inb, edge = np.ones(len(k), bool), np.zeros(len(k), bool)
        if rng.random() < 0.4:
            sig = rng.uniform(0.8, 3.0, 3) * np.array(spacing)
            cov = np.array([sig[0] ** 2, sig[1] ** 2, sig[2] ** 2, 0.2 * sig[0] * sig[1] * rng.uniform(-1, 1),
                            0.2 * sig[0] * sig[2] * rng.uniform(-1, 1), 0.2 * sig[1] * sig[2] * rng.uniform(-1, 1)])
            plan.set_narrow_band(cov, 0.02)
            S = np.array([[cov[0], cov[3], cov[4]], [cov[3], cov[1], cov[5]], [cov[4], cov[5], cov[2]]])
            quad, lim = 0.5 * np.einsum("ni,ij,nj->n", k, S, k), np.log(1 / 0.02)
            inb, edge = quad < lim, np.abs(quad - lim) < 1e-4 * lim
        vd = torch.as_tensor(v, device="cuda")
        F = plan.mesh_ft_forward(vd).cpu().numpy().reshape(-1)
        ref = (oracle.mesh_ft_forward_weighted(v, f, k, mode, w) if w is not None else oracle.mesh_ft_forward(v, f, k, mode))
        sure = inb & ~edge
        tag = (seed, case, len(f), n, mode)
        assert np.abs(F - ref)[sure].max() <= FWD_TOL * abs(ref[0]), tag
        assert (F[~inb & ~edge] == 0).all(), tag
        G = (rng.standard_normal(len(k)) + 1j * rng.standard_normal(len(k))).astype(np.complex64)
        G[edge] = 0
        dv = plan.mesh_ft_backward(vd, torch.as_tensor(G.reshape(n[0], n[1], n[2] // 2 + 1), device="cuda")).cpu().numpy()
        idx = np.nonzero(sure)[0]
        Gs = G[idx].astype(np.complex128)
        dref = (oracle.mesh_ft_backward_weighted(v, f, k[idx], mode, Gs, w) if w is not None
                else oracle.mesh_ft_backward(v, f, k[idx], mode, Gs))
        assert np.isfinite(dv).all(), tag
        assert np.linalg.norm(dv - dref) <= GRAD_TOL * np.linalg.norm(dref), (tag, np.linalg.norm(dv - dref) / np.linalg.norm(dref))
        plan.close()
