"""Pins P10 (erf box render) and P11 (adjoint of PSF multiply + inverse rFFT) for oracle/render.py."""
import numpy as np
import pytest
from scipy.special import erf

import oracle
from workloads import box_mesh, icosphere


def test_P10_blurred_box_matches_erf_closed_form():
    """u = 1_box * Gaussian: prod_a 1/2 [erf((x-c+h)/(sqrt2 s)) - erf((x-c-h)/(sqrt2 s))], periodised.
    Pins R5 (Sigma not Sigma^-1 in h_hat), R9/R11 (origin, 1/h^3 scale), R12 (sigma in voxels)."""
    n = (32, 40, 24)
    spacing = (1 / 32, 1 / 40, 1 / 24)
    origin = tuple(-0.5 + 0.5 * h for h in spacing)
    sig_vox = np.array([2.0, 2.5, 2.0])
    sig = sig_vox * np.array(spacing)
    cov = [sig[0] ** 2, sig[1] ** 2, sig[2] ** 2, 0, 0, 0]
    c = np.array([0.04, -0.06, 0.02])
    hw = np.array([0.17, 0.12, 0.2])
    v, f = box_mesh(c, hw)
    img = oracle.render(v, f, n, spacing, origin, cov, 0)
    prof = []
    for a in range(3):
        x = origin[a] + np.arange(n[a]) * spacing[a]
        p = np.zeros_like(x)
        for img_shift in (-2, -1, 0, 1, 2):                       # periodic images of the box
            xa = x - c[a] - img_shift * 1.0
            p += 0.5 * (erf((xa + hw[a]) / (np.sqrt(2) * sig[a])) - erf((xa - hw[a]) / (np.sqrt(2) * sig[a])))
        prof.append(p)
    ref = prof[0][:, None, None] * prof[1][None, :, None] * prof[2][None, None, :]
    assert np.abs(img - ref).max() < 1e-8 * ref.max()
    assert ref.max() > 0.9                                            # inside value ~1 (R11 scale)
    assert img.sum() * np.prod(spacing) == pytest.approx(8 * np.prod(hw), rel=1e-12)   # mass = volume


def test_P10_full_covariance_is_rotated_diagonal():
    """A rotated PSF on a rotated-by-symmetry problem: xy covariance swaps with a 90-degree turn of the sphere grid."""
    n = (16, 16, 16)
    spacing = (1 / 16,) * 3
    origin = (-0.5 + 1 / 32,) * 3
    v, f = icosphere(2, 0.25)
    cov_a = [6e-2, 4e-2, 5e-2, 1e-2, 0.0, 0.0]        # wide enough that Nyquist-plane content (R13) is < 1e-16:
    # smallest eigenvalue 0.036, k_Nyquist = 16 pi => exp(-45)
    img_a = oracle.render(v, f, n, spacing, origin, cov_a, 0)
    # rotate mesh and PSF by 90 degrees about z: (x,y) -> (-y,x); Sigma' = R Sigma R^T
    R = np.array([[0.0, -1.0, 0.0], [1.0, 0.0, 0.0], [0.0, 0.0, 1.0]])
    Sa = np.array([[6e-2, 1e-2, 0], [1e-2, 4e-2, 0], [0, 0, 5e-2]])
    Sb = R @ Sa @ R.T
    cov_b = [Sb[0, 0], Sb[1, 1], Sb[2, 2], Sb[0, 1], Sb[0, 2], Sb[1, 2]]
    img_b = oracle.render(v @ R.T, f, n, spacing, origin, cov_b, 0)
    # voxel (i,j) of image b sits at (x,y) = R (x',y'): x = -y', y = x'  => b[i,j] = a[j, N-1-i]
    assert np.abs(img_b - np.rot90(img_a, k=1, axes=(0, 1))).max() < 1e-12


def test_P11_adjoint_identity_and_torch_autograd():
    n = (6, 8, 10)
    spacing = (0.1, 0.12, 0.09)
    origin = (-0.25, -0.4, -0.41)
    cov = [0.02, 0.015, 0.03, 0.004, -0.003, 0.002]
    rng = np.random.default_rng(0)
    shp = (n[0], n[1], n[2] // 2 + 1)
    F = rng.standard_normal(shp) + 1j * rng.standard_normal(shp)
    y = rng.standard_normal(n)
    img = oracle.spectrum_to_image(F, n, spacing, origin, cov)
    G = oracle.image_to_spectrum_cotangent(y, n, spacing, origin, cov)
    lhs = float((img * y).sum())
    rhs = float(np.sum(G.real * F.real + G.imag * F.imag))
    assert lhs == pytest.approx(rhs, rel=1e-12)
    torch = pytest.importorskip("torch")
    c = torch.from_numpy(oracle.psf_shift_spectrum(n, spacing, origin, cov))
    Ft = torch.from_numpy(F).requires_grad_(True)
    out = torch.fft.irfftn(Ft * c, s=n, dim=(0, 1, 2))
    (out * torch.from_numpy(y)).sum().backward()
    # torch's complex gradient convention is dL/dRe + i dL/dIm (reading R14)
    assert np.abs(Ft.grad.numpy() - G).max() < 1e-14 * max(1.0, np.abs(G).max())


def test_render_backward_vs_finite_differences_through_the_whole_render():
    n = (8, 8, 8)
    spacing = (1 / 8,) * 3
    origin = (-0.5 + 1 / 16,) * 3
    cov = [(1.2 / 8) ** 2, (1.2 / 8) ** 2, (1.5 / 8) ** 2, 0, 0, 0]
    v, f = icosphere(0, 0.3, (0.02, 0.01, -0.03))
    rng = np.random.default_rng(5)
    y = rng.standard_normal(n)
    for mode in (0, 1):
        grad = oracle.render_backward(v, f, n, spacing, origin, cov, mode, y)
        fd = np.zeros_like(v)
        h = 1e-6
        for i in range(v.shape[0]):
            for d in range(3):
                vp, vm = v.copy(), v.copy()
                vp[i, d] += h
                vm[i, d] -= h
                fd[i, d] = ((oracle.render(vp, f, n, spacing, origin, cov, mode) * y).sum()
                            - (oracle.render(vm, f, n, spacing, origin, cov, mode) * y).sum()) / (2 * h)
        assert np.linalg.norm(grad - fd) / np.linalg.norm(fd) < 1e-7


def test_psf_gradient_vs_finite_differences_of_the_render():
    """NEXT 2: dL/dSigma of the oracle against central differences of its own render in each
    of the six covariance entries, with a full (non-diagonal) covariance and an anisotropic grid."""
    n = (8, 10, 12)
    spacing = (1 / 8, 1 / 10, 1 / 6)
    origin = tuple(-0.5 * nn * h + 0.5 * h for nn, h in zip(n, spacing))
    cov = np.array([0.020, 0.028, 0.045, 0.004, -0.006, 0.009])
    v, f = icosphere(1, 0.3, (0.02, 0.01, -0.03))
    y = np.random.default_rng(11).standard_normal(n)
    for mode in (0, 1):
        grad = oracle.render_backward_psf(v, f, n, spacing, origin, cov, mode, y)
        fd = np.zeros(6)
        for m in range(6):
            h = 1e-6
            cp, cm = cov.copy(), cov.copy()
            cp[m] += h
            cm[m] -= h
            fd[m] = ((oracle.render(v, f, n, spacing, origin, cp, mode) * y).sum()
                     - (oracle.render(v, f, n, spacing, origin, cm, mode) * y).sum()) / (2 * h)
        assert np.abs(grad - fd).max() <= 1e-7 * np.abs(fd).max(), (mode, grad, fd)


def test_psf_gradient_of_total_intensity_is_zero_and_blur_lowers_peak():
    """Closed-form checks: sum(image) = F(0)/voxel does not depend on Sigma (k = 0 has zero weight), so dL/dSigma = 0 for
    L = sum(image); and for L = image at the centre voxel of a small blob more blur lowers the peak: dL/dSigma_aa < 0."""
    n = (12, 12, 12)
    spacing = (1 / 12,) * 3
    origin = (-0.5 + 1 / 24,) * 3
    cov = [(1.5 / 12) ** 2] * 3 + [0, 0, 0]
    v, f = icosphere(1, 0.12, (1 / 24, 1 / 24, 1 / 24))
    g = oracle.render_backward_psf(v, f, n, spacing, origin, cov, 0, np.ones(n))
    img = oracle.render(v, f, n, spacing, origin, cov, 0)
    assert np.abs(g).max() <= 1e-9 * np.abs(img).sum()
    y = np.zeros(n)
    y[6, 6, 6] = 1.0
    g = oracle.render_backward_psf(v, f, n, spacing, origin, cov, 0, y)
    assert (g[:3] < 0).all()
