"""Image-formation reference around the mesh FT (step O7) -- TEST INFRASTRUCTURE, numpy fp64.

  image = irfftn( F . h_hat . exp(+i k.x0), s=N ) / (h_x h_y h_z)           PAPER.md:83-89 eq. 1-2
  h_hat(k) = exp(-1/2 k^T Sigma k)    (eq. 4 prints Sigma^-1; reading R5: the FT of the
                                       Gaussian of covariance Sigma in eq. 3 has Sigma, h_hat(0)=1)
  x0 = sample point of voxel (0,0,0) (readings R9, R11).  Sigma is given as (xx,yy,zz,xy,xz,yz) in
  physical units (R12: sigma_phys = sigma_vox * h per axis).

The inverse transform is numpy/pocketfft's irfftn, which *defines* the treatment of the self-conjugate
planes of a not-exactly-Hermitian half spectrum (reading R13).
"""
from __future__ import annotations

import numpy as np

from .mesh_ft import frequency_grid


def _cov_matrix(psf_cov) -> np.ndarray:
    xx, yy, zz, xy, xz, yz = (float(v) for v in psf_cov)
    return np.array([[xx, xy, xz], [xy, yy, yz], [xz, yz, zz]], dtype=np.float64)


def psf_shift_spectrum(n, spacing, origin, psf_cov) -> np.ndarray:
    """c(k) = h_hat(k) exp(+i k.x0) / (h_x h_y h_z) on the stored half spectrum, complex128."""
    k = frequency_grid(n, spacing)
    S = _cov_matrix(psf_cov)
    quad = np.einsum("...i,ij,...j->...", k, S, k)
    phase = k @ np.asarray(origin, dtype=np.float64)
    return np.exp(-0.5 * quad) * np.exp(1j * phase) / float(np.prod(np.asarray(spacing, dtype=np.float64)))


def spectrum_to_image(F, n, spacing, origin, psf_cov) -> np.ndarray:
    """image [N_x,N_y,N_z] float64 from the mesh spectrum F [N_x,N_y,N_z/2+1]."""
    n = tuple(int(v) for v in n)
    S = np.asarray(F, dtype=np.complex128) * psf_shift_spectrum(n, spacing, origin, psf_cov)
    return np.fft.irfftn(S, s=n, axes=(0, 1, 2))


def image_to_spectrum_cotangent(dL_dimage, n, spacing, origin, psf_cov) -> np.ndarray:
    """G = dL/dRe F + i dL/dIm F for every stored entry (reading R14).

    Adjoint of irfftn on independent stored entries: dL/dS = (w/N_tot) rfftn(dL/dimage) with w = 1 on
    the planes n_z = 0 and n_z = N_z/2, else 2; then G = conj(c) dL/dS.
    """
    n = tuple(int(v) for v in n)
    g = np.asarray(dL_dimage, dtype=np.float64).reshape(n)
    dS = np.fft.rfftn(g, axes=(0, 1, 2)) / float(np.prod(n))
    w = np.full(n[2] // 2 + 1, 2.0)
    w[0] = 1.0
    if n[2] % 2 == 0:
        w[-1] = 1.0
    dS = dS * w[None, None, :]
    return np.conj(psf_shift_spectrum(n, spacing, origin, psf_cov)) * dS


def render(vertices, faces, n, spacing, origin, psf_cov, mode: int) -> np.ndarray:
    from .mesh_ft import mesh_ft_forward_grid
    F = mesh_ft_forward_grid(vertices, faces, n, spacing, mode)
    return spectrum_to_image(F, n, spacing, origin, psf_cov)


def render_backward(vertices, faces, n, spacing, origin, psf_cov, mode: int, dL_dimage) -> np.ndarray:
    from .mesh_ft import mesh_ft_backward_grid
    G = image_to_spectrum_cotangent(dL_dimage, n, spacing, origin, psf_cov)
    return mesh_ft_backward_grid(vertices, faces, n, spacing, mode, G)


def render_backward_psf(vertices, faces, n, spacing, origin, psf_cov, mode: int, dL_dimage) -> np.ndarray:
    """dL/dSigma as 6 numbers in the order of ``psf_cov`` (xx, yy, zz, xy, xz, yz), the off-diagonal entries being the
    derivative with respect to the ONE number that fills both symmetric positions of Sigma (the
    PSF parameters are optimised by gradient descent; eq. 4 with reading R5).

    With S = F c, c = exp(-1/2 k^T Sigma k) e^{i k.x0}/(h_x h_y h_z):  dS/dSigma_aa = -1/2 k_a^2 S,
    dS/dSigma_ab = -k_a k_b S (a != b), and dL/dS = (w/N_tot) rfftn(dL/dimage) on independent stored entries
    (reading R14), so  dL/dSigma_m = sum_k Re( conj(dL/dS) dS/dSigma_m ).
    """
    from .mesh_ft import mesh_ft_forward_grid
    n = tuple(int(v) for v in n)
    F = mesh_ft_forward_grid(vertices, faces, n, spacing, mode)
    S = np.asarray(F, dtype=np.complex128) * psf_shift_spectrum(n, spacing, origin, psf_cov)
    g = np.asarray(dL_dimage, dtype=np.float64).reshape(n)
    dS = np.fft.rfftn(g, axes=(0, 1, 2)) / float(np.prod(n))
    w = np.full(n[2] // 2 + 1, 2.0)
    w[0] = 1.0
    if n[2] % 2 == 0:
        w[-1] = 1.0
    t = (np.conj(dS * w[None, None, :]) * S).real
    k = frequency_grid(n, spacing)
    kx, ky, kz = k[..., 0], k[..., 1], k[..., 2]
    q = [-0.5 * kx * kx, -0.5 * ky * ky, -0.5 * kz * kz, -kx * ky, -kx * kz, -ky * kz]
    return np.array([float((qm * t).sum()) for qm in q])
