"""Shape-optimisation step of deltaMic (section 5.1.3, eq. 17) -- TEST INFRASTRUCTURE, numpy fp64.

    Phi_1 = || u - m ||^2 * m  =  sum_voxels (u - m)^2 m          (kappa = 1)
    v <- v - eta (I + lambda L)^-2 dPhi_1/dv ,  lambda = 50       (eq. 17)

with L the connectivity (combinatorial) Laplacian of the triangle mesh and the step taken by AdamUniform (PAPER.md:244,
ref. [55]).  The paper solves with a sparse Cholesky factorisation; this oracle is the definition written out with DENSE
algebra (numpy.linalg.solve on (I + lambda L), applied twice), which is only feasible for a few hundred vertices.

Readings:
  R26  "connectivity Laplacian" = L = D - A of the vertex graph of the mesh: L_ii = number of distinct neighbours of
       vertex i, L_ij = -1 when i and j share an edge, else 0 (L 1 = 0, symmetric, positive semi-definite).
  R27  eq. 17 prints (I + lambda L)^-2 A = dPhi/dv for the system to solve; the operator applied to the gradient in the
       update is (I + lambda L)^-2, so the system is (I + lambda L)^2 A = dPhi/dv, one column per coordinate.
  R28  "AdamUniform" (ref. [55]; the paper gives no formula): Adam [32] whose second moment is ONE scalar per step, the
       largest squared entry of the (preconditioned) gradient:
           m_t = b1 m_{t-1} + (1 - b1) g,   s_t = b2 s_{t-1} + (1 - b2) max_i g_i^2,
           v <- v - eta (m_t / (1 - b1^t)) / (sqrt(s_t / (1 - b2^t)) + eps),
       so every coordinate is scaled alike (a per-coordinate scaling would undo the smoothing of the preconditioner).
       b1 = 0.9, b2 = 0.999, eps = 1e-8 (the defaults of [32]).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


def phi1(u, m) -> float:
    """Phi_1 = sum (u - m)^2 m."""
    u = np.asarray(u, dtype=np.float64)
    m = np.asarray(m, dtype=np.float64)
    return float(((u - m) ** 2 * m).sum())


def phi1_grad(u, m) -> np.ndarray:
    """dPhi_1/du = 2 (u - m) m."""
    u = np.asarray(u, dtype=np.float64)
    m = np.asarray(m, dtype=np.float64)
    return 2.0 * (u - m) * m


def connectivity_laplacian(faces, n_vertices: int) -> np.ndarray:
    """Dense L = D - A of the mesh's vertex graph (reading R26)."""
    f = np.asarray(faces, dtype=np.int64).reshape(-1, 3)
    A = np.zeros((n_vertices, n_vertices), dtype=np.float64)
    for tri in f:
        for a in range(3):
            i, j = int(tri[a]), int(tri[(a + 1) % 3])
            if i != j:
                A[i, j] = 1.0
                A[j, i] = 1.0
    return np.diag(A.sum(axis=1)) - A


def precondition(g, L, lam: float) -> np.ndarray:
    """(I + lambda L)^-2 g, column by column (eq. 17 with reading R27): two dense solves with I + lambda L."""
    M = np.eye(L.shape[0]) + float(lam) * np.asarray(L, dtype=np.float64)
    y = np.linalg.solve(M, np.asarray(g, dtype=np.float64))
    return np.linalg.solve(M, y)


@dataclass
class AdamUniformState:
    m: np.ndarray | None = None   # first moment [n_V, 3]
    s: float = 0.0                # scalar second moment
    t: int = 0                    # steps taken


def adam_uniform_step(x, g, state: AdamUniformState, lr: float, beta1: float = 0.9, beta2: float = 0.999,
                      eps: float = 1e-8) -> np.ndarray:
    """One AdamUniform update of x with gradient g (reading R28); ``state`` is updated in place."""
    g = np.asarray(g, dtype=np.float64)
    if state.m is None:
        state.m = np.zeros_like(g)
    state.t += 1
    state.m = beta1 * state.m + (1.0 - beta1) * g
    state.s = beta2 * state.s + (1.0 - beta2) * float((g * g).max())
    mhat = state.m / (1.0 - beta1 ** state.t)
    shat = state.s / (1.0 - beta2 ** state.t)
    return np.asarray(x, dtype=np.float64) - lr * mhat / (np.sqrt(shat) + eps)


@dataclass
class ShapeParams:
    lr: float = 1e-3
    lam: float = 50.0
    beta1: float = 0.9
    beta2: float = 0.999
    eps: float = 1e-8


@dataclass
class ShapeState:
    adam: AdamUniformState = field(default_factory=AdamUniformState)
    L: np.ndarray | None = None


def shape_step(vertices, faces, n, spacing, origin, psf_cov, mode: int, target, state: ShapeState,
               params: ShapeParams = ShapeParams(), band=None):
    """One shape-optimisation step: render, Phi_1, vertex gradient through the renderer, the
    (I + lambda L)^-2 preconditioner, AdamUniform.  Returns (new vertices [n_V,3] float64, Phi_1 before the step).

    ``band``: optional boolean mask over the stored half spectrum (the narrow band of PAPER.md:227-231, 5.1.2 (a)):
    the spectrum is zeroed outside it in the forward and the cotangent is zeroed outside it in the backward."""
    from .mesh_ft import mesh_ft_backward_grid, mesh_ft_forward_grid
    from .render import image_to_spectrum_cotangent, spectrum_to_image

    v = np.asarray(vertices, dtype=np.float64).reshape(-1, 3)
    F = mesh_ft_forward_grid(v, faces, n, spacing, mode)
    if band is not None:
        F = np.where(band, F, 0.0)
    u = spectrum_to_image(F, n, spacing, origin, psf_cov)
    loss = phi1(u, target)
    G = image_to_spectrum_cotangent(phi1_grad(u, target), n, spacing, origin, psf_cov)
    if band is not None:
        G = np.where(band, G, 0.0)
    g = mesh_ft_backward_grid(v, faces, n, spacing, mode, G)
    if state.L is None:
        state.L = connectivity_laplacian(faces, v.shape[0])
    gp = precondition(g, state.L, params.lam)
    v_new = adam_uniform_step(v, gp, state.adam, params.lr, params.beta1, params.beta2, params.eps)
    return v_new, loss
