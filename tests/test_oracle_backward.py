"""Pins P8 (central finite differences) and P9 (exact identities) for the oracle's backward."""
import numpy as np
import pytest

import oracle
from workloads import icosphere, perturb_radial, box_mesh

VOL, SURF = 0, 1


def _small_mesh(seed):
    rng = np.random.default_rng(seed)
    v, f = icosphere(1, 0.3, (0.03, -0.02, 0.05))       # 42 vertices, 80 triangles
    return perturb_radial(v, (0.03, -0.02, 0.05), 0.1, rng), f


def _loss(v, f, k, mode, G):
    F = oracle.mesh_ft_forward(v, f, k, mode)
    return float(np.sum(G.real * F.real + G.imag * F.imag))    # L with dL/dReF + i dL/dImF = G


@pytest.mark.parametrize("mode", [VOL, SURF])
def test_P8_backward_vs_central_finite_differences(mode):
    v, f = _small_mesh(10)
    rng = np.random.default_rng(11)
    k = rng.uniform(-35, 35, (24, 3))
    k[0] = 0.0                                           # the k = 0 row of the gradient
    k[1] = [0.0, 0.0, 12.0]                              # axis-aligned: exact coincidences a = b
    G = rng.standard_normal(24) + 1j * rng.standard_normal(24)
    grad = oracle.mesh_ft_backward(v, f, k, mode, G)
    fd = np.zeros_like(v)
    h = 1e-6
    for i in range(v.shape[0]):
        for d in range(3):
            vp, vm = v.copy(), v.copy()
            vp[i, d] += h
            vm[i, d] -= h
            fd[i, d] = (_loss(vp, f, k, mode, G) - _loss(vm, f, k, mode, G)) / (2 * h)
    rel = np.linalg.norm(grad - fd) / np.linalg.norm(fd)
    assert rel < 1e-7, rel


@pytest.mark.parametrize("mode", [VOL, SURF])
def test_P9_translation_identity_for_the_whole_backward(mode):
    """sum_p dg/da_p = -i g  =>  sum_v dL/dv = sum_k Re( conj(G) (-i k) F(k) )   (no finite differences)."""
    v, f = _small_mesh(12)
    rng = np.random.default_rng(13)
    k = rng.uniform(-60, 60, (50, 3))
    k[3] = 0.0
    G = rng.standard_normal(50) + 1j * rng.standard_normal(50)
    grad = oracle.mesh_ft_backward(v, f, k, mode, G)
    F = oracle.mesh_ft_forward(v, f, k, mode)
    rhs = np.real(np.conj(G)[:, None] * (-1j * k) * F[:, None]).sum(axis=0)
    assert np.abs(grad.sum(axis=0) - rhs).max() < 1e-12 * max(1.0, np.abs(rhs).max())


def test_P9_zero_frequency_rows_are_area_and_volume_gradients():
    """k = 0 only: surface gives d(area)/dv = sum -w_p/2, volume gives dV/dv."""
    v, f = _small_mesh(14)
    k0 = np.zeros((1, 3))
    G = np.array([1.0 + 0.0j])

    def area(vv):
        a, b, c = vv[f[:, 0]], vv[f[:, 1]], vv[f[:, 2]]
        return 0.5 * np.linalg.norm(np.cross(b - a, c - a), axis=1).sum()

    def vol(vv):
        a, b, c = vv[f[:, 0]], vv[f[:, 1]], vv[f[:, 2]]
        return np.einsum("ij,ij->", a, np.cross(b, c)) / 6.0

    for mode, fun in ((SURF, area), (VOL, vol)):
        grad = oracle.mesh_ft_backward(v, f, k0, mode, G)
        fd = np.zeros_like(v)
        h = 1e-6
        for i in range(v.shape[0]):
            for d in range(3):
                vp, vm = v.copy(), v.copy()
                vp[i, d] += h
                vm[i, d] -= h
                fd[i, d] = (fun(vp) - fun(vm)) / (2 * h)
        assert np.abs(grad - fd).max() < 1e-9
    # closed surface: total area gradient of every vertex star is minus the sum of w_p / 2
    _, corners = oracle.mesh_ft_backward(v, f, k0, SURF, G, return_corners=True)
    for t in (0, 17, 79):
        p0, p1, p2 = v[f[t]]
        e = [p2 - p1, p0 - p2, p1 - p0]                 # e_p = v_{p-} - v_{p+}
        m = np.cross(e[2], e[0])
        N = m / np.linalg.norm(m)
        for p in range(3):
            assert np.abs(corners[t, p] + 0.5 * np.cross(e[p], N)).max() < 1e-14


def test_backward_is_linear_in_G_and_additive_over_frequency_subsets():
    v, f = _small_mesh(15)
    rng = np.random.default_rng(16)
    k = rng.uniform(-30, 30, (20, 3))
    G = rng.standard_normal(20) + 1j * rng.standard_normal(20)
    full = oracle.mesh_ft_backward(v, f, k, VOL, G)
    part = oracle.mesh_ft_backward(v, f, k[:7], VOL, G[:7]) + oracle.mesh_ft_backward(v, f, k[7:], VOL, G[7:])
    assert np.abs(full - part).max() < 1e-13
    assert np.abs(oracle.mesh_ft_backward(v, f, k, VOL, 2.5 * G) - 2.5 * full).max() < 1e-13


def test_degenerate_triangle_contributes_zero_in_surface_mode():
    """Reading R19: a zero-area triangle has no normal; it contributes nothing."""
    v, f = box_mesh((0, 0, 0), (0.2, 0.2, 0.2))
    v2 = np.concatenate([v, [[0.3, 0.3, 0.3]]])
    f2 = np.concatenate([f, [[0, 0, 8]]]).astype(np.int32)      # repeated vertex => zero area
    k = np.random.default_rng(17).uniform(-20, 20, (10, 3))
    G = np.ones(10, dtype=complex)
    g1 = oracle.mesh_ft_backward(v, f, k, SURF, G)
    g2 = oracle.mesh_ft_backward(v2, f2, k, SURF, G)
    assert np.abs(g2[:8] - g1).max() < 1e-15 and np.all(g2[8] == 0)


def test_area_normalised_density_eq12_eq13():
    """NEXT 3: the area gradient -w_p/2 against central differences of the area, and
    the gradient of the normalised FT (eq. 13) against central differences of eq. 12; u_Lambda(0) = 1; scale invariance
    u_{s Lambda}(k) = u_Lambda(s k)."""
    from workloads import icosphere
    rng = np.random.default_rng(21)
    v, f = icosphere(1, 0.3, (0.03, -0.02, 0.01))
    v = (v + 0.02 * rng.standard_normal(v.shape)).astype(np.float32).astype(np.float64)
    k = rng.uniform(-25, 25, size=(40, 3))
    k[0] = 0.0
    G = rng.standard_normal(40) + 1j * rng.standard_normal(40)
    area, darea = oracle.surface_area_and_gradient(v, f)
    u = oracle.mesh_ft_forward_normalised(v, f, k)
    assert abs(u[0] - 1.0) < 1e-14
    assert np.abs(oracle.mesh_ft_forward_normalised(1.7 * v, f, k / 1.7) - u).max() < 1e-13
    grad = oracle.mesh_ft_backward_normalised(v, f, k, G)
    fd, fda = np.zeros_like(v), np.zeros_like(v)
    h = 1e-6
    for i in range(v.shape[0]):
        for d in range(3):
            vp, vm = v.copy(), v.copy()
            vp[i, d] += h
            vm[i, d] -= h
            fd[i, d] = ((np.conj(G) * oracle.mesh_ft_forward_normalised(vp, f, k)).real.sum()
                        - (np.conj(G) * oracle.mesh_ft_forward_normalised(vm, f, k)).real.sum()) / (2 * h)
            fda[i, d] = (oracle.surface_area_and_gradient(vp, f)[0] - oracle.surface_area_and_gradient(vm, f)[0]) / (2 * h)
    assert np.linalg.norm(darea - fda) <= 1e-8 * np.linalg.norm(fda)
    assert np.linalg.norm(grad - fd) <= 1e-7 * np.linalg.norm(fd)


# ---- per-face density weights (reading R23) ------------------------------------------------------------
def _weighted_case(seed):
    """42-vertex perturbed sphere; three distinct weights, one negative, assigned per face at random (so that a
    group mask applied to the wrong axis, or a dropped weight, changes the result)."""
    v, f = _small_mesh(seed)
    rng = np.random.default_rng(seed + 1)
    w = rng.choice([1.0, 0.35, -0.6], size=len(f))
    assert len(np.unique(w)) == 3
    return v, f, w


@pytest.mark.parametrize("mode", [VOL, SURF])
def test_weighted_backward_vs_central_finite_differences(mode):
    """P8 for oracle.mesh_ft_backward_weighted: central differences of oracle.mesh_ft_forward_weighted."""
    v, f, w = _weighted_case(20)
    rng = np.random.default_rng(21)
    k = rng.uniform(-35, 35, (20, 3))
    k[0] = 0.0
    k[1] = [0.0, 9.0, 0.0]
    G = rng.standard_normal(20) + 1j * rng.standard_normal(20)

    def loss(vv):
        F = oracle.mesh_ft_forward_weighted(vv, f, k, mode, w)
        return float(np.sum(G.real * F.real + G.imag * F.imag))

    grad = oracle.mesh_ft_backward_weighted(v, f, k, mode, G, w)
    fd = np.zeros_like(v)
    h = 1e-6
    for i in range(v.shape[0]):
        for d in range(3):
            vp, vm = v.copy(), v.copy()
            vp[i, d] += h
            vm[i, d] -= h
            fd[i, d] = (loss(vp) - loss(vm)) / (2 * h)
    rel = np.linalg.norm(grad - fd) / np.linalg.norm(fd)
    assert rel < 1e-7, rel


@pytest.mark.parametrize("mode", [VOL, SURF])
def test_weighted_backward_translation_identity_and_corner_sum(mode):
    """P9 with weights: sum_v dL/dv = sum_k Re(conj(G) (-ik) F_w(k)); and the weighted gradient equals the scatter of
    w_T times the UNWEIGHTED per-corner gradients (oracle_mesh_ft_backward's corner output), an assembly that never
    groups faces by weight."""
    v, f, w = _weighted_case(22)
    rng = np.random.default_rng(23)
    k = rng.uniform(-50, 50, (40, 3))
    if mode == SURF:
        k[5] = 0.0       # (volume mode: the k = 0 entry of a weighted, hence open, surface is the weighted sum of origin
                         #  cones, which is not translation invariant; its gradient is covered by the FD test above)
    G = rng.standard_normal(40) + 1j * rng.standard_normal(40)
    grad = oracle.mesh_ft_backward_weighted(v, f, k, mode, G, w)
    F = oracle.mesh_ft_forward_weighted(v, f, k, mode, w)
    rhs = np.real(np.conj(G)[:, None] * (-1j * k) * F[:, None]).sum(axis=0)
    assert np.abs(grad.sum(axis=0) - rhs).max() < 1e-12 * max(1.0, np.abs(rhs).max())
    _, corners = oracle.mesh_ft_backward(v, f, k, mode, G, return_corners=True)
    want = np.zeros_like(v)
    for t, tri in enumerate(f):
        for c in range(3):
            want[tri[c]] += w[t] * corners[t, c]
    assert np.abs(grad - want).max() < 1e-12 * np.abs(want).max()
