"""Pins of oracle/shape_step.py (eq. 17; readings R26-R28): the connectivity Laplacian, the
(I + lambda L)^-2 preconditioner, Phi_1 and AdamUniform -- against hand-computed values, closed forms and finite
differences, never against the oracle's own formulas."""
import numpy as np
import pytest

import oracle
from workloads import icosphere, tetrahedron_mesh


def test_laplacian_of_the_tetrahedron_by_hand():
    """Every vertex of a tetrahedron neighbours the other three: L = 4 I - J (3 on the diagonal, -1 elsewhere)."""
    _, f = tetrahedron_mesh([[0, 0, 0], [1, 0, 0], [0, 1, 0], [0, 0, 1]])
    L = oracle.connectivity_laplacian(f, 4)
    assert np.array_equal(L, 4 * np.eye(4) - np.ones((4, 4)))


def test_laplacian_structure_on_an_icosphere():
    v, f = icosphere(2, 1.0)
    n = len(v)
    L = oracle.connectivity_laplacian(f, n)
    assert np.array_equal(L, L.T)
    assert np.abs(L @ np.ones(n)).max() == 0.0                       # constants are in the kernel
    deg = np.diag(L)
    assert sorted(set(deg.tolist())) == [5.0, 6.0] and (deg == 5).sum() == 12     # 12 icosahedron vertices of valence 5
    assert L.trace() == 2 * (3 * len(f) // 2)                         # sum of degrees = 2 |E|, |E| = 3 n_T / 2 (closed)
    off = L - np.diag(deg)
    assert set(np.unique(off).tolist()) == {-1.0, 0.0}
    edges = {tuple(sorted((int(t[a]), int(t[(a + 1) % 3])))) for t in f for a in range(3)}
    assert all(off[i, j] == -1.0 for i, j in edges) and (off == -1).sum() == 2 * len(edges)
    w = np.linalg.eigvalsh(L)
    assert w[0] > -1e-12 and w[1] > 1e-6                              # positive semi-definite, connected: one zero mode
    x = np.random.default_rng(0).standard_normal(n)
    assert abs(x @ L @ x - sum((x[i] - x[j]) ** 2 for i, j in edges)) < 1e-9     # the graph Dirichlet energy


def test_preconditioner_closed_form_on_the_tetrahedron_and_residual():
    """L = 4I - J has eigenvalue 0 on constants and 4 on their complement, so (I + lambda L)^-2 g =
    mean(g) + (g - mean(g)) / (1 + 4 lambda)^2."""
    _, f = tetrahedron_mesh([[0, 0, 0], [1, 0, 0], [0, 1, 0], [0, 0, 1]])
    L = oracle.connectivity_laplacian(f, 4)
    g = np.random.default_rng(1).standard_normal((4, 3))
    lam = 50.0
    want = g.mean(axis=0) + (g - g.mean(axis=0)) / (1 + 4 * lam) ** 2
    assert np.abs(oracle.precondition(g, L, lam) - want).max() < 1e-14
    # generic mesh: residual of the defining system (I + lambda L)^2 x = g, and lambda = 0 is the identity
    v, f = icosphere(2, 0.3)
    L = oracle.connectivity_laplacian(f, len(v))
    g = np.random.default_rng(2).standard_normal((len(v), 3))
    x = oracle.precondition(g, L, lam)
    M = np.eye(len(v)) + lam * L
    assert np.abs(M @ (M @ x) - g).max() < 1e-9 * np.abs(g).max()
    assert np.abs(oracle.precondition(g, L, 0.0) - g).max() < 1e-15
    assert np.abs(x.sum(axis=0) - g.sum(axis=0)).max() < 1e-10        # the mean (translation) passes unchanged


def test_phi1_by_hand_and_finite_differences():
    u = np.array([[[1.0, 2.0]], [[0.5, -1.0]]])
    m = np.array([[[0.0, 1.0]], [[2.0, 3.0]]])
    # (1-0)^2*0 + (2-1)^2*1 + (0.5-2)^2*2 + (-1-3)^2*3 = 0 + 1 + 4.5 + 48
    assert oracle.phi1(u, m) == 53.5
    assert np.array_equal(oracle.phi1_grad(u, m), np.array([[[0.0, 2.0]], [[-6.0, -24.0]]]))
    rng = np.random.default_rng(3)
    u, m = rng.standard_normal((4, 3, 5)), rng.uniform(0, 2, (4, 3, 5))
    g = oracle.phi1_grad(u, m)
    h = 1e-6
    for idx in [(0, 0, 0), (3, 2, 4), (1, 1, 2)]:
        up, um = u.copy(), u.copy()
        up[idx] += h
        um[idx] -= h
        assert abs((oracle.phi1(up, m) - oracle.phi1(um, m)) / (2 * h) - g[idx]) < 1e-7
    assert oracle.phi1(m, m) == 0.0 and oracle.phi1(u, np.zeros_like(u)) == 0.0   # dark voxels carry no weight


def test_adam_uniform_steps_by_hand():
    """Reading R28, two steps computed by hand with b1 = 0.9, b2 = 0.999, eps = 0 and lr = 0.1.
    Step 1: m = 0.1 g, s = 0.001 max g^2; bias-corrected: m_hat = g, s_hat = max g^2: the update is lr g / max|g|."""
    x = np.array([[1.0, 2.0, 3.0], [0.0, -1.0, 0.5]])
    g1 = np.array([[0.2, -0.4, 0.1], [0.0, 0.3, -0.1]])
    st = oracle.AdamUniformState()
    x1 = oracle.adam_uniform_step(x, g1, st, lr=0.1, eps=0.0)
    assert np.abs(x1 - (x - 0.1 * g1 / 0.4)).max() < 1e-15
    assert st.t == 1 and abs(st.s - 0.001 * 0.16) < 1e-18
    # Step 2 with g2: m = 0.9*0.1 g1 + 0.1 g2, m_hat = m / 0.19; s = 0.999*0.00016 + 0.001*0.25, s_hat = s / 0.001999
    g2 = np.array([[0.5, 0.1, -0.2], [0.1, 0.0, 0.2]])
    x2 = oracle.adam_uniform_step(x1, g2, st, lr=0.1, eps=0.0)
    m_hat = (0.09 * g1 + 0.1 * g2) / 0.19
    s_hat = (0.999 * 0.00016 + 0.001 * 0.25) / (1 - 0.999 ** 2)
    assert np.abs(x2 - (x1 - 0.1 * m_hat / np.sqrt(s_hat))).max() < 1e-15
    # uniform scaling: the step direction is the first moment's, whatever the spread of the entries
    assert np.allclose((x1 - x2) / (x1 - x2)[0, 0], m_hat / m_hat[0, 0])


def test_shape_step_moves_towards_the_target_and_decreases_phi1():
    """A sphere of radius 0.25 fitted to the image of a sphere of radius 0.3: after one step every vertex has moved outwards
    and Phi_1 of the next render is smaller."""
    from workloads.configs import _grid
    v, f = icosphere(1, 0.25)
    vt, _ = icosphere(1, 0.30)
    n, spacing, origin = _grid((12, 12, 12))
    cov = np.array([(1.5 * spacing[0]) ** 2] * 3 + [0, 0, 0], dtype=np.float64)
    target = oracle.render(vt, f, n, spacing, origin, cov, 0)
    st = oracle.ShapeState()
    v1, l0 = oracle.shape_step(v, f, n, spacing, origin, cov, 0, target, st, oracle.ShapeParams(lr=5e-3))
    r0, r1 = np.linalg.norm(v, axis=1), np.linalg.norm(v1, axis=1)
    assert (r1 > r0).all()
    assert np.abs(np.linalg.norm(v1 - v, axis=1)).max() <= 5e-3 * np.sqrt(3) + 1e-12    # lr bounds every coordinate's move
    l1 = oracle.phi1(oracle.render(v1, f, n, spacing, origin, cov, 0), target)
    assert l1 < l0


# ---- the step as a COMPOSITION (eq. 17; band: PAPER.md:227-240) -----------------------------------------
# The pieces above are pinned one by one; what follows pins their order.  The gradient is re-derived here by central finite
# differences of Phi_1 o render (forward evaluations only -- never oracle.render_backward), the preconditioner is the
# tetrahedron's closed form, and AdamUniform's first step is lr * g~ / max|g~| (test_adam_uniform_steps_by_hand).  A step that
# skipped the preconditioner, differentiated another loss, or banded F but not G would miss these by orders of magnitude.
def _tetra_problem():
    from workloads.configs import _grid
    v, f = tetrahedron_mesh([[-0.2, -0.2, -0.2], [0.25, -0.15, -0.2], [-0.1, 0.3, -0.15], [0.0, 0.0, 0.3]])
    n, spacing, origin = _grid((8, 8, 8))
    cov = np.array([(1.2 * spacing[0]) ** 2, (1.0 * spacing[1]) ** 2, (1.5 * spacing[2]) ** 2, 0, 0, 0], dtype=np.float64)
    target = oracle.render(1.2 * v + 0.01, f, n, spacing, origin, cov, 0)
    return v, f, n, spacing, origin, cov, target


def _band_mask(n, spacing, cov, cutoff):
    k = oracle.frequency_grid(n, spacing)                               # [n_x, n_y, n_z/2+1, 3]
    quad = cov[0] * k[..., 0] ** 2 + cov[1] * k[..., 1] ** 2 + cov[2] * k[..., 2] ** 2
    return np.exp(-0.5 * quad) > cutoff


def _fd_gradient(loss_of_vertices, v, h=1e-6):
    g = np.zeros_like(v)
    for i in range(v.shape[0]):
        for d in range(3):
            vp, vm = v.copy(), v.copy()
            vp[i, d] += h
            vm[i, d] -= h
            g[i, d] = (loss_of_vertices(vp) - loss_of_vertices(vm)) / (2 * h)
    return g


@pytest.mark.parametrize("lam", [0.0, 50.0])
def test_first_shape_step_equals_the_preconditioned_finite_difference_gradient(lam):
    v, f, n, spacing, origin, cov, target = _tetra_problem()
    g = _fd_gradient(lambda x: oracle.phi1(oracle.render(x, f, n, spacing, origin, cov, 0), target), v)
    gp = g.mean(axis=0) + (g - g.mean(axis=0)) / (1 + 4 * lam) ** 2     # (I + lam L)^-2 on the tetrahedron, L = 4I - J
    lr = 2e-3
    want = v - lr * gp / np.abs(gp).max()
    v1, loss = oracle.shape_step(v, f, n, spacing, origin, cov, 0, target, oracle.ShapeState(),
                                 oracle.ShapeParams(lr=lr, lam=lam, eps=0.0))
    assert loss == oracle.phi1(oracle.render(v, f, n, spacing, origin, cov, 0), target)
    assert np.abs(v1 - want).max() <= 1e-5 * lr, np.abs(v1 - want).max() / lr
    if lam > 0:   # the preconditioner matters: the unpreconditioned step is somewhere else entirely
        assert np.abs(want - (v - lr * g / np.abs(g).max())).max() > 1e-2 * lr


def test_shape_step_band_branch():
    v, f, n, spacing, origin, cov, target = _tetra_problem()
    prm = oracle.ShapeParams(lr=2e-3, lam=50.0, eps=0.0)
    plain, loss_plain = oracle.shape_step(v, f, n, spacing, origin, cov, 0, target, oracle.ShapeState(), prm)
    full = np.ones((n[0], n[1], n[2] // 2 + 1), dtype=bool)
    allin, loss_all = oracle.shape_step(v, f, n, spacing, origin, cov, 0, target, oracle.ShapeState(), prm, band=full)
    assert np.array_equal(plain, allin) and loss_plain == loss_all      # an all-true band is no band, bit for bit
    band = _band_mask(n, spacing, cov, 0.05)
    assert 0.04 < band.mean() < 0.6 and band[0, 0, 0]                   # a real restriction that keeps k = 0

    def banded_loss(x):
        F = oracle.mesh_ft_forward_grid(x, f, n, spacing, 0)
        return oracle.phi1(oracle.spectrum_to_image(np.where(band, F, 0.0), n, spacing, origin, cov), target)

    g = _fd_gradient(banded_loss, v)
    gp = g.mean(axis=0) + (g - g.mean(axis=0)) / (1 + 4 * prm.lam) ** 2
    want = v - prm.lr * gp / np.abs(gp).max()
    got, loss = oracle.shape_step(v, f, n, spacing, origin, cov, 0, target, oracle.ShapeState(), prm, band=band)
    assert loss == banded_loss(v)
    assert np.abs(got - want).max() <= 1e-5 * prm.lr, np.abs(got - want).max() / prm.lr
    # and the band is not a no-op here: the unbanded step differs visibly
    assert np.abs(got - plain).max() > 1e-3 * prm.lr
