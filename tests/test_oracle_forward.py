"""Pins P1, P2, P3, P5, P6, P7 for the oracle's forward mesh FT (SURVEY.md §8(c) "Pins")."""
import numpy as np
import pytest

import oracle
from workloads import box_mesh, icosphere, tetrahedron_mesh, perturb_radial

VOL, SURF = 0, 1


def _sinc_factor(k, h):
    """S_a = int_{-h}^{h} e^{-ikx} dx = 2 sin(kh)/k  (-> 2h at k = 0)."""
    k = np.asarray(k, dtype=np.float64)
    safe = np.where(k == 0, 1.0, k)
    return np.where(k == 0, 2.0 * h, 2.0 * np.sin(safe * h) / safe)


def box_ft(k, c, h, mode):
    """Analytic FT of the axis-aligned box [c-h, c+h]: product of sincs (volume) / six faces (surface)."""
    S = [_sinc_factor(k[:, a], h[a]) for a in range(3)]
    ph = np.exp(-1j * (k @ c))
    if mode == VOL:
        return ph * S[0] * S[1] * S[2]
    C = [2.0 * np.cos(k[:, a] * h[a]) for a in range(3)]
    return ph * (C[0] * S[1] * S[2] + C[1] * S[0] * S[2] + C[2] * S[0] * S[1])


@pytest.mark.parametrize("mode", [VOL, SURF])
def test_P1_axis_aligned_box_on_grid_and_off_grid(mode):
    c = np.array([0.05, -0.02, 0.1])
    h = np.array([0.2, 0.15, 0.1])
    v, f = box_mesh(c, h)
    # on the grid: axis-aligned k makes a=b and a=b=c hold exactly (degenerate branches)
    k = oracle.frequency_grid((16, 12, 10), (1 / 16, 1 / 12, 1 / 10)).reshape(-1, 3)
    F = oracle.mesh_ft_forward(v, f, k, mode)
    assert np.abs(F - box_ft(k, c, h, mode)).max() < 1e-13
    # off the grid, generic directions, large |k|
    k = np.random.default_rng(0).uniform(-300, 300, (400, 3))
    F = oracle.mesh_ft_forward(v, f, k, mode)
    assert np.abs(F - box_ft(k, c, h, mode)).max() < 1e-13


def _volume_area(v, f):
    a, b, c = v[f[:, 0]], v[f[:, 1]], v[f[:, 2]]
    vol = np.einsum("ij,ij->", a, np.cross(b, c)) / 6.0
    area = 0.5 * np.linalg.norm(np.cross(b - a, c - a), axis=1).sum()
    return vol, area


def test_P2_zero_frequency_is_volume_and_area():
    rng = np.random.default_rng(1)
    v, f = icosphere(2, 0.3, (0.1, 0.0, -0.05))
    v = perturb_radial(v, (0.1, 0.0, -0.05), 0.05, rng)
    vol, area = _volume_area(v, f)
    k0 = np.zeros((1, 3))
    assert oracle.mesh_ft_forward(v, f, k0, VOL)[0] == pytest.approx(vol, rel=1e-14)
    assert oracle.mesh_ft_forward(v, f, k0, SURF)[0] == pytest.approx(area, rel=1e-14)
    assert abs(oracle.mesh_ft_forward(v, f, k0, VOL)[0].imag) == 0.0
    # volume mode is continuous at k -> 0 although its formula divides by |k|^2
    kk = np.array([[1e-5, -2e-5, 1.5e-5]])
    assert abs(oracle.mesh_ft_forward(v, f, kk, VOL)[0] - vol) < 1e-5


@pytest.mark.parametrize("mode", [VOL, SURF])
def test_P3_translation_scaling_orientation_additivity_hermitian(mode):
    rng = np.random.default_rng(2)
    v, f = icosphere(1, 0.25)
    v = perturb_radial(v, (0, 0, 0), 0.1, rng)
    k = rng.uniform(-40, 40, (64, 3))
    F = oracle.mesh_ft_forward(v, f, k, mode)
    t = np.array([0.11, -0.07, 0.2])
    Ft = oracle.mesh_ft_forward(v + t, f, k, mode)
    assert np.abs(Ft - np.exp(-1j * (k @ t)) * F).max() < 1e-12            # F_{x+t}(k) = e^{-ik.t} F_x(k)
    s = 1.7
    Fs = oracle.mesh_ft_forward(s * v, f, k / s, mode)
    assert np.abs(Fs - s ** (3 if mode == VOL else 2) * F).max() < 1e-12   # F_{sx}(k/s) = s^d F_x(k)
    Fneg = oracle.mesh_ft_forward(v, f, -k, mode)
    assert np.abs(Fneg - np.conj(F)).max() < 1e-13                          # real density
    Fflip = oracle.mesh_ft_forward(v, f[:, [0, 2, 1]], k, mode)
    assert np.abs(Fflip - (-F if mode == VOL else F)).max() < 1e-13         # orientation (R8)
    v2, f2 = box_mesh((0.3, 0.3, -0.2), (0.05, 0.08, 0.04))
    Fb = oracle.mesh_ft_forward(v2, f2, k, mode)
    Fsum = oracle.mesh_ft_forward(np.concatenate([v, v2]), np.concatenate([f, f2 + len(v)]), k, mode)
    assert np.abs(Fsum - (F + Fb)).max() < 1e-13                            # components add


def test_P3_hermitian_symmetry_inside_stored_grid():
    """F(-k) = conj F(k) checked on the n_z = 0 plane of the stored half spectrum (R10 ordering)."""
    v, f = icosphere(1, 0.3, (0.02, 0.05, -0.03))
    n = (8, 10, 6)
    F = oracle.mesh_ft_forward_grid(v, f, n, (1 / 8, 1 / 10, 1 / 6), VOL)
    assert F.shape == (8, 10, 4)
    for ix in range(1, 4):
        for iy in range(1, 5):
            assert abs(F[ix, iy, 0] - np.conj(F[-ix, -iy, 0])) < 1e-14
    k = oracle.frequency_grid(n, (1 / 8, 1 / 10, 1 / 6))
    assert np.allclose(k[3, 0, 0], [2 * np.pi * 3, 0, 0]) and np.allclose(k[5, 0, 0], [-2 * np.pi * 3, 0, 0])
    assert np.allclose(k[4, 0, 0], [-2 * np.pi * 4, 0, 0])        # Nyquist carries the negative sign (fftfreq)
    assert np.allclose(k[0, 0, 3], [0, 0, 2 * np.pi * 3])


def test_P5_surface_mode_vs_gauss_quadrature():
    """int_T e^{-ik.x} dS per triangle by tensor Gauss-Legendre on the Duffy square."""
    rng = np.random.default_rng(3)
    v, f = icosphere(0, 0.4)
    v = perturb_radial(v, (0, 0, 0), 0.15, rng)
    k = rng.uniform(-12, 12, (40, 3))
    x, w = np.polynomial.legendre.leggauss(40)
    x, w = 0.5 * (x + 1), 0.5 * w
    U, W = np.meshgrid(x, x, indexing="ij")
    wt = np.outer(w, w) * (1 - U)
    ref = np.zeros(len(k), dtype=complex)
    for tri in f:
        p0, p1, p2 = v[tri]
        pts = p0 + U[..., None] * (p1 - p0) + (W * (1 - U))[..., None] * (p2 - p0)
        twoA = np.linalg.norm(np.cross(p1 - p0, p2 - p0))
        ref += twoA * np.einsum("ij,ijq->q", wt, np.exp(-1j * np.einsum("ijd,qd->ijq", pts, k)))
    got = oracle.mesh_ft_forward(v, f, k, SURF)
    assert np.abs(got - ref).max() < 1e-12


def test_P6_volume_mode_vs_voxelised_indicator():
    """Brute force: DFT of a finely voxelised indicator of a convex mesh (first-order accurate)."""
    v, f = tetrahedron_mesh([[-0.3, -0.25, -0.2], [0.35, -0.2, -0.15], [-0.05, 0.4, -0.1], [0.0, 0.05, 0.38]])
    M = 160
    xs = (np.arange(M) + 0.5) / M - 0.5
    X, Y, Z = np.meshgrid(xs, xs, xs, indexing="ij")
    P = np.stack([X, Y, Z], axis=-1).reshape(-1, 3)
    inside = np.ones(len(P), dtype=bool)
    for tri in f:
        a, b, c = v[tri]
        nrm = np.cross(b - a, c - a)
        inside &= (P - a) @ nrm <= 0
    P = P[inside]
    k = 2 * np.pi * np.array([[0, 0, 0], [1, 0, 0], [0, 2, 0], [0, 0, 1], [1, -1, 2], [-2, 1, 1], [3, 2, -1], [2, 2, 2]], float)
    ref = np.exp(-1j * P @ k.T).sum(axis=0) / M ** 3
    got = oracle.mesh_ft_forward(v, f, k, VOL)
    vol = got[0].real
    assert vol > 0 and abs(ref[0] - vol) < 5e-3 * vol            # sign and scale: outward faces => +volume
    assert np.abs(got - ref).max() < 1e-2 * vol


def test_P7_fine_icosphere_vs_ball_and_shell():
    R = 0.4
    v, f = icosphere(5, R)
    kk = np.array([0.5, 3.0, 7.0, 15.0, 29.0])
    k = np.zeros((len(kk), 3))
    k[:, 1] = kk
    ball = 4 * np.pi * (np.sin(kk * R) - kk * R * np.cos(kk * R)) / kk ** 3
    shell = 4 * np.pi * R * np.sin(kk * R) / kk
    Fv = oracle.mesh_ft_forward(v, f, k, VOL)
    Fs = oracle.mesh_ft_forward(v, f, k, SURF)
    assert np.abs(Fv - ball).max() < 3e-3 * (4 / 3 * np.pi * R ** 3)
    assert np.abs(Fs - shell).max() < 3e-3 * (4 * np.pi * R ** 2)
    assert np.abs(Fv.imag).max() < 1e-12 and np.abs(Fs.imag).max() < 1e-12     # centred, symmetric


def test_bad_arguments_are_rejected():
    v, f = icosphere(0)
    bad = f.copy()
    bad[0, 0] = 99
    with pytest.raises(ValueError):
        oracle.mesh_ft_forward(v, bad, np.zeros((1, 3)), VOL)
    with pytest.raises(ValueError):
        oracle.mesh_ft_forward(v, f, np.zeros((1, 3)), 2)


def test_empty_mesh_and_empty_frequency_list():
    v, f = icosphere(0)
    assert oracle.mesh_ft_forward(v, f, np.zeros((0, 3)), VOL).shape == (0,)
    F = oracle.mesh_ft_forward(v, np.zeros((0, 3), np.int32), np.ones((3, 3)), SURF)
    assert np.all(F == 0)


def test_per_face_weights_are_linear_in_the_density():
    """PAPER.md:127 (reading R23): two nested closed surfaces with densities 1 and 0.5 in volume mode give the FT of
    a ball of density 1 minus half a ball -- i.e. F_outer - 0.5 F_inner with the inner sphere's faces weighted -0.5 --
    and F(0) is the weighted volume; in surface mode the weights scale each membrane's area."""
    from workloads import icosphere
    vo, fo = icosphere(2, 0.4)
    vi, fi = icosphere(1, 0.2, (0.03, 0.0, -0.02))
    v = np.vstack([vo, vi])
    f = np.vstack([fo, fi + len(vo)]).astype(np.int32)
    w = np.concatenate([np.ones(len(fo)), -0.5 * np.ones(len(fi))])
    k = np.random.default_rng(4).uniform(-30, 30, size=(25, 3))
    k[0] = 0
    for mode in (VOL, SURF):
        got = oracle.mesh_ft_forward_weighted(v, f, k, mode, w)
        want = oracle.mesh_ft_forward(vo, fo, k, mode) - 0.5 * oracle.mesh_ft_forward(vi, fi, k, mode)
        assert np.abs(got - want).max() <= 1e-13 * abs(want[0])
    vol = lambda vv, ff: np.einsum("ij,ij->i", vv[ff[:, 0]], np.cross(vv[ff[:, 1]], vv[ff[:, 2]])).sum() / 6.0
    assert abs(oracle.mesh_ft_forward_weighted(v, f, k[:1], VOL, w)[0] - (vol(vo, fo) - 0.5 * vol(vi, fi))) < 1e-14


def test_weighted_surface_forward_vs_gauss_quadrature():
    """Independent pin of oracle.mesh_ft_forward_weighted away from k = 0 (not its own linearity): per-face weights
    w_T times the tensor Gauss-Legendre quadrature of int_T e^{-ik.x} dS, three distinct weights incl. a negative one,
    assigned per face at random (reading R23)."""
    rng = np.random.default_rng(31)
    v, f = icosphere(1, 0.35, (0.02, 0.01, -0.03))
    v = perturb_radial(v, (0.02, 0.01, -0.03), 0.12, rng)
    wts = rng.choice([1.0, 0.4, -0.7], size=len(f))
    k = rng.uniform(-14, 14, (30, 3))
    x, w = np.polynomial.legendre.leggauss(32)
    x, w = 0.5 * (x + 1), 0.5 * w
    U, W = np.meshgrid(x, x, indexing="ij")
    wt = np.outer(w, w) * (1 - U)
    ref = np.zeros(len(k), dtype=complex)
    for t, tri in enumerate(f):
        p0, p1, p2 = v[tri]
        pts = p0 + U[..., None] * (p1 - p0) + (W * (1 - U))[..., None] * (p2 - p0)
        twoA = np.linalg.norm(np.cross(p1 - p0, p2 - p0))
        ref += wts[t] * twoA * np.einsum("ij,ijq->q", wt, np.exp(-1j * np.einsum("ijd,qd->ijq", pts, k)))
    got = oracle.mesh_ft_forward_weighted(v, f, k, SURF, wts)
    assert np.abs(got - ref).max() < 1e-12


def test_weighted_volume_forward_vs_per_face_divergence_terms():
    """Volume mode with per-face weights, away from k = 0: F_w(k) = (i/|k|^2) sum_T w_T (k.m_T) f_T(k) assembled face
    by face from one-triangle calls of the SURFACE-mode oracle (2 A_T f_T = the one-face surface FT, pinned by
    quadrature above), so neither the volume-mode code path nor the weight grouping is reused."""
    rng = np.random.default_rng(33)
    v, f = icosphere(1, 0.3, (-0.02, 0.03, 0.01))
    v = perturb_radial(v, (-0.02, 0.03, 0.01), 0.1, rng)
    wts = rng.choice([1.0, 0.5, -0.8], size=len(f))
    k = rng.uniform(-25, 25, (16, 3))
    want = np.zeros(len(k), dtype=complex)
    for t, tri in enumerate(f):
        p0, p1, p2 = v[tri]
        m = np.cross(p1 - p0, p2 - p0)
        surf = oracle.mesh_ft_forward(v, f[t:t + 1], k, SURF)          # |m_T| f_T(k)
        want += wts[t] * 1j * (k @ m) / np.linalg.norm(m) * surf / (k * k).sum(axis=1)
    got = oracle.mesh_ft_forward_weighted(v, f, k, VOL, wts)
    assert np.abs(got - want).max() < 1e-12 * np.abs(want).max()
