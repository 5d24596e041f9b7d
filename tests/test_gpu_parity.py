"""GPU parity: the CUDA path (through the C ABI binding) against the fp64 oracle, element by element.

Acceptance bars (BASELINE.json north_star):  forward max|dF| <= 1e-4 |F(0)|;  vertex gradient relative L2 <= 1e-3;
rendered image max abs diff <= 1e-4 max|image|.
"""
import numpy as np
import pytest

import oracle
from workloads import box_mesh, build_workload, icosphere, sampled_frequencies
from workloads.configs import image_cotangent, spectrum_cotangent

pytestmark = pytest.mark.gpu

FWD_TOL = 1e-4     # x |F(0)|
GRAD_TOL = 1e-3    # relative L2
IMG_TOL = 1e-4     # x max|image|


@pytest.fixture(scope="module")
def dm():
    import torch
    import paper_2303_10440_b200 as dm
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    dm.load_library()
    return dm


def _plan(dm, w, mode=None):
    import torch
    faces = torch.as_tensor(w.faces, device="cuda")
    return dm.Plan(w.n, w.spacing, w.origin, w.mode if mode is None else mode, faces, w.vertices.shape[0])


def _dev(a):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a), device="cuda")


def _rel_l2(a, b):
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def _forward_full(dm, w, mode):
    plan = _plan(dm, w, mode)
    F = plan.mesh_ft_forward(_dev(w.vertices)).cpu().numpy()
    ref = oracle.mesh_ft_forward_grid(w.vertices, w.faces, w.n, w.spacing, mode)
    return F, ref


@pytest.mark.parametrize("mode", [0, 1])
def test_forward_cfg1_full_grid(dm, mode):
    w = build_workload(1)
    F, ref = _forward_full(dm, w, mode)
    assert np.isfinite(F).all()
    err = np.abs(F - ref).max() / abs(ref[0, 0, 0])
    assert err <= FWD_TOL, err
    # the k = 0 entry (row A5) is the volume / area to fp32 rounding
    assert abs(F[0, 0, 0] - ref[0, 0, 0]) <= 2e-7 * abs(ref[0, 0, 0])


@pytest.mark.parametrize("mode", [0, 1])
def test_forward_box_exact_degeneracies(dm, mode):
    """Axis-aligned box on its own lattice: a=b and a=b=c hold exactly for axis-aligned k (eq. 15/16 cases), and
    the ragged grid (24x20x18, not a multiple of any tile) exercises the tails."""
    c = np.array([0.05, -0.02, 0.1])
    h = np.array([0.2, 0.15, 0.1])
    v, f = box_mesh(c, h)
    n = (24, 20, 18)
    spacing = (1 / 24, 1 / 20, 1 / 18)
    import torch
    plan = dm.Plan(n, spacing, (0, 0, 0), mode, torch.as_tensor(f, device="cuda"), v.shape[0])
    v32 = v.astype(np.float32)
    F = plan.mesh_ft_forward(_dev(v32)).cpu().numpy()
    ref = oracle.mesh_ft_forward_grid(v32, f, n, spacing, mode)
    assert np.abs(F - ref).max() <= FWD_TOL * abs(ref[0, 0, 0])


@pytest.mark.parametrize("mode", [0, 1])
def test_forward_cfg2_shape_reduced_grid(dm, mode):
    """cfg-2 mesh (5120 perturbed triangles: several triangle tiles + tail) on a 24x24x24 grid the oracle finishes
    in seconds."""
    w = build_workload(2, grid_override=(24, 24, 24))
    F, ref = _forward_full(dm, w, mode)
    assert np.abs(F - ref).max() <= FWD_TOL * abs(ref[0, 0, 0])


@pytest.mark.parametrize("mode", [0, 1])
def test_forward_anisotropic_offcentre(dm, mode):
    """Off-centre mesh partly outside the box on an anisotropic grid with L != 1 (exact phase reduction must use
    v/L mod 1, reading R10)."""
    v, f = icosphere(2, 0.45, (0.5, -0.3, 0.2))
    v32 = v.astype(np.float32)
    n = (16, 12, 20)
    spacing = (0.11, 0.13, 0.07)
    import torch
    plan = dm.Plan(n, spacing, (-0.8, -0.7, -0.6), mode, torch.as_tensor(f, device="cuda"), v.shape[0])
    F = plan.mesh_ft_forward(_dev(v32)).cpu().numpy()
    ref = oracle.mesh_ft_forward_grid(v32, f, n, spacing, mode)
    assert np.abs(F - ref).max() <= FWD_TOL * abs(ref[0, 0, 0])


@pytest.mark.parametrize("mode", [0, 1])
def test_backward_cfg1_full_grid(dm, mode):
    w = build_workload(1)
    G = spectrum_cotangent(w)
    plan = _plan(dm, w, mode)
    dv = plan.mesh_ft_backward(_dev(w.vertices), _dev(G)).cpu().numpy()
    ref = oracle.mesh_ft_backward_grid(w.vertices, w.faces, w.n, w.spacing, mode, G.astype(np.complex128))
    assert np.isfinite(dv).all()
    assert _rel_l2(dv, ref) <= GRAD_TOL
    # run-to-run bitwise reproducibility (atomic-free reduction + CSR gather, reading R22)
    dv2 = plan.mesh_ft_backward(_dev(w.vertices), _dev(G)).cpu().numpy()
    assert np.array_equal(dv, dv2)


@pytest.mark.parametrize("mode", [0, 1])
def test_backward_identity_P9(dm, mode):
    """sum_v dL/dv = sum_k Re(conj(G) (-i k) F(k)) -- exact identity, all on the GPU results (pin P9)."""
    w = build_workload(2, grid_override=(16, 16, 16))
    G = spectrum_cotangent(w)
    plan = _plan(dm, w, mode)
    vd = _dev(w.vertices)
    F = plan.mesh_ft_forward(vd).cpu().numpy().astype(np.complex128)
    dv = plan.mesh_ft_backward(vd, _dev(G)).cpu().numpy().astype(np.float64)
    k = oracle.frequency_grid(w.n, w.spacing)
    rhs = np.einsum("xyz,xyzd->d", np.real(np.conj(G.astype(np.complex128)) * (-1j) * F), k)
    scale = np.abs(dv).sum(axis=0)
    assert np.all(np.abs(dv.sum(axis=0) - rhs) <= 1e-4 * scale)


@pytest.mark.parametrize("mode", [0, 1])
def test_backward_cfg2_shape_reduced_grid(dm, mode):
    w = build_workload(2, grid_override=(16, 16, 16))
    G = spectrum_cotangent(w)
    plan = _plan(dm, w, mode)
    dv = plan.mesh_ft_backward(_dev(w.vertices), _dev(G)).cpu().numpy()
    ref = oracle.mesh_ft_backward_grid(w.vertices, w.faces, w.n, w.spacing, mode, G.astype(np.complex128))
    assert _rel_l2(dv, ref) <= GRAD_TOL


def test_slab_partition_matches_whole_grid(dm):
    """Two x-slabs reproduce the whole-grid forward bit for bit and their partial gradients add up."""
    w = build_workload(1)
    G = spectrum_cotangent(w)
    vd, Gd = _dev(w.vertices), _dev(G)
    plan = _plan(dm, w)
    F = plan.mesh_ft_forward(vd).clone()
    dv = plan.mesh_ft_backward(vd, Gd).cpu().numpy()
    import torch
    F2 = torch.zeros_like(F)
    parts = []
    for lo, hi in ((0, 13), (13, 32)):
        plan.set_slab(lo, hi)
        plan.mesh_ft_forward(vd, out=F2)
        parts.append(plan.mesh_ft_backward(vd, Gd).cpu().numpy())
    assert torch.equal(F, F2)
    assert _rel_l2(parts[0] + parts[1], dv) <= 1e-5


def test_render_and_backward_cfg1(dm):
    w = build_workload(1)
    plan = _plan(dm, w)
    vd = _dev(w.vertices)
    img = plan.render(vd, w.psf_cov).cpu().numpy()
    ref = oracle.render(w.vertices, w.faces, w.n, w.spacing, w.origin, w.psf_cov.astype(np.float64), w.mode)
    assert np.abs(img - ref).max() <= IMG_TOL * np.abs(ref).max()
    gi = image_cotangent(w)
    dv = plan.render_backward(vd, w.psf_cov, _dev(gi)).cpu().numpy()
    dref = oracle.render_backward(w.vertices, w.faces, w.n, w.spacing, w.origin, w.psf_cov.astype(np.float64), w.mode, gi)
    assert _rel_l2(dv, dref) <= GRAD_TOL
    ms = plan.stage_ms()
    assert ms["mesh_ft"] > 0 and ms["fft"] > 0 and ms["psf"] > 0 and ms["scatter"] > 0


def test_inverse_transform_semantics_R13(dm):
    """spectrum_to_image on a deliberately NON-Hermitian half spectrum equals numpy irfftn (reading R13), and
    image_to_spectrum_cotangent is its adjoint on independent stored entries (pin P11, reading R14)."""
    import torch
    n = (12, 10, 8)
    spacing = (0.1, 0.12, 0.09)
    origin = (-0.55, -0.6, -0.3)
    cov = [0.02, 0.03, 0.015, 0.004, -0.003, 0.002]
    v, f = icosphere(0, 0.3)
    plan = dm.Plan(n, spacing, origin, 0, torch.as_tensor(f, device="cuda"), v.shape[0])
    rng = np.random.default_rng(5)
    shape = (n[0], n[1], n[2] // 2 + 1)
    F = (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)).astype(np.complex64)
    img = plan.spectrum_to_image(_dev(F), cov).cpu().numpy()
    ref = oracle.spectrum_to_image(F, n, spacing, origin, cov)
    assert np.abs(img - ref).max() <= 1e-5 * np.abs(ref).max()
    y = rng.standard_normal(n).astype(np.float32)
    Gy = plan.image_to_spectrum_cotangent(_dev(y), cov).cpu().numpy()
    Gref = oracle.image_to_spectrum_cotangent(y, n, spacing, origin, cov)
    assert np.abs(Gy - Gref).max() <= 1e-5 * np.abs(Gref).max()
    lhs = float((img.astype(np.float64) * y).sum())
    rhs = float(np.real(np.conj(Gy.astype(np.complex128)) * F).sum())
    assert abs(lhs - rhs) <= 1e-4 * max(abs(lhs), 1.0)


def test_error_codes(dm):
    import torch
    v, f = icosphere(0, 0.3)
    bad = f.copy()
    bad[3, 1] = 99
    with pytest.raises(dm.DeltamicError) as e:
        dm.Plan((8, 8, 8), (1 / 8,) * 3, (0, 0, 0), 0, torch.as_tensor(bad, device="cuda"), v.shape[0])
    assert e.value.code == -2
    with pytest.raises(dm.DeltamicError) as e:
        dm.Plan((8, 8, 7), (1 / 8,) * 3, (0, 0, 0), 0, torch.as_tensor(f, device="cuda"), v.shape[0])
    assert e.value.code == -1
    plan = dm.Plan((8, 8, 8), (1 / 8,) * 3, (0, 0, 0), 0, torch.as_tensor(f, device="cuda"), v.shape[0])
    with pytest.raises(dm.DeltamicError):
        plan.set_slab(4, 4)


def test_psf_gradient_cfg1_and_full_covariance(dm):
    """NEXT 2: dL/dSigma from dm_render_backward against the oracle (relative error <= 1e-3 of the largest entry), with
    config 1's diagonal PSF and with a full covariance on an anisotropic grid; the vertex gradient of the same call
    must equal the one of a call without the PSF gradient, bit for bit."""
    import torch
    w = build_workload(1)
    cases = [(w.n, w.spacing, w.origin, w.psf_cov.astype(np.float64)),
             ((24, 32, 16), (1 / 24, 1 / 32, 1 / 8), (-0.5 + 1 / 48, -0.5 + 1 / 64, -1.0 + 1 / 16),
              np.array([0.0020, 0.0016, 0.0300, 0.0004, -0.0015, 0.0011]))]
    for n, spacing, origin, cov in cases:
        for mode in (0, 1):
            plan = dm.Plan(n, spacing, origin, mode, torch.as_tensor(w.faces, device="cuda"), w.vertices.shape[0])
            vd = torch.as_tensor(w.vertices, device="cuda")
            y = np.random.default_rng(3).standard_normal(n).astype(np.float32)
            yd = torch.as_tensor(y, device="cuda")
            dv0 = plan.render_backward(vd, cov, yd).clone()
            dv, dcov = plan.render_backward(vd, cov, yd, with_psf_grad=True)
            assert torch.equal(dv, dv0)
            ref = oracle.render_backward_psf(w.vertices, w.faces, n, spacing, origin, cov, mode, y.astype(np.float64))
            err = np.abs(np.array(dcov) - ref).max() / np.abs(ref).max()
            print(f"psf gradient n={n} mode={mode}: max err / max|dL/dSigma| = {err:.2e}")
            assert err <= 1e-3, (dcov, ref)
            plan.close()


def _band_mask(w, cov, cutoff):
    """In-band mask of the stored grid in fp64 and the mask of frequencies too close to the boundary to call."""
    k = oracle.frequency_grid(w.n, w.spacing)
    S = np.array([[cov[0], cov[3], cov[4]], [cov[3], cov[1], cov[5]], [cov[4], cov[5], cov[2]]], dtype=np.float64)
    quad = 0.5 * np.einsum("...i,ij,...j->...", k, S, k)
    lim = np.log(1.0 / cutoff)
    return quad < lim, np.abs(quad - lim) < 1e-4 * lim


@pytest.mark.parametrize("mode", [0, 1])
def test_narrow_band_forward_and_backward(dm, mode):
    """NEXT 1: with the band set, the forward equals the oracle inside the band and is exactly zero
    outside; the backward equals the oracle's gradient summed over the in-band frequencies only.  Anisotropic grid and
    a full covariance, so the band is a tilted ellipsoid cut by the grid."""
    import torch
    w = build_workload(2, subdiv_override=2, grid_override=(24, 32, 40))
    cov = np.array([1.2e-3, 0.7e-3, 4.5e-3, 2.0e-4, -0.8e-3, 3.0e-4])
    cutoff = 0.02
    inb, edge = _band_mask(w, cov, cutoff)
    assert 0.03 < inb.mean() < 0.7 and inb[0, 0, 0]
    plan, vd = _plan(dm, w, mode), _dev(w.vertices)
    plan.set_narrow_band(cov, cutoff)
    F = plan.mesh_ft_forward(vd).cpu().numpy()
    ref = oracle.mesh_ft_forward_grid(w.vertices, w.faces, w.n, w.spacing, mode)
    f0 = abs(ref[0, 0, 0])
    sure_in, sure_out = inb & ~edge, ~inb & ~edge
    assert np.abs(F - ref)[sure_in].max() <= FWD_TOL * f0
    assert (F[sure_out] == 0).all()
    G = spectrum_cotangent(w)
    G[edge] = 0
    dv = plan.mesh_ft_backward(vd, _dev(G)).cpu().numpy()
    idx = np.nonzero(sure_in.reshape(-1))[0]
    dref = oracle.mesh_ft_backward_grid(w.vertices, w.faces, w.n, w.spacing, mode, G.reshape(-1)[idx].astype(np.complex128),
                                        flat_indices=idx)
    assert _rel_l2(dv, dref) <= GRAD_TOL
    # the robust kernels honour the band too
    plan.set_option(dm.DM_OPT_FORWARD_PATH, 1)
    plan.set_option(dm.DM_OPT_BACKWARD_PATH, 1)
    Fr = plan.mesh_ft_forward(vd).cpu().numpy()
    assert np.abs(Fr - ref)[sure_in].max() <= FWD_TOL * f0 and (Fr[sure_out] == 0).all()
    assert _rel_l2(plan.mesh_ft_backward(vd, _dev(G)).cpu().numpy(), dref) <= GRAD_TOL
    # switching the band off restores the whole grid
    plan.set_option(dm.DM_OPT_FORWARD_PATH, 0)
    plan.set_narrow_band(None)
    F2 = plan.mesh_ft_forward(vd).cpu().numpy()
    assert np.abs(F2 - ref).max() <= FWD_TOL * f0
    plan.close()


def test_area_normalised_density_eq12_eq13(dm):
    """NEXT 3: u = F/|Lambda| and its gradient against the oracle on a full small grid."""
    w = build_workload(2, subdiv_override=2, grid_override=(16, 16, 16))
    plan, vd = _plan(dm, w, 1), _dev(w.vertices)
    plan.set_option(dm.DM_OPT_AREA_NORMALISED, 1)
    k = oracle.frequency_grid(w.n, w.spacing).reshape(-1, 3)
    u = plan.mesh_ft_forward(vd).cpu().numpy()
    uref = oracle.mesh_ft_forward_normalised(w.vertices, w.faces, k).reshape(u.shape)
    assert abs(u[0, 0, 0] - 1.0) <= 1e-6
    assert np.abs(u - uref).max() <= FWD_TOL          # |u(0)| = 1
    G = spectrum_cotangent(w)
    dv = plan.mesh_ft_backward(vd, _dev(G)).cpu().numpy()
    dref = oracle.mesh_ft_backward_normalised(w.vertices, w.faces, k, G.reshape(-1).astype(np.complex128))
    assert _rel_l2(dv, dref) <= GRAD_TOL
    plan.close()
    with pytest.raises(dm.DeltamicError):             # volume mode has no area normalisation
        _plan(dm, w, 0).set_option(dm.DM_OPT_AREA_NORMALISED, 1)


def test_degenerate_and_non_manifold_meshes_surface_mode(dm):
    """Edge cases of the input (readings R19, R20): a non-manifold "book" of four triangles on one edge, a zero-area
    triangle, a face that repeats a vertex, an isolated vertex no face uses, a single-triangle mesh and the smallest
    grid (2 x 2 x 2).  Surface mode is a plain sum over triangles, so the oracle defines every case; forward and
    backward (box-exact degeneracies included: the book's spine lies on the z axis) must match it."""
    import torch
    v = np.array([[0, 0, -0.2], [0, 0, 0.2], [0.3, 0, 0], [0, 0.25, 0.05], [-0.2, -0.1, 0], [0.1, -0.3, 0.1],
                  [0.05, 0.05, 0.05], [0.4, 0.4, 0.4]], dtype=np.float32)          # vertex 7 is used by no face
    f = np.array([[0, 1, 2], [0, 1, 3], [1, 0, 4], [0, 1, 5],                      # four pages on the edge (0,1)
                  [2, 6, 6],                                                        # repeated vertex (zero area)
                  [2, 3, 2]], dtype=np.int32)                                       # repeated vertex again
    vz = v.copy()
    vz = np.vstack([vz, 0.5 * (vz[2] + vz[3])[None]])                               # vertex 8 = midpoint of (2,3)
    fz = np.vstack([f, [[2, 8, 3]]]).astype(np.int32)                               # collinear: zero area, distinct vertices
    cases = [(vz.astype(np.float32), fz, (12, 10, 8)), (v[:3].copy(), f[:1].copy(), (8, 8, 8)), (v[:3].copy(), f[:1].copy(), (2, 2, 2))]
    for vv, ff, n in cases:
        spacing = tuple(1.0 / x for x in n)
        plan = dm.Plan(n, spacing, (0, 0, 0), 1, torch.as_tensor(ff, device="cuda"), vv.shape[0])
        F = plan.mesh_ft_forward(_dev(vv)).cpu().numpy()
        ref = oracle.mesh_ft_forward_grid(vv, ff, n, spacing, 1)
        assert np.isfinite(F.view(np.float32)).all()
        assert np.abs(F - ref).max() <= FWD_TOL * abs(ref[0, 0, 0])
        rng = np.random.default_rng(17)
        G = (rng.standard_normal(ref.shape) + 1j * rng.standard_normal(ref.shape)).astype(np.complex64)
        dv = plan.mesh_ft_backward(_dev(vv), _dev(G)).cpu().numpy()
        dref = oracle.mesh_ft_backward_grid(vv, ff, n, spacing, 1, G.astype(np.complex128))
        assert np.isfinite(dv).all()
        assert _rel_l2(dv, dref) <= GRAD_TOL, (n, _rel_l2(dv, dref))
        unused = sorted(set(range(vv.shape[0])) - set(ff.reshape(-1).tolist()))
        assert (dv[unused] == 0).all()                                              # no face, no gradient
        plan.close()


@pytest.mark.parametrize("mode", [0, 1])
def test_odd_grid_sizes_and_non_unit_box(dm, mode):
    """Odd N_x, N_y (no Nyquist rows), a box that is not the unit cube and a mesh that is not centred: forward, backward
    and render against the oracle on the full grid."""
    import torch
    n = (15, 9, 10)
    spacing = (0.07, 0.11, 0.13)
    origin = (-0.4, -0.5, -0.6)
    v, f = icosphere(2, 0.31, (0.05, -0.04, 0.02))
    v = v.astype(np.float32)
    plan = dm.Plan(n, spacing, origin, mode, torch.as_tensor(f, device="cuda"), v.shape[0])
    F = plan.mesh_ft_forward(_dev(v)).cpu().numpy()
    ref = oracle.mesh_ft_forward_grid(v, f, n, spacing, mode)
    assert np.abs(F - ref).max() <= FWD_TOL * abs(ref[0, 0, 0])
    rng = np.random.default_rng(23)
    G = (rng.standard_normal(ref.shape) + 1j * rng.standard_normal(ref.shape)).astype(np.complex64)
    dv = plan.mesh_ft_backward(_dev(v), _dev(G)).cpu().numpy()
    assert _rel_l2(dv, oracle.mesh_ft_backward_grid(v, f, n, spacing, mode, G.astype(np.complex128))) <= GRAD_TOL
    cov = np.array([0.012, 0.02, 0.03, 0.002, -0.004, 0.003])
    img = plan.render(_dev(v), cov).cpu().numpy()
    iref = oracle.render(v, f, n, spacing, origin, cov, mode)
    assert np.abs(img - iref).max() <= IMG_TOL * np.abs(iref).max()
    y = rng.standard_normal(n).astype(np.float32)
    dvr = plan.render_backward(_dev(v), cov, _dev(y)).cpu().numpy()
    assert _rel_l2(dvr, oracle.render_backward(v, f, n, spacing, origin, cov, mode, y.astype(np.float64))) <= GRAD_TOL
    plan.close()


@pytest.mark.parametrize("mode", [0, 1])
def test_per_face_density_weights(dm, mode):
    """PAPER.md:127 (reading R23): two nested surfaces with weights 1 and -0.5 (a shell of density 1 around a core of
    density 0.5 in volume mode): forward and backward of the fast and the robust kernels against the oracle."""
    import torch
    vo, fo = icosphere(2, 0.4)
    vi, fi = icosphere(2, 0.2, (0.03, 0.0, -0.02))
    v = np.vstack([vo, vi]).astype(np.float32)
    f = np.vstack([fo, fi + len(vo)]).astype(np.int32)
    wts = np.concatenate([np.ones(len(fo)), -0.5 * np.ones(len(fi))]).astype(np.float32)
    n, spacing = (16, 20, 12), (1 / 16, 1 / 20, 1 / 12)
    k = oracle.frequency_grid(n, spacing).reshape(-1, 3)
    plan = dm.Plan(n, spacing, (0, 0, 0), mode, torch.as_tensor(f, device="cuda"), v.shape[0])
    plan.set_face_weights(_dev(wts))
    ref = oracle.mesh_ft_forward_weighted(v, f, k, mode, wts)
    G = spectrum_cotangent(build_workload(1, grid_override=n))
    dref = oracle.mesh_ft_backward_weighted(v, f, k, mode, G.reshape(-1).astype(np.complex128), wts)
    for path in (0, 1):
        plan.set_option(dm.DM_OPT_FORWARD_PATH, path)
        plan.set_option(dm.DM_OPT_BACKWARD_PATH, path)
        F = plan.mesh_ft_forward(_dev(v)).cpu().numpy().reshape(-1)
        assert np.abs(F - ref).max() <= FWD_TOL * abs(ref[0]), path
        dv = plan.mesh_ft_backward(_dev(v), _dev(G)).cpu().numpy()
        assert _rel_l2(dv, dref) <= GRAD_TOL, path
    # the no-synchronisation update with a caller-asserted class: same routing and same bits as the classifying call
    plan.set_option(dm.DM_OPT_FORWARD_PATH, 0)
    plan.set_option(dm.DM_OPT_BACKWARD_PATH, 0)
    for wset, robust in ((wts, True), (np.abs(wts) * 1.5, False)):        # mixed signs -> robust; one sign per component -> fast
        plan.set_face_weights(_dev(wset))
        Fa = plan.mesh_ft_forward(_dev(v))
        dva = plan.mesh_ft_backward(_dev(v), _dev(G))
        assert plan.paths_used() == ((1, 1) if robust else (0, 0))
        plan.update_face_weights(_dev(np.ones_like(wset)), robust=False)    # something else in between
        plan.update_face_weights(_dev(wset), robust=robust)
        assert torch.equal(plan.mesh_ft_forward(_dev(v)), Fa) and torch.equal(plan.mesh_ft_backward(_dev(v), _dev(G)), dva)
        assert plan.paths_used() == ((1, 1) if robust else (0, 0))
    plan.set_face_weights(None)
    F1 = plan.mesh_ft_forward(_dev(v)).cpu().numpy().reshape(-1)
    assert np.abs(F1 - oracle.mesh_ft_forward(v, f, k, mode)).max() <= FWD_TOL * abs(ref[0])
    plan.close()


def test_sharded_backward_helper_single_rank_and_emulated_ranks(dm):
    """paper_2303_10440_b200.sharding on the GPU: without a process group the helper is the whole-grid backward; the
    partial gradients of the slabs of three emulated ranks (run one after the other, as the profiling guide asks for
    multi-rank paths on one GPU) add up to it."""
    import torch
    from paper_2303_10440_b200.sharding import sharded_mesh_ft_backward, slab_bounds
    w = build_workload(2, subdiv_override=2, grid_override=(20, 16, 16))
    plan, vd = _plan(dm, w), _dev(w.vertices)
    Gd = _dev(spectrum_cotangent(w))
    whole = plan.mesh_ft_backward(vd, Gd).clone()
    assert torch.equal(sharded_mesh_ft_backward(plan, vd, Gd), whole)
    total = torch.zeros_like(whole)
    for rank in range(3):
        b, e = slab_bounds(w.n[0], 3, rank)
        plan.set_slab(b, e)
        total += plan.mesh_ft_backward(vd, Gd)
    plan.set_slab(0, w.n[0])
    assert float(torch.linalg.norm(total - whole) / torch.linalg.norm(whole)) <= 1e-5
    plan.close()


@pytest.mark.parametrize("mode", [0, 1])
def test_coarse_meshes_large_gaps(dm, mode):
    """Meshes that are coarse for the grid (|k| h up to ~90, the regime of the paper's 80-triangle sphere of Fig. 6,
    PAPER.md:221): a 20-triangle and an 80-triangle sphere, and a fine sphere next to a coarse one.  The flag thresholds
    scale with (|k| h)^3 there; forward and gradient must stay within the tolerances."""
    import torch
    rng = np.random.default_rng(35)
    meshes = []
    for sub, R in ((0, 0.4), (1, 0.3)):
        v, f = icosphere(sub, R, (0.03, -0.02, 0.05))
        meshes.append((v.astype(np.float32), f))
    va, fa = icosphere(0, 0.17, (-0.25, 0.1, 0.05))
    vb, fb = icosphere(2, 0.15, (0.2, -0.1, 0.0))
    meshes.append((np.vstack([va, vb]).astype(np.float32), np.vstack([fa, fb + len(va)]).astype(np.int32)))
    n, spacing = (38, 22, 24), (1.35 / 38, 1.53 / 22, 0.77 / 24)
    for v, f in meshes:
        plan = dm.Plan(n, spacing, (-0.6, -0.7, -0.35), mode, torch.as_tensor(f, device="cuda"), v.shape[0])
        F = plan.mesh_ft_forward(_dev(v)).cpu().numpy()
        ref = oracle.mesh_ft_forward_grid(v, f, n, spacing, mode)
        assert np.abs(F - ref).max() <= FWD_TOL * abs(ref[0, 0, 0])
        G = (rng.standard_normal(ref.shape) + 1j * rng.standard_normal(ref.shape)).astype(np.complex64)
        dv = plan.mesh_ft_backward(_dev(v), _dev(G)).cpu().numpy()
        dref = oracle.mesh_ft_backward_grid(v, f, n, spacing, mode, G.astype(np.complex128))
        assert _rel_l2(dv, dref) <= GRAD_TOL, (len(f), _rel_l2(dv, dref))
        plan.close()


@pytest.mark.parametrize("mode", [0, 1])
def test_stretched_meshes_and_outlier_faces(dm, mode):
    """Anisotropically scaled meshes (aspect ratio up to 6) with a second, much finer or coarser component: the longest
    edge is several times the RMS edge, so the low-k kernel's ball shrinks and single faces are coarse for frequencies
    at which the mesh as a whole is not ("Stretched meshes and outlier faces")."""
    import torch
    from workloads.meshes import perturb_radial
    rng = np.random.default_rng(73)
    cases = []
    c = np.array([-0.08, 0.02, 0.05])
    v, f = icosphere(3, 0.3, c)
    v = c + (perturb_radial(v, c, 0.08, rng) - c) * np.array([0.9, 0.2, 1.3])
    v2, f2 = icosphere(1, 0.2, (0.02, 0.1, -0.2))
    v2 = v2 * np.array([0.3, 1.4, 1.0])
    cases.append((np.vstack([v, v2]), np.vstack([f, f2 + len(v)]), (33, 18, 16), (1.13, 1.66, 1.09)))
    c = np.array([0.05, 0.1, 0.06])
    v, f = icosphere(1, 0.42, c)
    v = c + (perturb_radial(v, c, 0.08, rng) - c) * np.array([1.25, 1.5, 1.4])
    v2, f2 = icosphere(2, 0.1, (-0.3, -0.35, -0.3))
    cases.append((np.vstack([v, v2]), np.vstack([f, f2 + len(v)]), (36, 34, 28), (1.58, 1.99, 1.72)))
    for v, f, n, L in cases:
        v, f = v.astype(np.float32), f.astype(np.int32)
        spacing = tuple(np.array(L) / np.array(n))
        origin = tuple(-np.array(L) / 2 + 0.3 * np.array(spacing))
        plan = dm.Plan(n, spacing, origin, mode, torch.as_tensor(f, device="cuda"), v.shape[0])
        F = plan.mesh_ft_forward(_dev(v)).cpu().numpy()
        ref = oracle.mesh_ft_forward_grid(v, f, n, spacing, mode)
        assert np.abs(F - ref).max() <= FWD_TOL * abs(ref[0, 0, 0]), (len(f), np.abs(F - ref).max() / abs(ref[0, 0, 0]))
        G = (rng.standard_normal(ref.shape) + 1j * rng.standard_normal(ref.shape)).astype(np.complex64)
        dv = plan.mesh_ft_backward(_dev(v), _dev(G)).cpu().numpy()
        dref = oracle.mesh_ft_backward_grid(v, f, n, spacing, mode, G.astype(np.complex128))
        assert _rel_l2(dv, dref) <= GRAD_TOL, (len(f), _rel_l2(dv, dref))
        plan.close()


@pytest.mark.parametrize("mode", [0, 1])
def test_tall_grid_fast_kernels(dm, mode):
    """A grid much longer along z than one super-segment of the backward kernel (N_z/2+1 = 321 > 288: two super-segments
    with their own exact start phases, 32-frequency seed spacing) -- the paper's image sizes go up to 2048^3
    (PAPER.md:59).  Both passes must stay on the fast kernels and match the oracle on the full grid."""
    w = build_workload(1, grid_override=(16, 16, 640))
    G = spectrum_cotangent(w)
    plan = _plan(dm, w, mode)
    vd = _dev(w.vertices)
    F = plan.mesh_ft_forward(vd).cpu().numpy()
    ref = oracle.mesh_ft_forward_grid(w.vertices, w.faces, w.n, w.spacing, mode)
    assert np.abs(F - ref).max() <= FWD_TOL * abs(ref[0, 0, 0])
    dv = plan.mesh_ft_backward(vd, _dev(G)).cpu().numpy()
    assert plan.paths_used() == (0, 0)
    dref = oracle.mesh_ft_backward_grid(w.vertices, w.faces, w.n, w.spacing, mode, G.astype(np.complex128))
    assert _rel_l2(dv, dref) <= GRAD_TOL
    # the same under a narrow band that cuts the rows short at different z
    cov = (np.array([2.0, 2.0, 3.0]) * np.array(w.spacing)) ** 2
    plan.set_narrow_band([cov[0], cov[1], cov[2], 0.0, 0.0, 0.0], 0.01)
    dvb = plan.mesh_ft_backward(vd, _dev(G)).cpu().numpy()
    Fb = plan.mesh_ft_forward(vd).cpu().numpy()
    inb = Fb != 0
    inb[0, 0, 0] = True
    Gb = np.where(inb, G, 0).astype(np.complex128)
    drefb = oracle.mesh_ft_backward_grid(w.vertices, w.faces, w.n, w.spacing, mode, Gb)
    assert _rel_l2(dvb, drefb) <= GRAD_TOL
    plan.close()


def test_reuse_of_the_render_spectrum(dm):
    """DM_OPT_REUSE_SPECTRUM / dm_mesh_ft_backward_with_spectrum (shape and PSF are fitted in one
    loop): the PSF gradient and eq. 13's extra term computed from the spectrum the forward call already produced must
    equal the recomputing path, use fewer launches, and refuse to run when the plan holds no such spectrum."""
    import torch
    w = build_workload(2, subdiv_override=2, grid_override=(24, 20, 16))
    cov = w.psf_cov.astype(np.float64)
    y = torch.as_tensor(np.random.default_rng(5).standard_normal(w.n).astype(np.float32), device="cuda")
    for mode, normalised in ((0, False), (1, False), (1, True)):
        plan, vd = _plan(dm, w, mode), _dev(w.vertices)
        if normalised:
            plan.set_option(dm.DM_OPT_AREA_NORMALISED, 1)
        plan.render(vd, cov)
        n0 = plan.launch_count()
        dv_a, dc_a = plan.render_backward(vd, cov, y, with_psf_grad=True)
        n_recompute = plan.launch_count() - n0
        dv_a = dv_a.clone()
        plan.set_option(dm.DM_OPT_REUSE_SPECTRUM, 1)
        with pytest.raises(dm.DeltamicError):          # the option change invalidated nothing, but the recompute did
            plan.render_backward(vd, cov, y, with_psf_grad=True)
        plan.render(vd, cov)
        n0 = plan.launch_count()
        dv_b, dc_b = plan.render_backward(vd, cov, y, with_psf_grad=True)
        n_reuse = plan.launch_count() - n0
        assert n_reuse < n_recompute
        assert torch.equal(dv_a, dv_b) or _rel_l2(dv_b.cpu().numpy(), dv_a.cpu().numpy()) <= 1e-6
        assert np.allclose(dc_a, dc_b, rtol=1e-5, atol=1e-6 * np.abs(dc_a).max())
        dv_c = plan.render_backward(vd, cov, y)        # may be called again: the spectrum stays valid
        assert _rel_l2(dv_c.cpu().numpy(), dv_a.cpu().numpy()) <= 1e-6
        plan.mesh_ft_forward(vd)                       # any other forward call invalidates it
        if normalised:
            with pytest.raises(dm.DeltamicError):
                plan.render_backward(vd, cov, y)
        plan.close()
    # the mesh-FT pair of calls with the area-normalised density
    plan, vd = _plan(dm, w, 1), _dev(w.vertices)
    plan.set_option(dm.DM_OPT_AREA_NORMALISED, 1)
    G = _dev(spectrum_cotangent(w))
    u = plan.mesh_ft_forward(vd)
    n0 = plan.launch_count()
    d1 = plan.mesh_ft_backward(vd, G).clone()
    n1 = plan.launch_count() - n0
    u = plan.mesh_ft_forward(vd)
    n0 = plan.launch_count()
    d2 = plan.mesh_ft_backward(vd, G, spectrum=u)
    n2 = plan.launch_count() - n0
    assert n2 < n1 and _rel_l2(d2.cpu().numpy(), d1.cpu().numpy()) <= 1e-6
    plan.close()


@pytest.mark.parametrize("n", [(2, 2, 4096), (4096, 1, 2), (1, 4096, 4)])
def test_maximum_grid_extents(dm, n):
    """The largest extent the plan accepts (4096 voxels) on each axis in turn, tiny on the others: N_z/2+1 = 2049 stored
    z-frequencies (the 12-bit frequency field of the backward's queue entries, eight super-segments per row), 4096 rows
    along x or y (row bookkeeping of the k-splits, fftfreq wrap of the row phases).  Surface mode, full grid vs the oracle."""
    w = build_workload(1, grid_override=n)
    G = spectrum_cotangent(w)
    plan = _plan(dm, w, 1)
    vd = _dev(w.vertices)
    F = plan.mesh_ft_forward(vd).cpu().numpy()
    ref = oracle.mesh_ft_forward_grid(w.vertices, w.faces, w.n, w.spacing, 1)
    assert np.abs(F - ref).max() <= FWD_TOL * abs(ref[0, 0, 0])
    dv = plan.mesh_ft_backward(vd, _dev(G)).cpu().numpy()
    assert plan.paths_used() == (0, 0)
    dref = oracle.mesh_ft_backward_grid(w.vertices, w.faces, w.n, w.spacing, 1, G.astype(np.complex128))
    assert _rel_l2(dv, dref) <= GRAD_TOL
    plan.close()
    import torch
    with pytest.raises(dm.DeltamicError):                                # one voxel more is refused, not mis-computed
        dm.Plan((4098, 2, 2), (1 / 4098, 0.5, 0.5), (0, 0, 0), 1, torch.as_tensor(w.faces, device="cuda"), w.vertices.shape[0])


def test_cuda_graph_capture_of_an_optimisation_step(dm):
    """dm_plan_set_stream: forward + backward, and a whole shape-optimisation step (render, Phi_1, backward, the two
    cooperative CG solves, AdamUniform), captured into CUDA graphs after one eager warm-up and replayed: same bits as the
    eager calls, no synchronisation inside."""
    import torch
    w = build_workload(1)
    plan, vd = _plan(dm, w, 0), _dev(w.vertices)
    Gd = _dev(spectrum_cotangent(w))
    F = torch.empty(w.spectrum_shape, dtype=torch.complex64, device="cuda")
    dv = torch.empty((w.vertices.shape[0], 3), dtype=torch.float32, device="cuda")
    plan.mesh_ft_forward(vd, out=F)
    plan.mesh_ft_backward(vd, Gd, out=dv)                 # eager warm-up: allocates the workspace
    F0, dv0 = F.clone(), dv.clone()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        plan.set_stream()                                  # the capturing stream
        plan.mesh_ft_forward(vd, out=F)
        plan.mesh_ft_backward(vd, Gd, out=dv)
    plan.set_stream()
    F.zero_()
    dv.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(F, F0) and torch.equal(dv, dv0)
    # a shape step: three eager steps against one eager warm-up + two replays of the captured step
    cov = w.psf_cov
    target = plan.render(_dev(build_workload(2, subdiv_override=2, grid_override=w.n).vertices), cov).clone()
    v_e = vd.clone()
    st = plan.shape_state(lr=1e-3)
    for _ in range(3):
        st.step(v_e, target, cov)
    st.close()
    v_g = vd.clone()
    st = plan.shape_state(lr=1e-3)
    st.step(v_g, target, cov)
    g2 = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g2):
        plan.set_stream()
        st.step(v_g, target, cov)
    plan.set_stream()
    g2.replay()                                            # (capturing records the step, it does not run it)
    g2.replay()
    torch.cuda.synchronize()
    assert torch.equal(v_g, v_e)
    st.close()
    plan.close()


def test_autograd_front_end(dm):
    """paper_2303_10440_b200.mesh_ft / render as torch.autograd functions: gradients through them equal the
    direct C-ABI calls bit for bit, for a loss on the complex spectrum (convention R14) and for an image loss w.r.t. both the
    vertices and the six PSF numbers."""
    import torch
    w = build_workload(1, grid_override=(16, 16, 16))
    plan = _plan(dm, w, 0)
    v = _dev(w.vertices).clone().requires_grad_(True)
    W = _dev(spectrum_cotangent(w))
    F = dm.mesh_ft(plan, v)
    loss = (F.real * W.real + F.imag * W.imag).sum()          # dL/dRe F + i dL/dIm F = W
    (gv,) = torch.autograd.grad(loss, v)
    assert torch.equal(gv, plan.mesh_ft_backward(v.detach(), W))
    cov = torch.tensor(w.psf_cov, dtype=torch.float32, requires_grad=True)
    target = torch.rand(w.n, device="cuda")
    img = dm.render(plan, v, cov)
    loss = ((img - target) ** 2).sum()
    gv, gc = torch.autograd.grad(loss, (v, cov))
    dv, dcov = plan.render_backward(v.detach(), w.psf_cov, (2 * (img.detach() - target)).contiguous(), with_psf_grad=True)
    assert torch.equal(gv, dv) and np.allclose(gc.numpy(), np.array(dcov, dtype=np.float32), rtol=0, atol=0)
    # vertices only: no PSF gradient is requested, so the call does not synchronise for it
    img = dm.render(plan, v, w.psf_cov)
    (gv2,) = torch.autograd.grad(((img - target) ** 2).sum(), v)
    assert torch.equal(gv2, dv)
    # a plan that changed between forward and backward is refused (the gradient would be the banded function's)
    img = dm.render(plan, v, w.psf_cov)
    plan.set_narrow_band(w.psf_cov, 0.01)
    with pytest.raises(RuntimeError, match="plan changed between forward and backward"):
        torch.autograd.grad(((img - target) ** 2).sum(), v)
    plan.set_narrow_band(None)
    # with DM_OPT_REUSE_SPECTRUM the backward reads the spectrum of the LAST render: one in between invalidates the graph
    plan.set_option(dm.DM_OPT_REUSE_SPECTRUM, 1)
    img = dm.render(plan, v, cov)
    (gv3, gc3) = torch.autograd.grad(((img - target) ** 2).sum(), (v, cov), retain_graph=True)
    assert torch.allclose(gv3, dv, rtol=1e-5, atol=1e-6 * float(dv.abs().max())) and np.allclose(gc3.numpy(), np.array(dcov, dtype=np.float32), rtol=1e-5)
    plan.render(_dev(w.vertices * 0.9), w.psf_cov)
    with pytest.raises(RuntimeError, match="plan changed between forward and backward"):
        torch.autograd.grad(((img - target) ** 2).sum(), (v, cov))
    plan.close()
