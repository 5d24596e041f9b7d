"""ctypes front end of the C oracle + the frequency-grid convention (reading R10).

TEST INFRASTRUCTURE (see oracle/__init__.py).  Host numpy arrays in, numpy arrays out, fp64.
"""
from __future__ import annotations

import ctypes

import numpy as np

from . import build as _build

_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(_build.build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int32)
        lib.oracle_g.argtypes = [ctypes.c_double] * 3 + [dp]
        lib.oracle_g.restype = None
        lib.oracle_g_grad.argtypes = [ctypes.c_double] * 3 + [dp]
        lib.oracle_g_grad.restype = None
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_mesh_ft_forward.argtypes = [dp, ctypes.c_int32, ip, ctypes.c_int32, dp, ctypes.c_int64,
                                               ctypes.c_int32, dp]
        lib.oracle_mesh_ft_forward.restype = ctypes.c_int
        lib.oracle_mesh_ft_backward.argtypes = [dp, ctypes.c_int32, ip, ctypes.c_int32, dp, ctypes.c_int64,
                                                ctypes.c_int32, dp, dp, dp]
        lib.oracle_mesh_ft_backward.restype = ctypes.c_int
        _lib = lib
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _ip(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def g_fun(a: float, b: float, c: float) -> complex:
    """f_T = g(a,b,c) = exp[-ia,-ib,-ic]  (eq. 9 / :194 eq. 14, made exact)."""
    out = np.zeros(2)
    _load().oracle_g(float(a), float(b), float(c), _dp(out))
    return complex(out[0], out[1])


def g_grad(a: float, b: float, c: float) -> np.ndarray:
    """(dg/da, dg/db, dg/dc) as complex128 [3]."""
    out = np.zeros(6)
    _load().oracle_g_grad(float(a), float(b), float(c), _dp(out))
    return out[0::2] + 1j * out[1::2]


def frequency_grid(n, spacing) -> np.ndarray:
    """Angular frequencies of the stored half spectrum, float64 [N_x, N_y, N_z/2+1, 3].

    Reading R10: array order [x][y][z], z fastest and halved; n_x, n_y in numpy fftfreq order
    (0..N/2-1, -N/2..-1), n_z = 0..N_z/2; k_a = 2 pi n_a / L_a with L_a = N_a h_a (PAPER.md:131
    uses the angular convention exp(-i z.xi)).
    """
    nx, ny, nz = (int(v) for v in n)
    hx, hy, hz = (float(v) for v in spacing)
    kx = 2.0 * np.pi * np.fft.fftfreq(nx, d=hx)
    ky = 2.0 * np.pi * np.fft.fftfreq(ny, d=hy)
    kz = 2.0 * np.pi * np.fft.rfftfreq(nz, d=hz)
    k = np.empty((nx, ny, nz // 2 + 1, 3), dtype=np.float64)
    k[..., 0] = kx[:, None, None]
    k[..., 1] = ky[None, :, None]
    k[..., 2] = kz[None, None, :]
    return k


def _prep(vertices, faces):
    v = np.ascontiguousarray(np.asarray(vertices, dtype=np.float64).reshape(-1, 3))  # O1: promote fp32 inputs
    f = np.ascontiguousarray(np.asarray(faces, dtype=np.int32).reshape(-1, 3))
    return v, f


def mesh_ft_forward(vertices, faces, kvec, mode: int) -> np.ndarray:
    """F(k) at an explicit list of angular frequencies kvec [n_k,3] -> complex128 [n_k]."""
    v, f = _prep(vertices, faces)
    k = np.ascontiguousarray(np.asarray(kvec, dtype=np.float64).reshape(-1, 3))
    out = np.zeros(2 * k.shape[0], dtype=np.float64)
    rc = _load().oracle_mesh_ft_forward(_dp(v), v.shape[0], _ip(f), f.shape[0], _dp(k), k.shape[0], int(mode), _dp(out))
    if rc != 0:
        raise ValueError(f"oracle_mesh_ft_forward failed with code {rc}")
    return out[0::2] + 1j * out[1::2]


def mesh_ft_forward_grid(vertices, faces, n, spacing, mode: int, flat_indices=None) -> np.ndarray:
    """F on the stored half-spectrum grid [N_x,N_y,N_z/2+1], or at ``flat_indices`` of it."""
    kg = frequency_grid(n, spacing).reshape(-1, 3)
    if flat_indices is not None:
        return mesh_ft_forward(vertices, faces, kg[np.asarray(flat_indices)], mode)
    return mesh_ft_forward(vertices, faces, kg, mode).reshape(int(n[0]), int(n[1]), int(n[2]) // 2 + 1)


def mesh_ft_backward(vertices, faces, kvec, mode: int, G, return_corners: bool = False):
    """dL/dv [n_V,3] = sum over the listed k of Re(conj(G) dF/dv); G complex [n_k]."""
    v, f = _prep(vertices, faces)
    k = np.ascontiguousarray(np.asarray(kvec, dtype=np.float64).reshape(-1, 3))
    Gc = np.asarray(G, dtype=np.complex128).reshape(-1)
    if Gc.shape[0] != k.shape[0]:
        raise ValueError("G and kvec disagree in length")
    Gi = np.empty(2 * k.shape[0], dtype=np.float64)
    Gi[0::2] = Gc.real
    Gi[1::2] = Gc.imag
    out = np.zeros((v.shape[0], 3), dtype=np.float64)
    corners = np.zeros((f.shape[0], 3, 3), dtype=np.float64)
    rc = _load().oracle_mesh_ft_backward(_dp(v), v.shape[0], _ip(f), f.shape[0], _dp(k), k.shape[0], int(mode),
                                         _dp(Gi), _dp(out), _dp(corners))
    if rc != 0:
        raise ValueError(f"oracle_mesh_ft_backward failed with code {rc}")
    return (out, corners) if return_corners else out


def mesh_ft_backward_grid(vertices, faces, n, spacing, mode: int, G, flat_indices=None) -> np.ndarray:
    """Backward over the whole stored grid (G [N_x,N_y,N_z/2+1]) or over ``flat_indices`` only
    (G then holds one value per listed index)."""
    kg = frequency_grid(n, spacing).reshape(-1, 3)
    if flat_indices is not None:
        return mesh_ft_backward(vertices, faces, kg[np.asarray(flat_indices)], mode, G)
    return mesh_ft_backward(vertices, faces, kg, mode, np.asarray(G).reshape(-1))


# ---- area-normalised membrane density (eq. 12-13; NEXT 3) ------------------------------------------------
def surface_area_and_gradient(vertices, faces):
    """|Lambda| = sum_T A_T and d|Lambda|/dv [n_V,3] = sum over the vertex star of dA_T/dv_p = -w_p/2, w_p = e_p x N_T,
    e_p = v_{p-} - v_{p+}.  Degenerate triangles contribute 0 (reading R19)."""
    v, f = _prep(vertices, faces)
    area, grad = 0.0, np.zeros_like(v)
    for tri in f:
        p = v[tri]
        m = np.cross(p[1] - p[0], p[2] - p[0])
        mn = float(np.linalg.norm(m))
        area += 0.5 * mn
        if mn < 1e-30:
            continue
        N = m / mn
        for c in range(3):
            e = p[(c + 2) % 3] - p[(c + 1) % 3]
            grad[tri[c]] += -0.5 * np.cross(e, N)
    return area, grad


def mesh_ft_forward_normalised(vertices, faces, kvec) -> np.ndarray:
    """eq. 12: u_Lambda(k) = (1/|Lambda|) sum_T 2 A_T f_T(k) -- the surface-mode FT divided by the total area."""
    area, _ = surface_area_and_gradient(vertices, faces)
    return mesh_ft_forward(vertices, faces, kvec, 1) / area


def mesh_ft_backward_normalised(vertices, faces, kvec, G) -> np.ndarray:
    """eq. 13: the gradient of eq. 12 by the quotient rule,
        dL/dv = (1/|Lambda|) sum_k Re(conj(G) dF/dv) - ( sum_k Re(conj(G) u_Lambda(k)) / |Lambda| ) d|Lambda|/dv ,
    F the un-normalised surface-mode FT."""
    area, darea = surface_area_and_gradient(vertices, faces)
    Gc = np.asarray(G, dtype=np.complex128).reshape(-1)
    bare = mesh_ft_backward(vertices, faces, kvec, 1, Gc)
    u = mesh_ft_forward(vertices, faces, kvec, 1) / area
    s = float((np.conj(Gc) * u).real.sum())
    return bare / area - (s / area) * darea


# ---- per-face density weights ("a weighted sum of the FT of surfaces with different densities") -------------
def _weight_groups(faces, weights):
    f = np.asarray(faces, dtype=np.int32).reshape(-1, 3)
    w = np.asarray(weights, dtype=np.float64).reshape(-1)
    if w.shape[0] != f.shape[0]:
        raise ValueError("one weight per face")
    return [(float(u), f[w == u]) for u in np.unique(w)]


def mesh_ft_forward_weighted(vertices, faces, kvec, mode: int, weights) -> np.ndarray:
    """F(k) = sum_T w_T (triangle term of T): by linearity, the sum over the groups of equal weight of w times the FT of
    the group's faces.  Meant for a few distinct weights (one per surface), as in the paper."""
    k = np.asarray(kvec, dtype=np.float64).reshape(-1, 3)
    out = np.zeros(k.shape[0], dtype=np.complex128)
    for u, fg in _weight_groups(faces, weights):
        out += u * mesh_ft_forward(vertices, fg, k, mode)
    return out


def mesh_ft_backward_weighted(vertices, faces, kvec, mode: int, G, weights) -> np.ndarray:
    """dL/dv of mesh_ft_forward_weighted, by the same linearity over the groups of equal weight.  Pinned by central
    finite differences of the weighted forward, the translation identity and a per-corner assembly that never groups
    faces (tests/test_oracle_backward.py::test_weighted_backward_*)."""
    v = np.asarray(vertices, dtype=np.float64).reshape(-1, 3)
    out = np.zeros_like(v)
    for u, fg in _weight_groups(faces, weights):
        out += u * mesh_ft_backward(vertices, fg, kvec, mode, G)
    return out
