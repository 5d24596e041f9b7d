"""Triangle-mesh generators for the synthetic workloads (data only, numpy).

All meshes are returned as ``(vertices float64 [n_V,3], faces int32 [n_T,3])`` with faces
counter-clockwise seen from outside (outward normal), which is the documented precondition of volume
mode.  Callers quantise vertices to fp32 themselves (R21).
"""
from __future__ import annotations

import numpy as np


def _orient_outward(vertices: np.ndarray, faces: np.ndarray, centre: np.ndarray) -> np.ndarray:
    """Flip faces whose normal points toward ``centre`` (valid for star-shaped meshes)."""
    a = vertices[faces[:, 0]]
    b = vertices[faces[:, 1]]
    c = vertices[faces[:, 2]]
    n = np.cross(b - a, c - a)
    out = np.einsum("ij,ij->i", n, (a + b + c) / 3.0 - centre)
    flipped = faces.copy()
    bad = out < 0
    flipped[bad, 1], flipped[bad, 2] = faces[bad, 2], faces[bad, 1]
    return flipped


def icosphere(subdiv: int, radius: float = 1.0, centre=(0.0, 0.0, 0.0)):
    """Icosahedron subdivided ``subdiv`` times, midpoints normalised to the sphere (R18).

    n_V = 10*4**s + 2, n_T = 20*4**s  (s=2: 162/320, s=4: 2562/5120, s=7: 163842/327680).
    """
    t = (1.0 + 5.0 ** 0.5) / 2.0
    v = np.array(
        [[-1, t, 0], [1, t, 0], [-1, -t, 0], [1, -t, 0],
         [0, -1, t], [0, 1, t], [0, -1, -t], [0, 1, -t],
         [t, 0, -1], [t, 0, 1], [-t, 0, -1], [-t, 0, 1]], dtype=np.float64)
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    f = np.array(
        [[0, 11, 5], [0, 5, 1], [0, 1, 7], [0, 7, 10], [0, 10, 11],
         [1, 5, 9], [5, 11, 4], [11, 10, 2], [10, 7, 6], [7, 1, 8],
         [3, 9, 4], [3, 4, 2], [3, 2, 6], [3, 6, 8], [3, 8, 9],
         [4, 9, 5], [2, 4, 11], [6, 2, 10], [8, 6, 7], [9, 8, 1]], dtype=np.int64)
    for _ in range(subdiv):
        n_v = v.shape[0]
        # the three edges of every face, as sorted vertex pairs
        e = np.concatenate([f[:, [0, 1]], f[:, [1, 2]], f[:, [2, 0]]], axis=0)
        e.sort(axis=1)
        key = e[:, 0] * n_v + e[:, 1]
        uniq, inv = np.unique(key, return_inverse=True)
        mid = v[uniq // n_v] + v[uniq % n_v]
        mid /= np.linalg.norm(mid, axis=1, keepdims=True)
        v = np.concatenate([v, mid], axis=0)
        n_f = f.shape[0]
        m01 = n_v + inv[:n_f]
        m12 = n_v + inv[n_f:2 * n_f]
        m20 = n_v + inv[2 * n_f:]
        f = np.concatenate([
            np.stack([f[:, 0], m01, m20], axis=1),
            np.stack([f[:, 1], m12, m01], axis=1),
            np.stack([f[:, 2], m20, m12], axis=1),
            np.stack([m01, m12, m20], axis=1)], axis=0)
    f = _orient_outward(v, f, np.zeros(3))
    v = v * radius + np.asarray(centre, dtype=np.float64)
    return v, f.astype(np.int32)


def box_mesh(centre, half_widths):
    """Axis-aligned box as 12 outward-oriented triangles (pin P1)."""
    c = np.asarray(centre, dtype=np.float64)
    h = np.asarray(half_widths, dtype=np.float64)
    s = np.array([[-1, -1, -1], [1, -1, -1], [1, 1, -1], [-1, 1, -1],
                  [-1, -1, 1], [1, -1, 1], [1, 1, 1], [-1, 1, 1]], dtype=np.float64)
    v = c + s * h
    quads = [[0, 3, 2, 1], [4, 5, 6, 7], [0, 1, 5, 4], [2, 3, 7, 6], [1, 2, 6, 5], [0, 4, 7, 3]]
    f = []
    for q in quads:
        f.append([q[0], q[1], q[2]])
        f.append([q[0], q[2], q[3]])
    f = _orient_outward(v, np.array(f, dtype=np.int64), c)
    return v, f.astype(np.int32)


def tetrahedron_mesh(vertices):
    """Closed tetrahedron on four given points, outward oriented."""
    v = np.asarray(vertices, dtype=np.float64).reshape(4, 3)
    f = np.array([[0, 1, 2], [0, 1, 3], [0, 2, 3], [1, 2, 3]], dtype=np.int64)
    f = _orient_outward(v, f, v.mean(axis=0))
    return v, f.astype(np.int32)


def perturb_radial(vertices, centre, sigma, rng: np.random.Generator):
    """r <- r * (1 + sigma * N(0,1)) about ``centre``; normals drawn in vertex order (R17)."""
    c = np.asarray(centre, dtype=np.float64)
    z = rng.standard_normal(vertices.shape[0])
    return c + (vertices - c) * (1.0 + sigma * z)[:, None]


def vertex_one_ring(n_vertices: int, faces: np.ndarray):
    """CSR adjacency (offsets, neighbours) of the vertex graph, duplicates removed."""
    f = faces.astype(np.int64)
    e = np.concatenate([f[:, [0, 1]], f[:, [1, 2]], f[:, [2, 0]],
                        f[:, [1, 0]], f[:, [2, 1]], f[:, [0, 2]]], axis=0)
    key = np.unique(e[:, 0] * n_vertices + e[:, 1])
    src = key // n_vertices
    dst = key % n_vertices
    offsets = np.zeros(n_vertices + 1, dtype=np.int64)
    np.add.at(offsets, src + 1, 1)
    offsets = np.cumsum(offsets)
    return offsets, dst


def laplacian_smooth(vertices, faces, steps: int = 1, lam: float = 0.5):
    """Uniform umbrella smoothing v <- v + lam*(mean of 1-ring - v), simultaneous update (R17)."""
    v = np.array(vertices, dtype=np.float64)
    offsets, nbr = vertex_one_ring(v.shape[0], faces)
    deg = np.diff(offsets).astype(np.float64)
    for _ in range(steps):
        acc = np.zeros_like(v)
        np.add.at(acc, np.repeat(np.arange(v.shape[0]), np.diff(offsets)), v[nbr])
        mean = acc / deg[:, None]
        v = v + lam * (mean - v)
    return v


def pack_spheres(n, r_lo, r_hi, half_extent, rng: np.random.Generator, margin: float = 1.25):
    """Centres uniform in [-half_extent, half_extent]^3 with |c_i-c_j| > margin*(r_i+r_j) (R17).

    Rejection sampling; restarts from scratch if it jams.  Returns (centres [n,3], radii [n]).
    """
    while True:
        centres, radii = [], []
        tries = 0
        while len(centres) < n and tries < 20000:
            tries += 1
            c = rng.uniform(-half_extent, half_extent, size=3)
            r = rng.uniform(r_lo, r_hi)
            ok = all(np.linalg.norm(c - cj) > margin * (r + rj) for cj, rj in zip(centres, radii))
            if ok:
                centres.append(c)
                radii.append(r)
        if len(centres) == n:
            return np.array(centres), np.array(radii)
