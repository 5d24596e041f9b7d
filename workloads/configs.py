"""BASELINE.json's five configurations as seeded synthetic workloads.

The paper measures on an 80-triangle sphere, meshes of growing size in a 100^3 box and
a 4000-vertex embryo mesh in a 205x285x134 confocal stack; none of those inputs
exist here, so these icosphere workloads stand in for them (roundish closed cells, edge length of
1-3 voxels, blur of 1-3 voxels, anisotropic z).  Data only: nothing here evaluates the method.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from .meshes import icosphere, laplacian_smooth, pack_spheres, perturb_radial

VOLUME, SURFACE = 0, 1


@dataclass
class Workload:
    name: str
    cfg: int
    mode: int                      # 0 = volume, 1 = surface
    vertices: np.ndarray           # float32 [n_V,3]  (the input of record, R21)
    faces: np.ndarray              # int32 [n_T,3], CCW seen from outside
    n: tuple                       # voxels (N_x, N_y, N_z); rfft half axis = z
    spacing: tuple                 # voxel size per axis, box length L_a = n[a]*spacing[a]
    origin: tuple                  # sample point of voxel (0,0,0) = -L/2 + h/2 (R9, R11)
    sigma_vox: tuple               # Gaussian PSF sigma in voxels of each axis (R12)
    seed: int
    meta: dict = field(default_factory=dict)

    @property
    def n_k(self) -> int:
        return self.n[0] * self.n[1] * (self.n[2] // 2 + 1)

    @property
    def pairs(self) -> int:
        return self.faces.shape[0] * self.n_k

    @property
    def spectrum_shape(self) -> tuple:
        return (self.n[0], self.n[1], self.n[2] // 2 + 1)

    @property
    def psf_cov(self) -> np.ndarray:
        """Covariance in physical units, order xx,yy,zz,xy,xz,yz (sigma_phys = sigma_vox*h, R12)."""
        s = np.asarray(self.sigma_vox, dtype=np.float64) * np.asarray(self.spacing, dtype=np.float64)
        return np.array([s[0] ** 2, s[1] ** 2, s[2] ** 2, 0.0, 0.0, 0.0], dtype=np.float32)


def _grid(n):
    n = tuple(int(x) for x in n)
    spacing = tuple(1.0 / x for x in n)                      # box [-0.5,0.5]^3, L = (1,1,1)
    origin = tuple(-0.5 + 0.5 * h for h in spacing)
    return n, spacing, origin


def _perturbed_sphere(subdiv, radius, centre, sigma, smooth_steps, rng):
    v, f = icosphere(subdiv, radius, centre)
    v = perturb_radial(v, centre, sigma, rng)
    v = laplacian_smooth(v, f, steps=smooth_steps)
    return v, f


def _aggregate(n_cells, subdiv, r_lo, r_hi, half_extent, sigma, rng):
    centres, radii = pack_spheres(n_cells, r_lo, r_hi, half_extent, rng)
    vs, fs, off = [], [], 0
    for c, r in zip(centres, radii):
        v, f = _perturbed_sphere(subdiv, r, c, sigma, 1, rng)
        vs.append(v)
        fs.append(f + off)
        off += v.shape[0]
    return np.concatenate(vs), np.concatenate(fs).astype(np.int32), centres, radii


def _mesh_for(cfg: int, seed: int, subdiv_override=None):
    rng = np.random.default_rng(seed)
    meta = {}
    if cfg == 1:
        v, f = icosphere(2 if subdiv_override is None else subdiv_override, 0.3)
    elif cfg == 2:
        v, f = _perturbed_sphere(4 if subdiv_override is None else subdiv_override, 0.35,
                                 np.zeros(3), 0.05, 1, rng)
    elif cfg == 3:
        v, f, c, r = _aggregate(8, 4 if subdiv_override is None else subdiv_override,
                                0.12, 0.18, 0.3, 0.05, rng)
        meta = {"centres": c, "radii": r}
    elif cfg == 4:
        v, f, c, r = _aggregate(20, 4 if subdiv_override is None else subdiv_override,
                                0.06, 0.12, 0.4, 0.05, rng)
        meta = {"centres": c, "radii": r}
    elif cfg == 5:
        v, f = _perturbed_sphere(7 if subdiv_override is None else subdiv_override, 0.4,
                                 np.zeros(3), 0.03, 2, rng)
    else:
        raise ValueError(f"unknown config {cfg}")
    return v.astype(np.float32), f.astype(np.int32), meta


_SPEC = {
    1: dict(name="cfg1_icosphere2_32", mode=VOLUME, n=(32, 32, 32), sigma=(1.0, 1.0, 2.0), seed=0),
    2: dict(name="cfg2_icosphere4_64", mode=VOLUME, n=(64, 64, 64), sigma=(1.5, 1.5, 3.0), seed=1),
    3: dict(name="cfg3_aggregate8_128x128x64", mode=VOLUME, n=(128, 128, 64), sigma=(1.2, 1.2, 2.5), seed=2),
    4: dict(name="cfg4_membranes20_128", mode=SURFACE, n=(128, 128, 128), sigma=(1.0, 1.0, 2.5), seed=3),
    5: dict(name="cfg5_icosphere7_256", mode=VOLUME, n=(256, 256, 256), sigma=(1.0, 1.0, 2.0), seed=4),
}
CONFIGS = tuple(sorted(_SPEC))


def build_workload(cfg: int, seed_offset: int = 0, subdiv_override=None, grid_override=None) -> Workload:
    """Workload ``cfg`` (1..5).  ``seed_offset=100`` gives the target mesh of cfg 2 / 4 (R16).

    ``subdiv_override`` / ``grid_override`` shrink a config for quick tests without changing its recipe.
    """
    s = _SPEC[cfg]
    seed = s["seed"] + seed_offset
    v, f, meta = _mesh_for(cfg, seed, subdiv_override)
    n, spacing, origin = _grid(s["n"] if grid_override is None else grid_override)
    return Workload(name=s["name"], cfg=cfg, mode=s["mode"], vertices=v, faces=f, n=n, spacing=spacing,
                    origin=origin, sigma_vox=s["sigma"], seed=seed, meta=meta)


def image_cotangent(w: Workload) -> np.ndarray:
    """dL/dimage ~ N(0,1), float32 [N_x,N_y,N_z]; seed 0 for cfg 1, 10+seed for cfg 3 and 5 (R16)."""
    seed = 0 if w.cfg == 1 else 10 + w.seed
    return np.random.default_rng(seed).standard_normal(w.n).astype(np.float32)


def spectrum_cotangent(w: Workload, seed: int = 7) -> np.ndarray:
    """Random complex dL/dF on the stored half spectrum, complex64 [N_x,N_y,N_z/2+1]."""
    rng = np.random.default_rng(seed + 31 * w.cfg)
    g = rng.standard_normal(w.spectrum_shape) + 1j * rng.standard_normal(w.spectrum_shape)
    return g.astype(np.complex64)


def sampled_frequencies(w: Workload, n_random: int = 4096, n_nyquist: int = 64) -> np.ndarray:
    """The sampled set S of stored-frequency flat indices used for parity at large configs.

    S = all |n_a| <= 4  U  ``n_nyquist`` random entries on each Nyquist plane  U  the three axes
        U  ``n_random`` uniform random entries (seed 1000+cfg).
    Flat index = (ix*N_y + iy)*(N_z/2+1) + iz with ix, iy in numpy fftfreq order.
    """
    nx, ny, nz = w.n
    nzh = nz // 2 + 1
    rng = np.random.default_rng(1000 + w.cfg)
    idx = []

    def flat(ix, iy, iz):
        return (np.asarray(ix) % nx * ny + np.asarray(iy) % ny) * nzh + np.asarray(iz)

    lo = [min(4, nx // 2 - 1), min(4, ny // 2 - 1), min(4, nzh - 1)]
    gx, gy, gz = np.meshgrid(np.arange(-lo[0], lo[0] + 1), np.arange(-lo[1], lo[1] + 1),
                             np.arange(0, lo[2] + 1), indexing="ij")
    idx.append(flat(gx.ravel(), gy.ravel(), gz.ravel()))
    # Nyquist planes: ix = N_x/2, iy = N_y/2, iz = N_z/2
    idx.append(flat(np.full(n_nyquist, nx // 2), rng.integers(0, ny, n_nyquist), rng.integers(0, nzh, n_nyquist)))
    idx.append(flat(rng.integers(0, nx, n_nyquist), np.full(n_nyquist, ny // 2), rng.integers(0, nzh, n_nyquist)))
    idx.append(flat(rng.integers(0, nx, n_nyquist), rng.integers(0, ny, n_nyquist), np.full(n_nyquist, nzh - 1)))
    # the three axes
    idx.append(flat(np.arange(nx), np.zeros(nx, int), np.zeros(nx, int)))
    idx.append(flat(np.zeros(ny, int), np.arange(ny), np.zeros(ny, int)))
    idx.append(flat(np.zeros(nzh, int), np.zeros(nzh, int), np.arange(nzh)))
    idx.append(rng.integers(0, nx * ny * nzh, n_random))
    return np.unique(np.concatenate(idx)).astype(np.int64)
