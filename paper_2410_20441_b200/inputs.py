"""Seeded synthetic voxel images (K, G fields) for the BASELINE.json configs.

This module holds NO arithmetic of the method (no stencil, no PT constants, no averaging):
it only paints moduli into (nz, ny, nx) float64 arrays, x fastest.  It is the one module
shared by the oracle tests and the CUDA path (both receive the *same arrays*).

The paper's only real data set (cracked Carrara marble) is not available; these
images stand in for its shapes, sizes and contrasts.  Voxel (i,j,k) has centre (i+.5,j+.5,k+.5);
"inside" tests use <=.  numpy default_rng(seed) is PCG64.
"""
from __future__ import annotations

import numpy as np

CALCITE = (70.2, 29.0)          # K, G in GPa (BASELINE.json configs 1, 2, 5)
QUARTZ_LIKE = (37.0, 44.0)      # configs 3, 4


def _two_phase(mask, matrix, incl):
    K = np.where(mask, incl[0], matrix[0]).astype(np.float64)
    G = np.where(mask, incl[1], matrix[1]).astype(np.float64)
    return np.ascontiguousarray(K), np.ascontiguousarray(G)


def _centres(n):
    return np.arange(n, dtype=np.float64) + 0.5


def homogeneous(n, K=CALCITE[0], G=CALCITE[1]):
    shape = (n, n, n) if np.isscalar(n) else tuple(n)[::-1]
    return np.full(shape, float(K)), np.full(shape, float(G))


def sphere_mask(n, centre, r):
    z, y, x = np.meshgrid(_centres(n), _centres(n), _centres(n), indexing="ij", sparse=True)
    return (x - centre[0]) ** 2 + (y - centre[1]) ** 2 + (z - centre[2]) ** 2 <= r * r


def config1_sphere(n=32, r=5.0, matrix=CALCITE, contrast=1e-6):
    """cfg 1: one centred spherical pore of radius r voxels, pore moduli = contrast x matrix."""
    m = sphere_mask(n, (n / 2.0,) * 3, r)
    return _two_phase(m, matrix, (matrix[0] * contrast, matrix[1] * contrast)) + (m,)


def config2_spheroid(n=191, semi=(40.0, 40.0, 8.0), matrix=CALCITE, incl=(2.2, 0.0)):
    """cfg 2: one centred oblate spheroid (fluid-like K=2.2, G=0)."""
    c = n / 2.0
    z, y, x = np.meshgrid(_centres(n), _centres(n), _centres(n), indexing="ij", sparse=True)
    m = ((x - c) / semi[0]) ** 2 + ((y - c) / semi[1]) ** 2 + ((z - c) / semi[2]) ** 2 <= 1.0
    return _two_phase(m, matrix, incl) + (m,)


def _paint_sphere(mask, c, r):
    nz, ny, nx = mask.shape
    lo = [max(int(np.floor(c[a] - r - 1)), 0) for a in range(3)]
    hi = [min(int(np.ceil(c[a] + r + 1)), (nx, ny, nz)[a]) for a in range(3)]
    if any(lo[a] >= hi[a] for a in range(3)):
        return
    x = np.arange(lo[0], hi[0]) + 0.5
    y = np.arange(lo[1], hi[1]) + 0.5
    z = np.arange(lo[2], hi[2]) + 0.5
    d2 = (x[None, None, :] - c[0]) ** 2 + (y[None, :, None] - c[1]) ** 2 + (z[:, None, None] - c[2]) ** 2
    mask[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]] |= d2 <= r * r


def config3_random_spheres(n=191, npores=200, rmin=3.0, rmax=10.0, seed=20241020,
                           matrix=QUARTZ_LIKE, contrast=1e-6):
    """cfg 3: union of npores spheres, centre = rng.uniform(0,n,3) then r = rng.uniform(rmin,rmax), clipped
    at the walls.  (This explicit recipe gives porosity ~4.4 % at n=191, not the ~10 % BASELINE mentions.)"""
    rng = np.random.default_rng(seed)
    m = np.zeros((n, n, n), dtype=bool)
    for _ in range(npores):
        c = rng.uniform(0, n, 3)
        r = rng.uniform(rmin, rmax)
        _paint_sphere(m, c, r)
    return _two_phase(m, matrix, (matrix[0] * contrast, matrix[1] * contrast)) + (m,)


def config4_grf(n=479, ell=12.0, soft_fraction=0.15, seed=20241021, matrix=QUARTZ_LIKE, soft=(5.0, 2.0)):
    """cfg 4: thresholded periodic Gaussian random field, covariance ~ exp(-r^2/ell^2); soft where the
    field is below its soft_fraction quantile."""
    rng = np.random.default_rng(seed)
    w = rng.standard_normal((n, n, n))
    kz = 2 * np.pi * np.fft.fftfreq(n)[:, None, None]
    ky = 2 * np.pi * np.fft.fftfreq(n)[None, :, None]
    kx = 2 * np.pi * np.fft.rfftfreq(n)[None, None, :]
    F = np.fft.rfftn(w)
    del w
    F *= np.exp(-(kx * kx + ky * ky + kz * kz) * (ell * ell / 8.0))
    f = np.fft.irfftn(F, s=(n, n, n), axes=(0, 1, 2))
    del F
    thr = np.quantile(f, soft_fraction)
    m = f < thr
    return _two_phase(m, matrix, soft) + (m,)


def config5_penny_cracks(n=703, ncracks=400, rmin=20.0, rmax=60.0, half_aperture=1.0, kappa=4.0,
                         seed=20241022, matrix=CALCITE, contrast=1e-6):
    """cfg 5: union of oblate spheroids (penny cracks), normals from von Mises-Fisher(kappa) about +z."""
    rng = np.random.default_rng(seed)
    m = np.zeros((n, n, n), dtype=bool)
    for _ in range(ncracks):
        c = rng.uniform(0, n, 3)
        r = rng.uniform(rmin, rmax)
        u = rng.uniform()
        wz = 1.0 + np.log(u + (1.0 - u) * np.exp(-2.0 * kappa)) / kappa
        az = rng.uniform(0, 2 * np.pi)
        s = np.sqrt(max(0.0, 1.0 - wz * wz))
        nvec = np.array([s * np.cos(az), s * np.sin(az), wz])
        lo = [max(int(np.floor(c[a] - r - 1)), 0) for a in range(3)]
        hi = [min(int(np.ceil(c[a] + r + 1)), n) for a in range(3)]
        if any(lo[a] >= hi[a] for a in range(3)):
            continue
        x = (np.arange(lo[0], hi[0]) + 0.5 - c[0])[None, None, :]
        y = (np.arange(lo[1], hi[1]) + 0.5 - c[1])[None, :, None]
        z = (np.arange(lo[2], hi[2]) + 0.5 - c[2])[:, None, None]
        dn = x * nvec[0] + y * nvec[1] + z * nvec[2]
        dt2 = x * x + y * y + z * z - dn * dn
        m[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]] |= dt2 / (r * r) + dn * dn / (half_aperture ** 2) <= 1.0
    return _two_phase(m, matrix, (matrix[0] * contrast, matrix[1] * contrast)) + (m,)


def layered(nx, ny, nz, thickness=15, soft=(7.2, 8.8), stiff=(36.0, 44.0)):
    """Model 1 of the paper: layers normal to z, `thickness` cells each, soft first."""
    k = np.arange(nz)
    is_stiff = (k // thickness) % 2 == 1
    K = np.where(is_stiff, stiff[0], soft[0])[:, None, None] * np.ones((nz, ny, nx))
    G = np.where(is_stiff, stiff[1], soft[1])[:, None, None] * np.ones((nz, ny, nx))
    return np.ascontiguousarray(K), np.ascontiguousarray(G), is_stiff


def random_two_phase(n, frac=0.3, seed=0, matrix=QUARTZ_LIKE, incl=(5.0, 2.0)):
    """voxel-noise two-phase medium (small test images, any shape n or (nx,ny,nz))."""
    shape = (n, n, n) if np.isscalar(n) else tuple(n)[::-1]
    rng = np.random.default_rng(seed)
    m = rng.uniform(size=shape) < frac
    return _two_phase(m, matrix, incl) + (m,)


def random_smooth(n, seed=0, Krange=(5.0, 70.0), Grange=(2.0, 45.0)):
    """fully heterogeneous moduli (every voxel different), for parity tests."""
    shape = (n, n, n) if np.isscalar(n) else tuple(n)[::-1]
    rng = np.random.default_rng(seed)
    K = rng.uniform(Krange[0], Krange[1], size=shape)
    G = rng.uniform(Grange[0], Grange[1], size=shape)
    return K, G
