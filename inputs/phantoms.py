"""Seeded synthetic CT phantoms for BASELINE.json configs C1, C3, C4, C5.

They stand in for the paper's homogeneous phantoms and patient
CTs (L166), none of which are in the container.  HU grids are int16 with x
fastest, then y, then z (array shape (nz, ny, nx)); voxel sizes in cm.
"""
from __future__ import annotations

import numpy as np


def phantom_c1():
    """50x50x100, 2 mm voxels, HU = 0 (water)."""
    return np.zeros((100, 50, 50), dtype=np.int16), (0.2, 0.2, 0.2)


def phantom_c3(nx=200, ny=200, nz=300, d=0.1):
    """Slab phantom: water 5 cm | bone HU 1200 2 cm | lung HU -700 5 cm | water; Ti block 1 cm^3 at centre."""
    hu = np.zeros((nz, ny, nx), dtype=np.int16)
    z = (np.arange(nz) + 0.5) * d
    hu[(z >= 5.0) & (z < 7.0)] = 1200
    hu[(z >= 7.0) & (z < 12.0)] = -700
    x = (np.arange(nx) + 0.5) * d
    y = (np.arange(ny) + 0.5) * d
    cx, cy = 0.5 * nx * d, 0.5 * ny * d
    mz = (z >= 14.5) & (z < 15.5)
    my = (y >= cy - 0.5) & (y < cy + 0.5)
    mx = (x >= cx - 0.5) & (x < cx + 0.5)
    hu[np.ix_(mz, my, mx)] = 3071
    return hu, (d, d, d)


def _ellipsoid_mask(shape, vox, centre, radii):
    nz, ny, nx = shape
    x = ((np.arange(nx) + 0.5) * vox[0] - centre[0]) / radii[0]
    y = ((np.arange(ny) + 0.5) * vox[1] - centre[1]) / radii[1]
    z = ((np.arange(nz) + 0.5) * vox[2] - centre[2]) / radii[2]
    return (z * z)[:, None, None] + (y * y)[None, :, None] + (x * x)[None, None, :] <= 1.0


def phantom_c4(seed=4, nx=256, ny=256, nz=120, vox=(0.1, 0.1, 0.25)):
    """Synthetic head-and-neck: returns (hu, vox, targets) with targets = list of (centre, radii) in cm."""
    rng = np.random.default_rng(seed)
    shape = (nz, ny, nx)
    hu = np.full(shape, -1000, dtype=np.int16)
    lx, ly, lz = nx * vox[0], ny * vox[1], nz * vox[2]
    cx, cy = 0.5 * lx, 0.5 * ly
    soft = np.clip(rng.normal(40.0, 20.0, size=shape), -100, 120).astype(np.int16)
    head_c, head_r = (cx, cy, 0.68 * lz), (8.0, 9.5, 0.30 * lz)
    neck_c, neck_r = (cx, cy + 0.5, 0.22 * lz), (5.5, 6.0, 0.30 * lz)
    # shoulders (low slices): wide enough that a lateral field to the low-neck target needs ~20 cm WET (~190 MeV)
    sh_c, sh_r = (cx, cy + 0.5, 0.0), (12.4, 7.0, 0.22 * lz)
    body = (_ellipsoid_mask(shape, vox, head_c, head_r) | _ellipsoid_mask(shape, vox, neck_c, neck_r)
            | _ellipsoid_mask(shape, vox, sh_c, sh_r))
    hu[body] = soft[body]
    for sgn in (-1.0, 1.0):     # humeral heads
        m = _ellipsoid_mask(shape, vox, (cx + sgn * 9.0, cy + 0.5, 0.05 * lz), (2.2, 2.2, 0.12 * lz))
        hu[m] = rng.integers(700, 1501, size=int(m.sum())).astype(np.int16)
    # skull shell
    inner = _ellipsoid_mask(shape, vox, head_c, tuple(r - 0.7 for r in head_r))
    outer = _ellipsoid_mask(shape, vox, head_c, tuple(r - 0.2 for r in head_r))
    shell = outer & ~inner
    hu[shell] = rng.integers(700, 1501, size=int(shell.sum())).astype(np.int16)
    # vertebral column (posterior = +y)
    col = _ellipsoid_mask(shape, vox, (cx, cy + 3.0, 0.30 * lz), (1.3, 1.3, 0.42 * lz))
    hu[col] = rng.integers(700, 1501, size=int(col.sum())).astype(np.int16)
    # airway + sinuses
    for c, r in [((cx, cy - 1.0, 0.25 * lz), (0.9, 0.9, 0.30 * lz)),
                 ((cx - 2.0, cy - 5.0, 0.62 * lz), (1.4, 1.6, 2.0)),
                 ((cx + 2.0, cy - 5.0, 0.62 * lz), (1.4, 1.6, 2.0)),
                 ((cx, cy - 6.0, 0.75 * lz), (1.2, 1.0, 1.5))]:
        hu[_ellipsoid_mask(shape, vox, c, r)] = -1000
    # dental arc
    for k in range(14):
        ang = np.pi * (0.15 + 0.7 * k / 13.0)
        c = (cx + 3.2 * np.cos(ang), cy - 3.5 - 3.0 * np.sin(ang), 0.47 * lz)
        m = _ellipsoid_mask(shape, vox, c, (0.35, 0.35, 0.6))
        hu[m] = rng.integers(2000, 3001, size=int(m.sum())).astype(np.int16)
    targets = [((cx - 2.5, cy + 0.5, 0.40 * lz), (1.4, 1.5, 1.9)),
               ((cx + 3.0, cy - 1.0, 0.30 * lz), (1.0, 1.0, 1.4)),
               ((cx + 4.5, cy + 0.5, 0.09 * lz), (1.2, 1.2, 1.3))]      # low-neck node behind the shoulder
    return hu, vox, targets


def phantom_c5(seed=5, nx=512, ny=512, nz=200, vox=(0.1, 0.1, 0.2)):
    """Synthetic pelvis with bilateral Ti hip implants: returns (hu, vox, targets)."""
    rng = np.random.default_rng(seed)
    shape = (nz, ny, nx)
    hu = np.full(shape, -1000, dtype=np.int16)
    lx, ly, lz = nx * vox[0], ny * vox[1], nz * vox[2]
    cx, cy, cz = 0.5 * lx, 0.5 * ly, 0.5 * lz
    body = _ellipsoid_mask(shape, vox, (cx, cy, cz), (19.0, 12.5, 10 * lz))
    inner = _ellipsoid_mask(shape, vox, (cx, cy, cz), (17.5, 11.0, 10 * lz))
    hu[body] = -100
    soft = np.clip(rng.normal(40.0, 20.0, size=shape), -100, 120).astype(np.int16)
    hu[inner] = soft[inner]
    for sgn in (-1.0, 1.0):
        for c, r in [((cx + sgn * 8.0, cy + 1.0, cz + 4.0), (4.5, 3.0, 7.0)),     # iliac wing
                     ((cx + sgn * 10.5, cy, cz - 8.0), (1.8, 1.8, 9.0))]:          # femur shaft
            m = _ellipsoid_mask(shape, vox, c, r)
            hu[m] = rng.integers(300, 1401, size=int(m.sum())).astype(np.int16)
        hu[_ellipsoid_mask(shape, vox, (cx + sgn * 9.5, cy, cz), (2.4, 2.4, 2.4))] = 3071   # head
        hu[_ellipsoid_mask(shape, vox, (cx + sgn * 10.5, cy, cz - 6.0), (0.8, 0.8, 6.0))] = 3071  # stem
    sac = _ellipsoid_mask(shape, vox, (cx, cy + 5.5, cz + 3.0), (3.5, 2.0, 6.0))
    hu[sac] = rng.integers(300, 1401, size=int(sac.sum())).astype(np.int16)
    targets = [((cx, cy - 1.0, cz), (4.0, 3.5, 4.5))]
    return hu, vox, targets
