"""3-D gamma index (ref [34]; Low et al. 1998) — fp64 oracle, TEST INFRASTRUCTURE ONLY.

The plain definition written out (DESIGN.md Reading R10), no blocking or early exits:

    gamma(r) = min over r' of sqrt( |r' - r|^2 / DTA^2 + (D_eval(r') - D_ref(r))^2 / dD^2 ),
    dD = dd_frac * max(D_ref)                       (global dose-difference criterion, e.g. 2 %)

for every reference voxel r with D_ref(r) >= low_dose_frac * max(D_ref); r' runs over the centres of the evaluated
grid's voxels with |r' - r| <= search_cm (no sub-voxel interpolation).  Voxels below the threshold get -1.
Only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import this module; it shares nothing with the CUDA
path.
"""
from __future__ import annotations

import numpy as np


def gamma_index(ref, ev, vox_cm, dd_frac=0.02, dta_cm=0.2, low_dose_frac=0.1, search_cm=None):
    """ref, ev: (nz, ny, nx) arrays; vox_cm = (dx, dy, dz).  Returns (gamma (nz, ny, nx) float64, pass_rate)."""
    ref = np.asarray(ref, dtype=np.float64); ev = np.asarray(ev, dtype=np.float64)
    assert ref.shape == ev.shape and ref.ndim == 3
    dx, dy, dz = (float(v) for v in vox_cm)
    if search_cm is None:
        search_cm = 2.0 * dta_cm
    dmax = ref.max()
    dd = dd_frac * dmax
    nz, ny, nx = ref.shape
    rx, ry, rz = int(np.floor(search_cm / dx + 1e-9)), int(np.floor(search_cm / dy + 1e-9)), int(np.floor(search_cm / dz + 1e-9))
    g2 = np.full(ref.shape, np.inf)
    for k in range(-rz, rz + 1):
        for j in range(-ry, ry + 1):
            for i in range(-rx, rx + 1):
                d2 = (i * dx) ** 2 + (j * dy) ** 2 + (k * dz) ** 2
                if d2 > search_cm * search_cm * (1 + 1e-12):
                    continue
                # evaluated dose at r + (i, j, k), where that voxel exists
                z0, z1 = max(0, -k), min(nz, nz - k)
                y0, y1 = max(0, -j), min(ny, ny - j)
                x0, x1 = max(0, -i), min(nx, nx - i)
                if z0 >= z1 or y0 >= y1 or x0 >= x1:
                    continue
                diff = ev[z0 + k:z1 + k, y0 + j:y1 + j, x0 + i:x1 + i] - ref[z0:z1, y0:y1, x0:x1]
                cand = d2 / (dta_cm * dta_cm) + diff * diff / (dd * dd)
                np.minimum(g2[z0:z1, y0:y1, x0:x1], cand, out=g2[z0:z1, y0:y1, x0:x1])
    gamma = np.sqrt(g2)
    mask = ref >= low_dose_frac * dmax
    gamma = np.where(mask, gamma, -1.0)
    n = int(mask.sum())
    return gamma, (float(np.mean(gamma[mask] <= 1.0)) if n else 1.0)
