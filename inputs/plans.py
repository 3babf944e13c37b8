"""Seeded synthetic scanned-pencil-beam plans (stand-ins for the TPS plans).

A plan is a float64 array of shape (nspots, 13) with columns
  pos_cm[3], dir[3], e_mev, sigma_e_mev, sigma_x_cm, sigma_y_cm, div_x_rad, div_y_rad, weight
(the field order of `pmc_spot` in include/pmc.h).  The paper's nozzle phase space
(L98-106) is vendor data and is replaced by these parametric Gaussian spots.
"""
from __future__ import annotations

import numpy as np

SPOT_COLS = 13


def bev_axes(d):
    """Transverse basis (e_x, e_y) of the plane normal to unit axis d (same convention as pmc.h)."""
    d = np.asarray(d, dtype=np.float64)
    a = np.array([0.0, 1.0, 0.0]) if abs(d[2]) >= 0.9 else np.array([0.0, 0.0, 1.0])
    ex = np.cross(a, d); ex /= np.linalg.norm(ex)
    ey = np.cross(d, ex)
    return ex, ey


def plan_single_spot(pos, e_mev, sigma_cm, direction=(0.0, 0.0, 1.0), sigma_e=0.0, div=0.0):
    s = np.zeros((1, SPOT_COLS))
    s[0, 0:3] = pos; s[0, 3:6] = direction
    s[0, 6] = e_mev; s[0, 7] = sigma_e; s[0, 8] = s[0, 9] = sigma_cm
    s[0, 10] = s[0, 11] = div; s[0, 12] = 1.0
    return s


def _rho_of_hu(hu):
    hu = hu.astype(np.float64)
    return np.where(hu <= 0, np.maximum(0.0012, 1.0 + hu / 1000.0), 1.0 + 0.0006 * hu)


def _field_spots(hu, vox, targets, direction, rng, spacing, layer_wet, e_lo, e_hi, src_dist, div):
    nz, ny, nx = hu.shape
    size = np.array([nx * vox[0], ny * vox[1], nz * vox[2]])
    d = np.asarray(direction, dtype=np.float64); d /= np.linalg.norm(d)
    ex, ey = bev_axes(d)
    iso = np.mean([np.asarray(c) for c, _ in targets], axis=0)
    rmax = max(max(r) for _, r in targets) + max(np.linalg.norm(np.asarray(c) - iso) for c, _ in targets)
    g = np.arange(-np.ceil(rmax / spacing), np.ceil(rmax / spacing) + 1) * spacing
    gu, gv = np.meshgrid(g, g, indexing="ij")
    gu, gv = gu.ravel(), gv.ravel()
    p0 = iso[None, :] + gu[:, None] * ex[None, :] + gv[:, None] * ey[None, :] - src_dist * d[None, :]
    # chord through each target ellipsoid
    ds = 0.05
    s = np.arange(0.0, src_dist + rmax + 1.0, ds) + 0.5 * ds
    pts = p0[:, None, :] + s[None, :, None] * d[None, None, :]
    idx = np.floor(pts / np.asarray(vox)[None, None, :]).astype(np.int64)
    inside = np.all((idx >= 0) & (idx < np.array([nx, ny, nz])[None, None, :]), axis=2)
    idc = np.clip(idx, 0, np.array([nx, ny, nz]) - 1)
    rho = np.where(inside, _rho_of_hu(hu[idc[..., 2], idc[..., 1], idc[..., 0]]), 0.0012)
    wet = np.cumsum(rho * ds, axis=1)
    in_t = np.zeros(pts.shape[:2], dtype=bool)
    for c, r in targets:
        q = (pts - np.asarray(c)[None, None, :]) / np.asarray(r)[None, None, :]
        in_t |= np.sum(q * q, axis=2) <= 1.0
    hit = in_t.any(axis=1)
    big = 1e9
    prox = np.where(in_t, wet, big).min(axis=1)
    dist = np.where(in_t, wet, -big).max(axis=1)
    lo, hi = prox[hit].min(), dist[hit].max()
    rows = []
    for lw in np.arange(lo, hi + layer_wet, layer_wet):
        e = np.clip((lw / 0.0022) ** (1.0 / 1.77), e_lo, e_hi)      # Bragg-Kleeman inverse (plan design only)
        sel = hit & (prox <= lw) & (dist + layer_wet >= lw)
        sig = 0.6 + (0.3 - 0.6) * (e - 70.0) / (200.0 - 70.0)
        sig = float(np.clip(sig, 0.25, 0.6))
        for k in np.nonzero(sel)[0]:
            rows.append(np.concatenate([p0[k], d, [e, 0.005 * e, sig, sig, div, div,
                                                   rng.lognormal(0.0, 0.5)]]))
    del size
    return rows


def plan_c4(hu, vox, targets, seed=40):
    """3 fields (two lateral, one posterior), 5 mm spot grid, 2 mm-WET layers, 70-200 MeV."""
    rng = np.random.default_rng(seed)
    rows = []
    for direction in [(1.0, 0.0, 0.0), (-1.0, 0.0, 0.0), (0.0, -1.0, 0.0)]:
        rows += _field_spots(hu, vox, targets, direction, rng, 0.5, 0.2, 70.0, 200.0, 40.0, 0.002)
    return np.ascontiguousarray(np.array(rows, dtype=np.float64))


def plan_c5(hu, vox, targets, seed=50):
    """2 opposed lateral fields, 100-230 MeV."""
    rng = np.random.default_rng(seed)
    rows = []
    for direction in [(1.0, 0.0, 0.0), (-1.0, 0.0, 0.0)]:
        rows += _field_spots(hu, vox, targets, direction, rng, 0.5, 0.2, 100.0, 230.0, 40.0, 0.002)
    return np.ascontiguousarray(np.array(rows, dtype=np.float64))
