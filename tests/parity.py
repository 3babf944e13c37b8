"""Statistical-parity helpers applied identically to the oracle's and the CUDA path's outputs.

Holds no physics of the method: only the comparison statistics north_star names (integrated dose, voxel
z-scores, R80 / distal fall-off, yields).
"""
from __future__ import annotations

import numpy as np

GY_PER_MEV_G = 1.602176634e-10


def depth_dose(dose, axis=0):
    """Integrated depth dose along `axis` of a (nz, ny, nx) grid."""
    other = tuple(a for a in range(3) if a != axis)
    return np.asarray(dose, dtype=np.float64).sum(axis=other)


def distal_depth(dd, d_cm, level):
    """Depth (cm, slab centres) on the distal side of the peak where dd falls to level * max."""
    dd = np.asarray(dd, dtype=np.float64)
    ipk = int(np.argmax(dd))
    thr = level * dd[ipk]
    for i in range(ipk, len(dd) - 1):
        if dd[i] >= thr > dd[i + 1]:
            f = (dd[i] - thr) / (dd[i] - dd[i + 1])
            return (i + 0.5 + f) * d_cm
    return float("nan")


def distal_depth_from_end(dd, d_cm, level):
    """The same level crossing searched from the far end of the profile (a spread-out Bragg peak has a rippled plateau:
    its maximum is not a landmark, its distal edge is)."""
    dd = np.asarray(dd, dtype=np.float64)
    thr = level * dd.max()
    for i in range(len(dd) - 2, -1, -1):
        if dd[i] >= thr > dd[i + 1]:
            f = (dd[i] - thr) / (dd[i] - dd[i + 1])
            return (i + 0.5 + f) * d_cm
    return float("nan")


def r80_and_falloff(dd, d_cm):
    r80 = distal_depth(dd, d_cm, 0.8)
    r20 = distal_depth(dd, d_cm, 0.2)
    return r80, r20 - r80


def zscore_pass(d_a, s_a, d_b, s_b, frac_of_max=0.1, nsig=3.0, region=None):
    """Fraction of voxels with d_b > frac*max within nsig combined sigma; also mean and rms z.  `region` (bool grid)
    restricts both the maximum and the voxels compared (e.g. to tissue, leaving out air voxels whose dose-to-medium
    is a 1000x spike whenever a single proton stops in them)."""
    d_a = np.asarray(d_a, dtype=np.float64); d_b = np.asarray(d_b, dtype=np.float64)
    s = np.sqrt(np.asarray(s_a, dtype=np.float64) ** 2 + np.asarray(s_b, dtype=np.float64) ** 2)
    if region is None:
        region = np.ones(d_b.shape, dtype=bool)
    m = region & (d_b > frac_of_max * d_b[region].max()) & (s > 0)
    z = (d_a[m] - d_b[m]) / s[m]
    return float(np.mean(np.abs(z) <= nsig)), float(z.mean()), float(z.std()), int(m.sum())


def species_yields(sec, off):
    """Per-event multiplicities of n, p, d, t, 3He, alpha (INC + evaporation): array (n_events, 6)."""
    n = len(off) - 1
    ev = np.repeat(np.arange(n), np.diff(off).astype(np.int64))
    out = np.zeros((n, 6))
    for j, (z, a) in enumerate([(0, 1), (1, 1), (1, 2), (1, 3), (2, 3), (2, 4)]):
        m = (sec["Z"] == z) & (sec["A"] == a) & (sec["origin"] < 2)
        out[:, j] = np.bincount(ev[m], minlength=n)
    return out


def chi2_hist(a, b, bins):
    """Two-sample chi^2 per degree of freedom of histograms with Poisson errors (bins with >= 20 entries)."""
    ha, _ = np.histogram(a, bins=bins)
    hb, _ = np.histogram(b, bins=bins)
    m = (ha + hb) >= 40
    na, nb = ha.sum(), hb.sum()
    if m.sum() < 2:
        return 0.0, 0
    k1, k2 = np.sqrt(nb / na), np.sqrt(na / nb)
    chi2 = np.sum((k1 * ha[m] - k2 * hb[m]) ** 2 / (ha[m] + hb[m]))
    return float(chi2 / m.sum()), int(m.sum())
