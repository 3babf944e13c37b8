"""HU -> material tables (synthetic, Schneider-shaped).

The paper's own 26-material table is not in the container and is not
reproduced.  Each bin carries density (linear in HU inside the bin), elemental
mass fractions over inputs.ELEMENTS, the water-scaling factor f_m of Eq.1/Eq.2
("tabulated as a function of HU") and the radiation length
("pre-calculated"), i.e. the quantities the paper takes as inputs.
"""
from __future__ import annotations

import numpy as np

from .physics_tables import (ELEMENTS, ELEM_I_EV, ELEM_ATOMIC_WEIGHT, bethe_mass_stopping)

MAX_ELEM = 8
HU_MIN, HU_MAX = -1024, 32767

W_AIR = {7: 0.765, 8: 0.235}
W_WATER = {1: 0.1119, 8: 0.8881}
W_SOFT = {1: 0.101, 6: 0.111, 7: 0.026, 8: 0.762}
W_CORT = {1: 0.034, 6: 0.155, 7: 0.042, 8: 0.435, 15: 0.103, 20: 0.225}
W_TI = {22: 1.0}


def _wvec(wd):
    w = np.zeros(MAX_ELEM)
    for i, (_, z, _) in enumerate(ELEMENTS):
        w[i] = wd.get(z, 0.0)
    return w / w.sum()


def _x0_elem(z, aw):
    return 716.4 * aw / (z * (z + 1) * np.log(287.0 / np.sqrt(z)))


def _derived(w):
    """(f_m at 100 MeV, X0 in g/cm^2) from Bragg additivity — generator-side data preparation."""
    zoa = 0.0; lni = 0.0; inv_x0 = 0.0
    for i, (_, z, _) in enumerate(ELEMENTS):
        if w[i] <= 0:
            continue
        aw = ELEM_ATOMIC_WEIGHT[z]
        zoa += w[i] * z / aw
        lni += w[i] * z / aw * np.log(ELEM_I_EV[z])
        inv_x0 += w[i] / _x0_elem(z, aw)
    i_ev = float(np.exp(lni / zoa))
    f_m = float(bethe_mass_stopping(100.0, zoa, i_ev) / bethe_mass_stopping(100.0, 0.555087, 75.0))
    return f_m, 1.0 / inv_x0


def _rho(hu):
    return max(0.0012, 1.0 + hu / 1000.0) if hu <= 0 else 1.0 + 0.0006 * hu


def _bin(lo, hi, w, table_id=0, rho=None, exact_water=False):
    f_m, x0 = _derived(w)
    if exact_water:
        f_m, x0 = 1.0, 36.08
    r_lo, r_hi = (rho, rho) if rho is not None else (_rho(lo), _rho(hi))
    return dict(hu_lo=int(lo), hu_hi=int(hi), rho_lo=float(r_lo), rho_hi=float(r_hi),
                w=w.copy(), f_m=f_m, x0_gcm2=float(x0), table_id=int(table_id))


def make_materials_c1():
    """3 bins: air / exact water (rho = 1.000) / titanium."""
    return [_bin(HU_MIN, -5, _wvec(W_AIR), table_id=1, rho=0.0012),
            _bin(-5, 6, _wvec(W_WATER), rho=1.0, exact_water=True),
            _bin(6, HU_MAX + 1, _wvec(W_TI), table_id=2, rho=4.5)]


def make_materials_24():
    soft, cort = _wvec(W_SOFT), _wvec(W_CORT)
    bins = [_bin(HU_MIN, -950, _wvec(W_AIR), table_id=1, rho=0.0012),
            _bin(-950, -120, soft)]
    for lo, hi in [(-120, -70), (-70, -20), (-20, -5)]:
        bins.append(_bin(lo, hi, soft))
    bins.append(_bin(-5, 6, _wvec(W_WATER), rho=1.0, exact_water=True))
    for lo, hi in [(6, 40), (40, 80), (80, 120)]:
        bins.append(_bin(lo, hi, soft))
    edges = [120, 300] + list(range(400, 1501, 100)) + [3060]
    for lo, hi in zip(edges[:-1], edges[1:]):
        t = min(1.0, max(0.0, (0.5 * (lo + min(hi, 1500)) - 120.0) / (1500.0 - 120.0)))
        w = (1 - t) * soft + t * cort
        bins.append(_bin(lo, hi, w / w.sum()))
    bins.append(_bin(3060, HU_MAX + 1, _wvec(W_TI), table_id=2, rho=4.5))
    assert len(bins) == 24
    return bins
