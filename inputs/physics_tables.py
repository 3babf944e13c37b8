"""Physics input tables (stand-ins for the paper's Geant4-derived tables).

The paper reads these from Geant4.9.6p2 (PAPER.md:L53 dE/dx for water, air,
titanium + CSDA range tables with precomputed spline second derivatives; L75
non-elastic and L83 elastic cross-section tables; ref [21] evaporation
parameters).  None of that is in the container, so they are generated here from
closed formulas and handed, as plain
arrays, to BOTH the oracle and the CUDA library through their
`*_load_physics_tables` calls.  This is data generation, not the method.
"""
from __future__ import annotations

import functools

import numpy as np
from scipy.interpolate import CubicSpline

M_P = 938.27208816      # MeV
M_N = 939.56542052
M_E = 0.51099895
K_BETHE = 0.307075      # MeV cm^2 / mol

# element list used by all configs (one isotope per element)
ELEMENTS = [("H", 1, 1), ("C", 6, 12), ("N", 7, 14), ("O", 8, 16),
            ("P", 15, 31), ("Ca", 20, 40), ("Ti", 22, 48)]
ELEM_I_EV = {1: 19.2, 6: 81.0, 7: 82.0, 8: 95.0, 15: 173.0, 20: 191.0, 22: 233.0}
ELEM_ATOMIC_WEIGHT = {1: 1.008, 6: 12.011, 7: 14.007, 8: 15.999, 15: 30.974,
                      20: 40.078, 22: 47.867}

# dedicated stopping/range tables: id 0 water (scaled by Eq.1/2), 1 air, 2 titanium
SR_MEDIA = [("water", 0.555087, 75.0), ("air", 0.499190, 85.7), ("titanium", 22 / 47.867, 233.0)]

N_E = 256
E_MIN, E_MAX = 0.05, 300.0
N_R = 256
MASS_ZDIM, MASS_ADIM = 24, 51
EJECTILES = [(0, 1), (1, 1), (1, 2), (1, 3), (2, 3), (2, 4)]   # n p d t 3He alpha


def bethe_mass_stopping(e_mev, z_over_a, i_ev):
    """Plain Bethe formula, MeV cm^2/g (no shell/density/Barkas terms); power law below 1 MeV."""
    e = np.asarray(e_mev, dtype=np.float64)

    def bethe(t):
        g = 1.0 + t / M_P
        b2 = 1.0 - 1.0 / (g * g)
        bg2 = b2 * g * g
        tmax = 2 * M_E * bg2 / (1 + 2 * g * M_E / M_P + (M_E / M_P) ** 2)
        i = i_ev * 1e-6
        return K_BETHE * z_over_a / b2 * (0.5 * np.log(2 * M_E * bg2 * tmax / (i * i)) - b2)

    s1 = bethe(1.0)
    return np.where(e >= 1.0, bethe(np.maximum(e, 1.0)), s1 * np.power(e, -0.77))


def _csda_range(e_knots, z_over_a, i_ev):
    """R(E)=int_0^E dE'/S, Gauss-Legendre (8 pt) on 16 log sub-intervals per knot interval."""
    s0 = bethe_mass_stopping(e_knots[0], z_over_a, i_ev)
    r0 = e_knots[0] / (1.77 * s0)          # analytic integral of the E^-0.77 power law from 0
    xg, wg = np.polynomial.legendre.leggauss(8)
    lk = np.log(e_knots)
    out = np.empty_like(e_knots)
    out[0] = r0
    acc = r0
    nsub = 16
    for i in range(len(e_knots) - 1):
        edges = np.linspace(lk[i], lk[i + 1], nsub + 1)
        a, b = edges[:-1, None], edges[1:, None]
        x = 0.5 * (b - a) * xg[None, :] + 0.5 * (b + a)
        ee = np.exp(x)
        f = ee / bethe_mass_stopping(ee, z_over_a, i_ev)     # dE = E dlnE
        acc += float(np.sum(0.5 * (b - a) * f * wg[None, :]))
        out[i + 1] = acc
    return out


def letaw_sigma_ne_mb(a, e_mev):
    e = np.maximum(np.asarray(e_mev, dtype=np.float64), 1e-3)
    s = 45.0 * a ** 0.7 * (1 + 0.016 * np.sin(5.3 - 2.63 * np.log(a)))
    return s * (1 - 0.62 * np.exp(-e / 200.0) * np.sin(10.9 * e ** -0.28))


def cugnon_sigma_pp_mb(p_gev):
    p = np.asarray(p_gev, dtype=np.float64)
    return np.where(p < 0.44, 34.0 * (np.maximum(p, 1e-6) / 0.4) ** -2.104,
           np.where(p < 0.8, 23.5 + 1000.0 * (p - 0.7) ** 4,
           np.where(p < 2.0, 1250.0 / (p + 50.0) - 4.0 * (p - 1.3) ** 2, 77.0 / (p + 1.5))))


def semi_empirical_mass_table():
    """Nuclear ground-state masses (MeV); 0 marks "not a nuclide".  Bethe-Weizsaecker + exact light ones."""
    m = np.zeros((MASS_ZDIM, MASS_ADIM))
    av, as_, ac, aa, ap = 15.75, 17.8, 0.711, 23.7, 11.18
    for z in range(MASS_ZDIM):
        for a in range(1, MASS_ADIM):
            n = a - z
            if n < 0:
                continue
            if a == 1:
                m[z, a] = M_P if z == 1 else M_N
                continue
            if z == 0 or n == 0:
                continue                      # di-neutron, di-proton ... : unbound
            b = av * a - as_ * a ** (2 / 3) - ac * z * (z - 1) / a ** (1 / 3) - aa * (a - 2 * z) ** 2 / a
            if z % 2 == 0 and n % 2 == 0:
                b += ap / np.sqrt(a)
            elif z % 2 == 1 and n % 2 == 1:
                b -= ap / np.sqrt(a)
            if b <= 0:
                continue
            m[z, a] = z * M_P + n * M_N - b
    for (z, a, b) in [(1, 2, 2.2246), (1, 3, 8.4818), (2, 3, 7.7180), (2, 4, 28.2957)]:
        m[z, a] = z * M_P + (a - z) * M_N - b
    return m


def _dostrovsky_tables():
    zk = np.array([10.0, 20.0, 30.0, 50.0, 70.0])
    kp = np.array([0.42, 0.58, 0.68, 0.77, 0.80]); cp = np.array([0.50, 0.28, 0.20, 0.15, 0.10])
    ka = np.array([0.68, 0.82, 0.91, 0.97, 0.98]); ca = np.array([0.10, 0.10, 0.10, 0.08, 0.06])
    zd = np.arange(MASS_ZDIM, dtype=np.float64)
    kp_z, cp_z = np.interp(zd, zk, kp), np.interp(zd, zk, cp)
    ka_z, ca_z = np.interp(zd, zk, ka), np.interp(zd, zk, ca)
    k = np.zeros((6, MASS_ZDIM)); c = np.zeros((6, MASS_ZDIM))
    k[1], c[1] = kp_z, cp_z
    k[2], c[2] = kp_z + 0.06, cp_z / 2
    k[3], c[3] = kp_z + 0.12, cp_z / 3
    k[4], c[4] = ka_z - 0.06, 4 * ca_z / 3
    k[5], c[5] = ka_z, ca_z
    return k, c


MOL_N, MOL_DTHETA = 241, 0.05     # reduced-angle grid 0 .. 12 of the Moliere tables


@functools.lru_cache(maxsize=2)
def moliere_tables(n=MOL_N, dtheta=MOL_DTHETA):
    """Cumulative Moliere functions on a uniform grid of the reduced angle ("full Moliere"; Bethe 1953):
    C_k[m] = int_0^{theta_m} theta f^(k)(theta) dtheta, k = 0, 1, 2, with
    f^(k)(theta) = 1/k! int_0^inf u du J0(theta u) exp(-u^2/4) [(u^2/4) ln(u^2/4)]^k     (f^(0) = 2 exp(-theta^2)).
    Plain quadrature of the defining integrals (Simpson in u, trapezoid in theta on a 4x finer grid)."""
    from scipy.special import j0
    fine = 4
    th = np.arange((n - 1) * fine + 1) * (dtheta / fine)
    u = np.linspace(0.0, 16.0, 16001)
    w = np.ones_like(u); w[1:-1:2] = 4.0; w[2:-1:2] = 2.0; w *= (u[1] - u[0]) / 3.0      # Simpson
    s = u * u / 4.0
    sl = np.where(s > 0, s * np.log(np.maximum(s, 1e-300)), 0.0)
    base = w * u * np.exp(-s)
    out = []
    for k, fac in ((0, 1.0), (1, 1.0), (2, 0.5)):
        g = base * sl ** k * fac
        f = np.array([np.dot(g, j0(t * u)) for t in th])
        integrand = th * f
        cum = np.concatenate([[0.0], np.cumsum(0.5 * (integrand[1:] + integrand[:-1]) * (dtheta / fine))])
        out.append(np.ascontiguousarray(cum[::fine]))
    return out


def make_physics_tables(e_cut_mev=0.1, highland_factor=1.07, kappa_gauss=10.0,
                        s_max_wet_cm=0.2, n_batches=10):
    """Return a dict of C-contiguous float64/int32 arrays + scalar options."""
    e = np.exp(np.linspace(np.log(E_MIN), np.log(E_MAX), N_E))
    mol = moliere_tables()
    n_sr = len(SR_MEDIA)
    stop = np.empty((n_sr, N_E)); ln_r = np.empty((n_sr, N_E)); ln_r_d2 = np.empty((n_sr, N_E))
    ln_r_lo = np.empty(n_sr); ln_r_hi = np.empty(n_sr)
    ln_e = np.empty((n_sr, N_R)); ln_e_d2 = np.empty((n_sr, N_R))
    x = np.log(e)
    # dense forward table for the inverse (16x finer than the knots)
    e_dense = np.exp(np.linspace(np.log(E_MIN), np.log(E_MAX), (N_E - 1) * 16 + 1))
    for t, (_, zoa, i_ev) in enumerate(SR_MEDIA):
        stop[t] = bethe_mass_stopping(e, zoa, i_ev)
        r_dense = _csda_range(e_dense, zoa, i_ev)
        r = r_dense[::16]
        ln_r[t] = np.log(r)
        ln_r_d2[t] = CubicSpline(x, ln_r[t], bc_type="natural")(x, 2)
        ln_r_lo[t], ln_r_hi[t] = ln_r[t, 0], ln_r[t, -1]
        xr = np.linspace(ln_r_lo[t], ln_r_hi[t], N_R)
        dense_spl = CubicSpline(np.log(r_dense), np.log(e_dense))   # very dense: error ~1e-10
        ln_e[t] = dense_spl(xr)
        ln_e[t, 0], ln_e[t, -1] = x[0], x[-1]
        ln_e_d2[t] = CubicSpline(xr, ln_e[t], bc_type="natural")(xr, 2)

    n_el = len(ELEMENTS)
    s_ne = np.zeros((n_el, N_E)); s_el = np.zeros((n_el, N_E))
    p_gev = np.sqrt(e * (e + 2 * M_P)) / 1000.0
    for i, (_, z, a) in enumerate(ELEMENTS):
        if a == 1:
            s_el[i] = np.minimum(cugnon_sigma_pp_mb(p_gev), 1000.0)
            continue
        e_b = 1.44 * z / (1.3 * (a ** (1 / 3) + 1.0))           # Coulomb barrier, MeV
        cut = 1.0 / (1.0 + np.exp((e_b - e) / (0.25 * e_b)))
        s_ne[i] = np.maximum(letaw_sigma_ne_mb(a, e), 0.0) * cut
        s_el[i] = s_ne[i] * (0.3 + 0.7 * np.exp(-e / 150.0))     # placeholder magnitude (not from the paper)
    masses = semi_empirical_mass_table()
    ek, ec = _dostrovsky_tables()
    c = np.ascontiguousarray
    return dict(
        n_e=N_E, e_min=E_MIN, e_max=E_MAX, n_sr=n_sr,
        stop_mass=c(stop), ln_range=c(ln_r), ln_range_d2=c(ln_r_d2),
        n_r=N_R, ln_r_lo=c(ln_r_lo), ln_r_hi=c(ln_r_hi), ln_energy=c(ln_e), ln_energy_d2=c(ln_e_d2),
        n_elem=n_el,
        elem_z=np.array([z for _, z, _ in ELEMENTS], dtype=np.int32),
        elem_a=np.array([a for _, _, a in ELEMENTS], dtype=np.int32),
        sigma_ne_mb=c(s_ne), sigma_el_mb=c(s_el),
        mass_zdim=MASS_ZDIM, mass_adim=MASS_ADIM, nuclear_mass=c(masses),
        evap_k=c(ek), evap_c=c(ec),
        e_cut=float(e_cut_mev), highland_factor=float(highland_factor), kappa_gauss=float(kappa_gauss),
        s_max_wet_cm=float(s_max_wet_cm), n_batches=int(n_batches),
        mol_n=MOL_N, mol_dtheta=MOL_DTHETA, mol_c0=mol[0], mol_c1=mol[1], mol_c2=mol[2],
    )
