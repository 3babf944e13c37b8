"""ctypes binding of oracle/opmc.cpp (TEST INFRASTRUCTURE ONLY)."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libopmc.so")
MAX_ELEM = 8
_D = C.POINTER(C.c_double)
_I = C.POINTER(C.c_int32)


def build_oracle(force=False):
    src = os.path.join(_HERE, "opmc.cpp")
    hdr = os.path.join(_HERE, "opmc.h")
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(src), os.path.getmtime(hdr))):
        return _SO
    cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-o", _SO, src]
    subprocess.run(cmd, check=True)
    return _SO


class Tables(C.Structure):
    _fields_ = [("n_e", C.c_int32), ("e_min", C.c_double), ("e_max", C.c_double), ("n_sr", C.c_int32),
                ("stop_mass", _D), ("ln_range", _D), ("ln_range_d2", _D), ("n_r", C.c_int32),
                ("ln_r_lo", _D), ("ln_r_hi", _D), ("ln_energy", _D), ("ln_energy_d2", _D),
                ("n_elem", C.c_int32), ("elem_z", _I), ("elem_a", _I), ("sigma_ne_mb", _D), ("sigma_el_mb", _D),
                ("mass_zdim", C.c_int32), ("mass_adim", C.c_int32), ("nuclear_mass", _D),
                ("evap_k", _D), ("evap_c", _D),
                ("e_cut", C.c_double), ("highland_factor", C.c_double), ("kappa_gauss", C.c_double),
                ("s_max_wet_cm", C.c_double), ("n_batches", C.c_int32),
                ("mol_n", C.c_int32), ("mol_dtheta", C.c_double), ("mol_c0", _D), ("mol_c1", _D), ("mol_c2", _D)]


class HuBin(C.Structure):
    _fields_ = [("hu_lo", C.c_int32), ("hu_hi", C.c_int32), ("rho_lo", C.c_double), ("rho_hi", C.c_double),
                ("w", C.c_double * MAX_ELEM), ("f_m", C.c_double), ("x0_gcm2", C.c_double), ("table_id", C.c_int32)]


class Counters(C.Structure):
    _fields_ = [(k, C.c_uint64) for k in ("n_steps", "n_draws", "n_elastic", "n_nonelastic", "n_secondary_protons",
                                          "n_missed", "n_inc_tries")] + \
               [(k, C.c_double) for k in ("e_source", "e_deposit", "e_escape", "e_neutron", "e_gamma", "e_q", "e_air",
                                          "max_ledger_residual", "max_event_residual")] + \
               [(k, C.c_uint64) for k in ("n_zab_violations", "n_inc_guard_trips", "n_inc_stack_trips", "inc_max_stack",
                                          "inc_max_out")]


SECONDARY_DTYPE = np.dtype([("Z", "<i2"), ("A", "<i2"), ("origin", "u1"), ("pad", "u1", (3,)),
                            ("ke", "<f4"), ("dir", "<f4", (3,))])
assert SECONDARY_DTYPE.itemsize == 24

_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build_oracle())
        _lib.opmc_last_error.restype = C.c_char_p
        for f in ("opmc_test_range_gcm2", "opmc_test_energy_of_range", "opmc_test_inc_uniform_sphere",
                  "opmc_test_nucleus", "opmc_test_nucleus_neutron", "opmc_test_fermi_p2", "opmc_test_cugnon"):
            getattr(_lib, f).restype = C.c_double
    return _lib


def _dp(a):
    return a.ctypes.data_as(_D)


def philox4x32_10(ctr, key):
    lib = _load()
    c = (C.c_uint32 * 4)(*ctr); k = (C.c_uint32 * 2)(*key); o = (C.c_uint32 * 4)()
    lib.opmc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def cugnon(which, p_gev):
    return _load().opmc_test_cugnon(C.c_int(which), C.c_double(p_gev))


def inc_uniform_sphere(radius_fm, rho_fm3, sigma_mb, t_mev, n, seed):
    return _load().opmc_test_inc_uniform_sphere(C.c_double(radius_fm), C.c_double(rho_fm3), C.c_double(sigma_mb),
                                                C.c_double(t_mev), C.c_uint64(n), C.c_uint64(seed))


def nn_cos(same_type, p_lab_gev, pcm_mev, n, seed):
    out = np.zeros(n)
    _load().opmc_test_nn_cos(C.c_int(int(same_type)), C.c_double(p_lab_gev), C.c_double(pcm_mev), C.c_uint64(n),
                             C.c_uint64(seed), _dp(out))
    return out


def inc_custom(rout, rho, pF, V, t_in, n, seed, coulomb=-1e9, pauli=False, const_sigma_mb=-1.0):
    """Cascade attempts on a hand-made shell nucleus; rho, pF, V have shape (2, nshell) (proton row, neutron row).
    Returns (n_out[n], rec[n][4][5]) with rec = type (0 p, 1 n), KE, direction of the first four outgoing nucleons;
    n_out < 0 marks a rejected attempt with -1 - n_out nucleons out."""
    rout = np.ascontiguousarray(rout, dtype=np.float64); ns = rout.size
    arrs = [np.ascontiguousarray(a, dtype=np.float64).reshape(2, ns) for a in (rho, pF, V)]
    out_n = np.zeros(n, dtype=np.int32); rec = np.zeros((n, 4, 5))
    rc = _load().opmc_test_inc_custom(C.c_int(ns), _dp(rout), _dp(arrs[0]), _dp(arrs[1]), _dp(arrs[2]), C.c_double(coulomb),
                                      C.c_int(int(pauli)), C.c_double(const_sigma_mb), C.c_double(t_in), C.c_uint64(n),
                                      C.c_uint64(seed), out_n.ctypes.data_as(_I), _dp(rec))
    assert rc == 0
    return out_n, rec


class Oracle:
    """Host-pointer mirror of the five pmc_* calls, driven by the dicts of `inputs`."""

    def __init__(self, tables=None, materials=None):
        self.lib = _load()
        self.ctx = C.c_void_p()
        assert self.lib.opmc_create(C.byref(self.ctx)) == 0
        self._keep = []
        self.nvox = 0
        if tables is not None:
            self.load_physics_tables(tables)
        if materials is not None:
            self.set_hu_materials(materials)

    def __del__(self):
        try:
            self.lib.opmc_destroy(self.ctx)
        except Exception:
            pass

    def _chk(self, rc):
        if rc != 0:
            raise RuntimeError("oracle: " + self.lib.opmc_last_error(self.ctx).decode())

    def load_physics_tables(self, t):
        s = Tables()
        keep = {}
        for name, ct in Tables._fields_:
            v = t[name]
            if ct is _D:
                keep[name] = np.ascontiguousarray(v, dtype=np.float64); setattr(s, name, _dp(keep[name]))
            elif ct is _I:
                keep[name] = np.ascontiguousarray(v, dtype=np.int32); setattr(s, name, keep[name].ctypes.data_as(_I))
            else:
                setattr(s, name, v)
        self._keep.append(keep)
        self._chk(self.lib.opmc_load_physics_tables(self.ctx, C.byref(s)))

    def set_hu_materials(self, bins):
        arr = (HuBin * len(bins))()
        for i, b in enumerate(bins):
            arr[i].hu_lo, arr[i].hu_hi = b["hu_lo"], b["hu_hi"]
            arr[i].rho_lo, arr[i].rho_hi = b["rho_lo"], b["rho_hi"]
            for k in range(MAX_ELEM):
                arr[i].w[k] = float(b["w"][k])
            arr[i].f_m, arr[i].x0_gcm2, arr[i].table_id = b["f_m"], b["x0_gcm2"], b["table_id"]
        self._chk(self.lib.opmc_set_hu_materials(self.ctx, arr, len(bins)))

    def load_ct(self, hu, vox, origin=(0.0, 0.0, 0.0)):
        hu = np.ascontiguousarray(hu, dtype=np.int16)
        nz, ny, nx = hu.shape
        self.shape = hu.shape
        self.nvox = hu.size
        org = (C.c_double * 3)(*origin)
        self._chk(self.lib.opmc_load_ct(self.ctx, hu.ctypes.data_as(C.POINTER(C.c_int16)), nx, ny, nz,
                                        C.c_double(vox[0]), C.c_double(vox[1]), C.c_double(vox[2]), org))

    def set_option(self, key, value):
        self._chk(self.lib.opmc_set_option(self.ctx, key.encode(), C.c_double(value)))

    def simulate(self, spots, n_histories, seed):
        spots = np.ascontiguousarray(spots, dtype=np.float64)
        dose = np.zeros(self.nvox); sigma = np.zeros(self.nvox)
        self._chk(self.lib.opmc_simulate(self.ctx, spots.ctypes.data_as(C.c_void_p), spots.shape[0],
                                         C.c_uint64(n_histories), C.c_uint64(seed), _dp(dose), _dp(sigma)))
        return dose.reshape(self.shape), sigma.reshape(self.shape)

    def set_dose_influence(self, roi_voxels):
        roi = np.ascontiguousarray(roi_voxels, dtype=np.int32)
        self.n_roi = int(roi.size)
        self._chk(self.lib.opmc_set_dose_influence(self.ctx, roi.ctypes.data_as(C.POINTER(C.c_int32)), C.c_int(self.n_roi)))

    def dose_influence(self, nspots):
        out = np.zeros((nspots, self.n_roi), dtype=np.float64)
        self._chk(self.lib.opmc_get_dose_influence(self.ctx, _dp(out)))
        return out

    def letd(self):
        """LET_d map (keV/um) of the last simulate() made with set_option("score_letd", 1)."""
        out = np.zeros(self.shape, dtype=np.float64)
        self._chk(self.lib.opmc_get_letd(self.ctx, _dp(out)))
        return out

    def nonelastic(self, Z, A, e_mev, n, seed, capacity=None):
        capacity = capacity or 24 * n + 64
        out = np.zeros(capacity, dtype=SECONDARY_DTYPE)
        off = np.zeros(n + 1, dtype=np.uint32)
        n_out = C.c_uint64()
        self._chk(self.lib.opmc_nonelastic(self.ctx, Z, A, C.c_double(e_mev), C.c_uint64(n), C.c_uint64(seed),
                                           out.ctypes.data_as(C.c_void_p), C.c_uint64(capacity),
                                           off.ctypes.data_as(C.POINTER(C.c_uint32)), C.byref(n_out)))
        return out[:n_out.value], off

    def counters(self):
        c = Counters()
        self.lib.opmc_get_counters(self.ctx, C.byref(c))
        return {k: getattr(c, k) for k, _ in Counters._fields_}

    # ---- pin-test hooks
    def range_gcm2(self, table, e):
        return self.lib.opmc_test_range_gcm2(self.ctx, table, C.c_double(e))

    def energy_of_range(self, table, r):
        return self.lib.opmc_test_energy_of_range(self.ctx, table, C.c_double(r))

    def straggle(self, e, mean_loss, rho_l, zoa, n, seed):
        out = np.zeros(n)
        self.lib.opmc_test_straggle(self.ctx, C.c_double(e), C.c_double(mean_loss), C.c_double(rho_l), C.c_double(zoa),
                                    C.c_uint64(n), C.c_uint64(seed), _dp(out))
        return out

    def first_steps(self, spot, n, seed, max_steps):
        spot = np.ascontiguousarray(spot, dtype=np.float64)
        out = np.zeros((n, 8))
        self.lib.opmc_test_first_steps(self.ctx, spot.ctypes.data_as(C.c_void_p), C.c_uint64(n), C.c_uint64(seed),
                                       max_steps, _dp(out))
        return out

    def elastic(self, Z, A, t_mev, n, seed):
        out = np.zeros((n, 4))
        self.lib.opmc_test_elastic(self.ctx, Z, A, C.c_double(t_mev), C.c_uint64(n), C.c_uint64(seed), _dp(out))
        return out

    def sample_primaries(self, spots, n, seed):
        spots = np.ascontiguousarray(spots, dtype=np.float64)
        out = np.zeros((n, 8))
        assert self.lib.opmc_test_sample_primaries(self.ctx, spots.ctypes.data_as(C.c_void_p), spots.shape[0], C.c_uint64(n),
                                                   C.c_uint64(seed), _dp(out)) == 0
        return out

    def event_counts(self):
        out = np.zeros(16, dtype=np.uint64)
        self.lib.opmc_test_event_counts(self.ctx, out.ctypes.data_as(C.POINTER(C.c_uint64)))
        return out[:8].astype(np.int64), out[8:].astype(np.int64)

    def nucleus(self, Z, A):
        out = np.zeros((15, 6))
        rmax = self.lib.opmc_test_nucleus(self.ctx, Z, A, _dp(out))
        return rmax, out

    def nucleus_neutron(self, Z, A):
        """-> (Coulomb barrier B_C, [15][3] = pF_n, EF_n, V_n)."""
        out = np.zeros((15, 3))
        bc = self.lib.opmc_test_nucleus_neutron(self.ctx, Z, A, _dp(out))
        return bc, out

    def fermi_p2(self, Z, A, n, seed):
        return self.lib.opmc_test_fermi_p2(self.ctx, Z, A, C.c_uint64(n), C.c_uint64(seed))

    def evap_first(self, Z, A, estar, mask, n, seed):
        widths = np.zeros(6); ch = np.zeros(n, dtype=np.int32); eps = np.zeros(n); cs = np.zeros(n)
        self.lib.opmc_test_evap_first(self.ctx, Z, A, C.c_double(estar), C.c_uint32(mask), C.c_uint64(n),
                                      C.c_uint64(seed), _dp(widths), ch.ctypes.data_as(_I), _dp(eps), _dp(cs))
        return widths, ch, eps, cs
