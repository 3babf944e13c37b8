"""Thin ctypes binding of libpmc (include/pmc.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C-ABI; PyTorch is used here only to hold device
memory and to name the CUDA stream.  There is no CPU fallback: if libpmc.so is missing or no CUDA device is
present, construction fails loudly.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpmc.so")
MAX_ELEM = 8
_D = C.POINTER(C.c_double)
_I = C.POINTER(C.c_int32)

EXPORTS = ["pmc_create", "pmc_create_with_allocator", "pmc_destroy", "pmc_load_physics_tables", "pmc_set_hu_materials", "pmc_load_ct",
           "pmc_load_ct_host", "pmc_set_option", "pmc_simulate", "pmc_simulate_host", "pmc_nonelastic",
           "pmc_get_counters", "pmc_get_timing", "pmc_get_letd", "pmc_gamma_index", "pmc_gamma_index_static", "pmc_set_dose_influence", "pmc_last_error", "pmc_philox4x32_10", "pmc_range_of_energy",
           "pmc_energy_of_range", "pmc_step_range_of_energy", "pmc_step_energy_of_range", "pmc_straggle", "pmc_elastic", "pmc_first_steps"]


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
    _fields_ = [(k, C.c_uint64) for k in ("n_steps", "n_elastic", "n_nonelastic", "n_secondary_protons", "n_missed",
                                          "n_inc_tries", "n_generations")] + \
               [(k, C.c_double) for k in ("e_source", "e_deposit", "e_escape", "e_neutron", "e_gamma", "e_q", "e_air")] + \
               [(k, C.c_uint64) for k in ("n_zab_violations", "n_inc_guard_trips", "n_inc_cap_trips", "inc_max_stack",
                                          "inc_max_out", "n_host_waits")]


class Timing(C.Structure):
    _fields_ = [(k, C.c_float) for k in ("total_ms", "sampler_ms", "transport_ms", "elastic_ms", "inc_ms",
                                         "evaporation_ms", "statistics_ms")] + \
               [("launches_total", C.c_uint32), ("launches_transport", C.c_uint32)]


SECONDARY_DTYPE = np.dtype([("Z", "<i2"), ("A", "<i2"), ("origin", "u1"), ("pad", "u1", (3,)),
                            ("ke", "<f4"), ("dir", "<f4", (3,))])
assert SECONDARY_DTYPE.itemsize == 24

_ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)      # pmc_alloc_fn
_FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)               # pmc_free_fn

_lib = None


def load_library():
    """dlopen libpmc.so (never builds, never falls back)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                               "(there is no CPU fallback)")
        _lib = C.CDLL(LIB_PATH)
        _lib.pmc_last_error.restype = C.c_char_p
        _lib.pmc_last_error.argtypes = [C.c_void_p]
        _lib.pmc_destroy.restype = None
        _lib.pmc_destroy.argtypes = [C.c_void_p]
    return _lib


class PmcError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libpmc error {code}: {msg}")
        self.code = code


def _ptr(t):
    """Raw device pointer of a CUDA torch tensor (contiguous)."""
    assert t.is_cuda and t.is_contiguous()
    return C.c_void_p(t.data_ptr())


class Pmc:
    """One libpmc context on one CUDA device; methods carry the names of the C calls."""

    def __init__(self, device=0, stream=None, torch_allocator=True):
        """torch_allocator: the context's device scratch (queues, tallies, tables) comes from PyTorch's caching allocator
        through pmc_create_with_allocator, so that torch sees and accounts for it; False: plain cudaMalloc (pmc_create)."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("libpmc needs a CUDA device (no CPU fallback)")
        self.torch = torch
        self.lib = load_library()
        self.device = torch.device("cuda", device)
        self.stream = stream
        self.ctx = C.c_void_p()
        sp = C.c_void_p(stream.cuda_stream if stream is not None else 0)
        if torch_allocator:
            raw_stream = stream.cuda_stream if stream is not None else 0

            def _alloc(nbytes, _user):
                try:
                    return torch.cuda.caching_allocator_alloc(int(nbytes), device, raw_stream)
                except Exception:               # out of memory: NULL -> PMC_E_CUDA from the call that needed it
                    return None

            def _free(ptr, _user):
                torch.cuda.caching_allocator_delete(ptr)

            self._alloc_cb = _ALLOC_FN(_alloc); self._free_cb = _FREE_FN(_free)     # kept alive with the context
            rc = self.lib.pmc_create_with_allocator(C.byref(self.ctx), C.c_int(device), sp, self._alloc_cb, self._free_cb, None)
        else:
            rc = self.lib.pmc_create(C.byref(self.ctx), C.c_int(device), sp)
        if rc != 0:
            raise PmcError(rc, "pmc_create failed (no usable CUDA device?)")
        self._keep = {}
        self.shape = None

    def close(self):
        import sys
        if self.ctx and not sys.is_finalizing():      # at interpreter exit the allocator callbacks may be gone already
            self.lib.pmc_destroy(self.ctx)
        self.ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, rc):
        if rc != 0:
            raise PmcError(rc, self.lib.pmc_last_error(self.ctx).decode())

    # ---- the five calls of the paper's problem statement
    def load_physics_tables(self, t):
        s = Tables()
        keep = {}
        for name, ct in Tables._fields_:
            v = t[name]
            if ct is _D:
                keep[name] = np.ascontiguousarray(v, dtype=np.float64)
                setattr(s, name, keep[name].ctypes.data_as(_D))
            elif ct is _I:
                keep[name] = np.ascontiguousarray(v, dtype=np.int32)
                setattr(s, name, keep[name].ctypes.data_as(_I))
            else:
                setattr(s, name, v)
        self._chk(self.lib.pmc_load_physics_tables(self.ctx, C.byref(s)))

    def set_hu_materials(self, bins):
        arr = (HuBin * len(bins))()
        for i, b in enumerate(bins):
            arr[i].hu_lo, arr[i].hu_hi = b["hu_lo"], b["hu_hi"]
            arr[i].rho_lo, arr[i].rho_hi = b["rho_lo"], b["rho_hi"]
            for k in range(MAX_ELEM):
                arr[i].w[k] = float(b["w"][k])
            arr[i].f_m, arr[i].x0_gcm2, arr[i].table_id = b["f_m"], b["x0_gcm2"], b["table_id"]
        self._chk(self.lib.pmc_set_hu_materials(self.ctx, arr, len(bins)))

    def load_ct(self, hu, vox, origin=(0.0, 0.0, 0.0)):
        """hu: CUDA int16 tensor (nz, ny, nx) — borrowed — or a host numpy array (copied by the library)."""
        org = (C.c_double * 3)(*origin)
        nz, ny, nx = hu.shape
        self.shape = (nz, ny, nx)
        args = (C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_double(vox[0]), C.c_double(vox[1]), C.c_double(vox[2]), org)
        if isinstance(hu, np.ndarray):
            h = np.ascontiguousarray(hu, dtype=np.int16)
            self._chk(self.lib.pmc_load_ct_host(self.ctx, h.ctypes.data_as(C.c_void_p), *args))
        else:
            assert hu.dtype == self.torch.int16
            self._keep["hu"] = hu
            self._chk(self.lib.pmc_load_ct(self.ctx, _ptr(hu), *args))

    def set_option(self, key, value):
        self._chk(self.lib.pmc_set_option(self.ctx, key.encode(), C.c_double(value)))

    def simulate(self, spots, n_histories, seed, out=None):
        """-> (dose, sigma): CUDA float32 tensors (nz, ny, nx), Gy per primary."""
        spots = np.ascontiguousarray(spots, dtype=np.float64)
        if out is None:
            out = (self.torch.empty(self.shape, dtype=self.torch.float32, device=self.device),
                   self.torch.empty(self.shape, dtype=self.torch.float32, device=self.device))
        self._chk(self.lib.pmc_simulate(self.ctx, spots.ctypes.data_as(C.c_void_p), C.c_int(spots.shape[0]),
                                        C.c_uint64(n_histories), C.c_uint64(seed), _ptr(out[0]), _ptr(out[1])))
        return out

    def simulate_host(self, spots, n_histories, seed, dose_host, sigma_host):
        """Host-buffer variant: dose_host/sigma_host are float32 numpy arrays (or pinned tensors' numpy views)."""
        spots = np.ascontiguousarray(spots, dtype=np.float64)
        self._chk(self.lib.pmc_simulate_host(self.ctx, spots.ctypes.data_as(C.c_void_p), C.c_int(spots.shape[0]),
                                             C.c_uint64(n_histories), C.c_uint64(seed),
                                             dose_host.ctypes.data_as(C.c_void_p), sigma_host.ctypes.data_as(C.c_void_p)))

    def set_dose_influence(self, roi_voxels, nspots):
        """Score D[spot][roi] (Gy per primary) in the following simulate() calls; returns the CUDA tensor (nspots, n_roi)
        the library writes into.  roi_voxels: linear voxel indices (x fastest); an empty list switches it off."""
        roi = np.ascontiguousarray(roi_voxels, dtype=np.int32)
        if roi.size == 0:
            self._chk(self.lib.pmc_set_dose_influence(self.ctx, None, C.c_int(0), None, C.c_uint64(0)))
            self._dij = None
            return None
        self._dij = self.torch.zeros((int(nspots), int(roi.size)), dtype=self.torch.float32, device=self.device)
        self._chk(self.lib.pmc_set_dose_influence(self.ctx, roi.ctypes.data_as(C.c_void_p), C.c_int(roi.size), _ptr(self._dij),
                                                  C.c_uint64(self._dij.numel())))
        return self._dij

    def letd(self, out=None):
        """-> LET_d map (keV/um), CUDA float32 tensor (nz, ny, nx), of the last simulate() with score_letd = 1."""
        if out is None:
            out = self.torch.empty(self.shape, dtype=self.torch.float32, device=self.device)
        self._chk(self.lib.pmc_get_letd(self.ctx, _ptr(out)))
        return out

    def gamma_index(self, ref, ev, vox, dd_frac=0.02, dta_cm=0.2, low_dose_frac=0.1, search_cm=0.0, out=None):
        """-> (gamma: CUDA float32 tensor like ref, -1 below the dose threshold; pass rate).  ref, ev: CUDA float32."""
        t = self.torch
        ref = ref.contiguous(); ev = ev.contiguous()
        if ref.dtype != t.float32 or ev.dtype != t.float32 or ref.shape != ev.shape or ref.dim() != 3:
            raise ValueError("ref and ev must be float32 CUDA tensors of the same (nz, ny, nx) shape")
        if out is None:
            out = t.empty_like(ref)
        nz, ny, nx = ref.shape
        rate = C.c_double(0.0)
        self._chk(self.lib.pmc_gamma_index(self.ctx, _ptr(ref), _ptr(ev), C.c_int(nx), C.c_int(ny), C.c_int(nz),
                                           C.c_double(vox[0]), C.c_double(vox[1]), C.c_double(vox[2]),
                                           C.c_double(dd_frac), C.c_double(dta_cm), C.c_double(low_dose_frac),
                                           C.c_double(search_cm), _ptr(out), C.byref(rate)))
        return out, rate.value

    def gamma_index_static(self, ref, ev, vox, dd_frac=0.02, dta_cm=0.2, low_dose_frac=0.1, search_cm=0.0, out=None):
        """gamma_index() for callers that may not allocate on the device (their framework's pool owns all of the GPU's
        memory, they have a latency budget that a cudaMalloc would break, or they allow no allocation once started):
        pmc_gamma_index_static keeps its working memory in a fixed array inside libpmc, so the call fails with
        PMC_E_CAPACITY when the search sphere holds more than 8192 voxel centres.  Same results as gamma_index().
        Pass `out` (and contiguous float32 inputs) if this wrapper is not to ask torch for memory either.  Every call
        shares that one array per GPU; the library serialises the calls.  Make the first call on a device outside any
        stream capture (it looks up the array's device address then)."""
        t = self.torch
        ref = ref.contiguous(); ev = ev.contiguous()
        if ref.dtype != t.float32 or ev.dtype != t.float32 or ref.shape != ev.shape or ref.dim() != 3:
            raise ValueError("ref and ev must be float32 CUDA tensors of the same (nz, ny, nx) shape")
        if out is None:
            out = t.empty_like(ref)
        nz, ny, nx = ref.shape
        rate = C.c_double(0.0)
        self._chk(self.lib.pmc_gamma_index_static(self.ctx, _ptr(ref), _ptr(ev), C.c_int(nx), C.c_int(ny), C.c_int(nz),
                                                  C.c_double(vox[0]), C.c_double(vox[1]), C.c_double(vox[2]),
                                                  C.c_double(dd_frac), C.c_double(dta_cm), C.c_double(low_dose_frac),
                                                  C.c_double(search_cm), _ptr(out), C.byref(rate)))
        return out, rate.value

    def nonelastic(self, Z, A, e_mev, n, seed, capacity=None):
        """-> (records: numpy structured array, offsets: numpy uint32 [n+1])."""
        t = self.torch
        capacity = capacity or 24 * n + 64
        out = t.zeros(capacity * 24, dtype=t.uint8, device=self.device)
        off = t.zeros(n + 1, dtype=t.int32, device=self.device)
        n_out = C.c_uint64()
        self._chk(self.lib.pmc_nonelastic(self.ctx, C.c_int(Z), C.c_int(A), C.c_double(e_mev), C.c_uint64(n),
                                          C.c_uint64(seed), _ptr(out), C.c_uint64(capacity), _ptr(off), C.byref(n_out)))
        rec = out[: n_out.value * 24].cpu().numpy().view(SECONDARY_DTYPE)
        return rec, off.cpu().numpy().view(np.uint32)

    def counters(self):
        c = Counters()
        self.lib.pmc_get_counters(self.ctx, C.byref(c))
        return {k: getattr(c, k) for k, _ in Counters._fields_}

    def timing(self):
        c = Timing()
        self.lib.pmc_get_timing(self.ctx, C.byref(c))
        return {k: getattr(c, k) for k, _ in Timing._fields_}

    # ---- sub-step entry points
    def philox4x32_10(self, ctr_key):
        t = self.torch
        a = t.as_tensor(np.ascontiguousarray(ctr_key, dtype=np.uint32).view(np.int32), device=self.device)
        out = t.empty((a.shape[0], 4), dtype=t.int32, device=self.device)
        self._chk(self.lib.pmc_philox4x32_10(self.ctx, _ptr(a), C.c_uint64(a.shape[0]), _ptr(out)))
        return out.cpu().numpy().view(np.uint32)

    def range_of_energy(self, table, e):
        t = self.torch
        a = t.as_tensor(np.ascontiguousarray(e, dtype=np.float32), device=self.device)
        out = t.empty_like(a)
        self._chk(self.lib.pmc_range_of_energy(self.ctx, C.c_int(table), _ptr(a), C.c_uint64(a.numel()), _ptr(out)))
        return out.cpu().numpy()

    def energy_of_range(self, table, r):
        t = self.torch
        a = t.as_tensor(np.ascontiguousarray(r, dtype=np.float32), device=self.device)
        out = t.empty_like(a)
        self._chk(self.lib.pmc_energy_of_range(self.ctx, C.c_int(table), _ptr(a), C.c_uint64(a.numel()), _ptr(out)))
        return out.cpu().numpy()

    def step_range_of_energy(self, hu_bin, e):
        """R(E) of HU bin hu_bin through the step kernel's shared-memory look-up (g/cm2 of the table medium)."""
        t = self.torch
        a = t.as_tensor(np.ascontiguousarray(e, dtype=np.float32), device=self.device)
        out = t.empty_like(a)
        self._chk(self.lib.pmc_step_range_of_energy(self.ctx, C.c_int(hu_bin), _ptr(a), C.c_uint64(a.numel()), _ptr(out)))
        return out.cpu().numpy()

    def step_energy_of_range(self, hu_bin, r):
        t = self.torch
        a = t.as_tensor(np.ascontiguousarray(r, dtype=np.float32), device=self.device)
        out = t.empty_like(a)
        self._chk(self.lib.pmc_step_energy_of_range(self.ctx, C.c_int(hu_bin), _ptr(a), C.c_uint64(a.numel()), _ptr(out)))
        return out.cpu().numpy()

    def straggle(self, e, mean_loss, rho_l, zoa, n, seed):
        t = self.torch
        out = t.empty(n, dtype=t.float32, device=self.device)
        self._chk(self.lib.pmc_straggle(self.ctx, C.c_double(e), C.c_double(mean_loss), C.c_double(rho_l), C.c_double(zoa),
                                        C.c_uint64(n), C.c_uint64(seed), _ptr(out)))
        return out.cpu().numpy()

    def elastic(self, Z, A, t_mev, n, seed):
        t = self.torch
        out = t.empty((n, 4), dtype=t.float32, device=self.device)
        self._chk(self.lib.pmc_elastic(self.ctx, C.c_int(Z), C.c_int(A), C.c_double(t_mev), C.c_uint64(n), C.c_uint64(seed),
                                       _ptr(out)))
        return out.cpu().numpy()

    def first_steps(self, spot, n, seed, max_steps):
        t = self.torch
        spot = np.ascontiguousarray(spot, dtype=np.float64)
        out = t.zeros((n, 8), dtype=t.float32, device=self.device)
        self._chk(self.lib.pmc_first_steps(self.ctx, spot.ctypes.data_as(C.c_void_p), C.c_uint64(n), C.c_uint64(seed),
                                           C.c_int(max_steps), _ptr(out)))
        return out.cpu().numpy()
