"""Thin ctypes binding of include/picsarqed.h -- argument marshalling only.

Every step of the hot path runs in the CUDA kernels of ``libpicsarqed.so``; PyTorch is used
for device memory and streams.  There is no CPU fallback: if the library cannot be loaded
(or built with nvcc) the import of this module raises.
"""
import ctypes as C
from dataclasses import dataclass

import numpy as np
import torch

from .build import build

F32, F64 = 0, 1
LEPTON, PHOTON = 0, 1
UNITS_LIBRARY, UNITS_SI, UNITS_NORM_OMEGA, UNITS_NORM_LAMBDA, UNITS_HL_MEV = 0, 1, 2, 3, 4
TAB_LNG, TAB_QS_LNP, TAB_LNT, TAB_BW_P = 0, 1, 2, 3
NOALLOC_MAX_N = 1 << 24   # PICSARQED_NOALLOC_MAX_N

_vp, _u64, _i64, _i, _d = C.c_void_p, C.c_uint64, C.c_longlong, C.c_int, C.c_double


class _CSpecies(C.Structure):
    _fields_ = [("px", _vp), ("py", _vp), ("pz", _vp), ("tau", _vp), ("n", _i64), ("capacity", _i64),
                ("id_base", _u64)]


class _CParams(C.Structure):
    _fields_ = [("qs_chi_min", _d), ("qs_chi_max", _d), ("qs_n_chi", _i), ("qs_xi_min", _d),
                ("qs_n_xi", _i), ("bw_chi_min", _d), ("bw_chi_max", _d), ("bw_n_chi", _i),
                ("bw_n_xi", _i), ("qs_n_chi_2d", _i), ("bw_n_chi_2d", _i)]


@dataclass
class TableParams:
    """Table geometry; defaults are the paper's benchmark set."""
    qs_chi_min: float = 1e-3
    qs_chi_max: float = 1e3
    qs_n_chi: int = 256
    qs_xi_min: float = 1e-12
    qs_n_xi: int = 256
    bw_chi_min: float = 2e-2
    bw_chi_max: float = 1e3
    bw_n_chi: int = 256
    bw_n_xi: int = 256
    qs_n_chi_2d: int = 0      # rows of the 2D tables when they differ from the 1D counts (0 = the same grid)
    bw_n_chi_2d: int = 0

    def _c(self):
        return _CParams(self.qs_chi_min, self.qs_chi_max, self.qs_n_chi, self.qs_xi_min, self.qs_n_xi,
                        self.bw_chi_min, self.bw_chi_max, self.bw_n_chi, self.bw_n_xi, self.qs_n_chi_2d, self.bw_n_chi_2d)

    def rows_2d(self):
        return (self.qs_n_chi_2d or self.qs_n_chi, self.bw_n_chi_2d or self.bw_n_chi)

    def sizes(self):
        rq, rb = self.rows_2d()
        return (self.qs_n_chi, rq * self.qs_n_xi, self.bw_n_chi, rb * self.bw_n_xi)


_SIGNATURES = {
    "picsarqed_version": (_i, []),
    "picsarqed_create": (_i, [C.POINTER(_vp), _i, _vp]),
    "picsarqed_destroy": (_i, [_vp]),
    "picsarqed_last_error": (C.c_char_p, [_vp]),
    "picsarqed_set_option": (_i, [_vp, C.c_char_p, _i64]),
    "picsarqed_set_units": (_i, [_vp, _i, _d]),
    "picsarqed_get_unit_scales": (_i, [_vp, C.POINTER(_d)]),
    "picsarqed_get_timing": (_i, [_vp, C.POINTER(_d), C.POINTER(_i64)]),
    "picsarqed_build_tables": (_i, [_vp, C.POINTER(_CParams)]),
    "picsarqed_get_table_build_ms": (_i, [_vp, C.POINTER(_d)]),
    "picsarqed_set_chi_threshold": (_i, [_vp, _d]),
    "picsarqed_classical_loss": (_i, [_vp, _i, _i64] + [_vp] * 9 + [_d]),
    "picsarqed_export_tables": (_i, [_vp, _i, _vp, C.c_size_t]),
    "picsarqed_import_tables": (_i, [_vp, C.POINTER(_CParams), _vp, _vp, _vp, _vp]),
    "picsarqed_chi": (_i, [_vp, _i, _i, _i64] + [_vp] * 10),
    "picsarqed_schwinger_rate": (_i, [_vp, _i, _i64] + [_vp] * 7),
    "picsarqed_init_optical_depth": (_i, [_vp, _i, _i, _i64, _u64, _u64, _vp]),
    "picsarqed_evolve_optical_depth": (_i, [_vp, _i, _i, _i, _i64] + [_vp] * 9 + [_d, _vp, _vp]),
    "picsarqed_generate_photons": (_i, [_vp, _i, _i, _i64] + [_vp] * 10 + [_u64, _u64, _u64, _i64] + [_vp] * 6),
    "picsarqed_generate_photons_noalloc": (_i, [_vp, _i, _i, _i64] + [_vp] * 10 + [_u64, _u64, _u64, _i64] + [_vp] * 6),
    "picsarqed_generate_pairs": (_i, [_vp, _i, _i, _i64] + [_vp] * 10 + [_u64, _u64, _u64, _i64] + [_vp] * 10),
    "picsarqed_qed_step": (_i, [_vp, _i, _i, _i, _i64] + [_vp] * 10 + [_d, _u64, _u64, _u64, _i64] + [_vp] * 10),
    "picsarqed_read_count": (_i, [_vp, _vp, C.POINTER(_u64)]),
    "picsarqed_step_host": (_i, [_vp, _i, _i, _i, _i64] + [_vp] * 10 + [_d, _u64, _u64, _u64, _i64, _vp, _vp,
                                                                     C.POINTER(_u64)]),
    "picsarqed_boris_push_uniform": (_i, [_vp, _i, _i64, _vp, _vp, _vp, _i, C.POINTER(_d), C.POINTER(_d), _d]),
    "picsarqed_append_secondaries": (_i, [_vp, _i, _i, _i64] + [_vp] * 5 + [_d] + [_vp] * 4 + [_i64, _i64, _vp]),
    "picsarqed_energy_spectrum": (_i, [_vp, _i, _i, _i64, _vp, _vp, _vp, _d, _d, _i, _vp]),
    "picsarqed_table_function": (_i, [_vp, _i, _i, _i64, _vp, _vp]),
    "picsarqed_sample_xi": (_i, [_vp, _i, _i, _i64, _vp, _vp, _vp]),
    "picsarqed_cascade_step": (_i, [_vp, _i, _i, C.POINTER(_CSpecies), C.POINTER(_CSpecies), C.POINTER(_CSpecies),
                                    C.POINTER(_d), C.POINTER(_d), _d, _u64, _u64, _d, _i, C.POINTER(_u64)]),
}

_lib = None


def lib():
    """The loaded C-ABI library (built with nvcc on first use)."""
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        for name, (res, args) in _SIGNATURES.items():
            f = getattr(L, name)
            f.restype = res
            f.argtypes = args
        _lib = L
    return _lib


class PicsarQedError(RuntimeError):
    pass


_TORCH_DTYPE = {F32: torch.float32, F64: torch.float64}


def _code(dtype):
    return F64 if dtype == torch.float64 else F32


def _dev(t, dtype=None):
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous()):
        raise PicsarQedError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise PicsarQedError("dtype mismatch: %s vs %s" % (t.dtype, dtype))
    return t.data_ptr()


class Context:
    """One library context bound to a device and a stream (picsarqed_create)."""

    def __init__(self, device=0, stream=None):
        self._h = _vp()
        self.device = torch.device("cuda", device) if isinstance(device, int) else torch.device(device)
        if not torch.cuda.is_available():
            raise PicsarQedError("no CUDA device: picsarqed has no CPU fallback")
        idx = self.device.index or 0
        with torch.cuda.device(idx):
            self.stream = stream if stream is not None else torch.cuda.current_stream()
            rc = lib().picsarqed_create(C.byref(self._h), idx, _vp(self.stream.cuda_stream))
        if rc != 0:
            raise PicsarQedError("picsarqed_create failed with status %d (needs an sm_100 device)" % rc)
        self.params = None

    def close(self):
        if self._h:
            lib().picsarqed_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != 0:
            msg = lib().picsarqed_last_error(self._h)
            raise PicsarQedError("status %d: %s" % (rc, msg.decode() if msg else ""))

    # ---- options / tables ---------------------------------------------------------------
    def set_option(self, name, value):
        self._check(lib().picsarqed_set_option(self._h, name.encode(), int(value)))

    def get_timing(self):
        """(evolve-pass ms, event-pass ms, calls) accumulated by qed_step since the last call ("time_kernels" = 1)"""
        ms = (_d * 2)()
        calls = _i64(0)
        self._check(lib().picsarqed_get_timing(self._h, ms, C.byref(calls)))
        return float(ms[0]), float(ms[1]), int(calls.value)

    def build_tables(self, params):
        cp = params._c()
        self._check(lib().picsarqed_build_tables(self._h, C.byref(cp)))
        self.params = params

    def table_build_ms(self):
        """device time of the quadrature kernels of the last build_tables, in milliseconds"""
        ms = _d(0.0)
        self._check(lib().picsarqed_get_table_build_ms(self._h, C.byref(ms)))
        return ms.value

    def import_tables(self, params, lnG, qs_lnP, lnT, bw_P):
        arrs = [np.ascontiguousarray(a, dtype=np.float64).ravel() for a in (lnG, qs_lnP, lnT, bw_P)]
        for a, n in zip(arrs, params.sizes()):
            if a.size != n:
                raise PicsarQedError("table size mismatch")
        cp = params._c()
        self._check(lib().picsarqed_import_tables(self._h, C.byref(cp), *[a.ctypes.data for a in arrs]))
        self.params = params

    def export_tables(self, which):
        n = self.params.sizes()[which]
        out = np.empty(n, dtype=np.float64)
        self._check(lib().picsarqed_export_tables(self._h, which, out.ctypes.data, n))
        p = self.params
        if which == TAB_QS_LNP:
            return out.reshape(p.rows_2d()[0], p.qs_n_xi)
        if which == TAB_BW_P:
            return out.reshape(p.rows_2d()[1], p.bw_n_xi)
        return out

    # ---- runtime calls (device tensors) ---------------------------------------------------
    def chi(self, species, p, e, b, out=None):
        dt = p[0].dtype
        n = p[0].numel()
        if out is None:
            out = torch.empty(n, dtype=dt, device=p[0].device)
        ptrs = [_dev(t, dt) for t in (*p, *e, *b, out)]
        self._check(lib().picsarqed_chi(self._h, species, _code(dt), n, *ptrs))
        return out

    def schwinger_rate(self, e, b, out=None):
        """pairs per m^3 per s (fp64) for fields in units of E_s (picsarqed_schwinger_rate)"""
        d = e[0].dtype
        n = e[0].numel()
        if out is None:
            out = torch.empty(n, dtype=torch.float64, device=e[0].device)
        self._check(lib().picsarqed_schwinger_rate(self._h, _code(d), n, *[_dev(t, d) for t in (*e, *b)],
                                                   _dev(out, torch.float64)))
        return out

    def init_optical_depth(self, species, tau, seed, id_base=0):
        self._check(lib().picsarqed_init_optical_depth(self._h, species, _code(tau.dtype), tau.numel(), seed,
                                                       id_base, _dev(tau)))
        return tau

    def evolve_optical_depth(self, species, p, e, b, dt, tau, n_events=None):
        d = p[0].dtype
        ptrs = [_dev(t, d) for t in (*p, *e, *b)]
        self._check(lib().picsarqed_evolve_optical_depth(self._h, species, _code(d), _code(tau.dtype), tau.numel(),
                                                         *ptrs, float(dt), _dev(tau),
                                                         _dev(n_events, torch.int64) if n_events is not None else None))

    def generate_photons(self, p, e, b, tau, seed, step, id_base, capacity, ph_p, ph_tau, ph_parent, n_out):
        d = p[0].dtype
        ptrs = [_dev(t, d) for t in (*p, *e, *b)]
        self._check(lib().picsarqed_generate_photons(
            self._h, _code(d), _code(tau.dtype), tau.numel(), *ptrs, _dev(tau), seed, step, id_base, capacity,
            *[_dev(t, d) for t in ph_p], _dev(ph_tau, tau.dtype),
            _dev(ph_parent, torch.int64) if ph_parent is not None else None, _dev(n_out, torch.int64)))

    def generate_photons_noalloc(self, p, e, b, tau, seed, step, id_base, capacity, ph_p, ph_tau, ph_parent, n_out):
        """generate_photons on the library's static scratch: allocates nothing, n <= NOALLOC_MAX_N"""
        d = p[0].dtype
        ptrs = [_dev(t, d) for t in (*p, *e, *b)]
        self._check(lib().picsarqed_generate_photons_noalloc(
            self._h, _code(d), _code(tau.dtype), tau.numel(), *ptrs, _dev(tau), seed, step, id_base, capacity,
            *[_dev(t, d) for t in ph_p], _dev(ph_tau, tau.dtype),
            _dev(ph_parent, torch.int64) if ph_parent is not None else None, _dev(n_out, torch.int64)))

    def generate_pairs(self, p, e, b, tau, seed, step, id_base, capacity, el_p, el_tau, po_p, po_tau, parent, n_out):
        d = p[0].dtype
        ptrs = [_dev(t, d) for t in (*p, *e, *b)]
        self._check(lib().picsarqed_generate_pairs(
            self._h, _code(d), _code(tau.dtype), tau.numel(), *ptrs, _dev(tau), seed, step, id_base, capacity,
            *[_dev(t, d) for t in el_p], _dev(el_tau, tau.dtype), *[_dev(t, d) for t in po_p],
            _dev(po_tau, tau.dtype), _dev(parent, torch.int64) if parent is not None else None,
            _dev(n_out, torch.int64)))

    def qed_step(self, species, p, e, b, tau, dt, seed, step, id_base, capacity, s1_p, s1_tau, s2_p=None,
                 s2_tau=None, parent=None, n_out=None):
        """evolve + event generation in one kernel (picsarqed_qed_step); s1 = photon (leptons) or electron
        (photons) buffers, s2 = positron buffers"""
        d = p[0].dtype
        ptrs = [_dev(t, d) for t in (*p, *e, *b)]
        s2 = [_dev(t, d) for t in s2_p] if s2_p is not None else [None] * 3
        self._check(lib().picsarqed_qed_step(
            self._h, species, _code(d), _code(tau.dtype), tau.numel(), *ptrs, _dev(tau), float(dt), seed, step,
            id_base, capacity, *[_dev(t, d) for t in s1_p], _dev(s1_tau, tau.dtype), *s2,
            _dev(s2_tau, tau.dtype) if s2_tau is not None else None,
            _dev(parent, torch.int64) if parent is not None else None, _dev(n_out, torch.int64)))

    def read_count(self, counter):
        v = _u64(0)
        self._check(lib().picsarqed_read_count(self._h, _dev(counter, torch.int64), C.byref(v)))
        return int(v.value)

    # ---- host-buffer path -----------------------------------------------------------------
    def step_host(self, species, p, e, b, tau, dt, seed, step, id_base, capacity, sec, parent=None):
        """One QED step on HOST tensors (CPU, ideally pinned); p, tau and sec are overwritten.
        Returns the total number of fired parents."""
        for t in (*p, *e, *b, tau, *sec):
            if t.is_cuda or not t.is_contiguous():
                raise PicsarQedError("step_host expects contiguous CPU tensors")
        d = p[0].dtype
        n_out = _u64(0)
        sec_ptrs = (_vp * len(sec))(*[t.data_ptr() for t in sec])
        self._check(lib().picsarqed_step_host(
            self._h, species, _code(d), _code(tau.dtype), tau.numel(), *[t.data_ptr() for t in (*p, *e, *b)],
            tau.data_ptr(), float(dt), seed, step, id_base, capacity, C.cast(sec_ptrs, _vp),
            parent.data_ptr() if parent is not None else None, C.byref(n_out)))
        return int(n_out.value)

    # ---- unit systems ---------------------------------------------------------
    def set_units(self, system, reference=0.0):
        self._check(lib().picsarqed_set_units(self._h, system, float(reference)))

    def unit_scales(self):
        """multipliers (p, E, B, t) from the caller's unit system to the library's"""
        v = (_d * 4)()
        self._check(lib().picsarqed_get_unit_scales(self._h, v))
        return tuple(v)

    # ---- table functions per value -----------------------------------------
    def table_function(self, kind, chi, out):
        """out = G(chi) (kind LEPTON) or T(chi) (kind PHOTON) as the evolve pass evaluates them"""
        self._check(lib().picsarqed_table_function(self._h, kind, _code(chi.dtype), chi.numel(), _dev(chi),
                                                   _dev(out, chi.dtype)))

    def sample_xi(self, kind, chi, r, xi):
        self._check(lib().picsarqed_sample_xi(self._h, kind, _code(chi.dtype), chi.numel(), _dev(chi),
                                              _dev(r, chi.dtype), _dev(xi, chi.dtype)))

    # ---- closed loop in a uniform field ------------------------------
    def set_chi_threshold(self, chi_min):
        """no event of either kind below chi_min (0 = off)"""
        self._check(lib().picsarqed_set_chi_threshold(self._h, float(chi_min)))

    def classical_loss(self, p, e, b, dt):
        """one step of the classical radiation reaction for the leptons below the chi threshold (momenta in place)"""
        d = p[0].dtype
        self._check(lib().picsarqed_classical_loss(self._h, _code(d), p[0].numel(), *[_dev(t, d) for t in (*p, *e, *b)],
                                                   float(dt)))

    def boris_push_uniform(self, p, charge_sign, e, b, dt):
        d = p[0].dtype
        self._check(lib().picsarqed_boris_push_uniform(
            self._h, _code(d), p[0].numel(), *[_dev(t, d) for t in p], int(charge_sign), (_d * 3)(*e), (_d * 3)(*b),
            float(dt)))

    def append_secondaries(self, m_max, src_p, src_tau, count, min_energy, dst_p, dst_tau, dst_n, new_n):
        """ordered, filtering append of the first min(count, m_max) source entries to dst[dst_n:]"""
        d = src_p[0].dtype
        self._check(lib().picsarqed_append_secondaries(
            self._h, _code(d), _code(src_tau.dtype), m_max, *[_dev(t, d) for t in src_p], _dev(src_tau),
            _dev(count, torch.int64), float(min_energy), *[_dev(t, d) for t in dst_p], _dev(dst_tau, src_tau.dtype),
            dst_n, dst_tau.numel(), _dev(new_n, torch.int64)))

    def energy_spectrum(self, species, p, e_min, e_max, hist):
        d = p[0].dtype
        self._check(lib().picsarqed_energy_spectrum(
            self._h, species, _code(d), p[0].numel(), *[_dev(t, d) for t in p], float(e_min), float(e_max),
            hist.numel(), _dev(hist, torch.int64)))

    def cascade_step(self, pops, e, b, dt, seed, step, photon_min_energy=0.0, push=True):
        """one time step of the closed loop; pops: dict electrons / positrons / photons -> Species.
        Returns the event counts (electrons, positrons, photons)."""
        cs = {k: pops[k]._c() for k in ("electrons", "positrons", "photons")}
        d, td = pops["electrons"].p[0].dtype, pops["electrons"].tau.dtype
        ev = (_u64 * 3)()
        rc = lib().picsarqed_cascade_step(
            self._h, _code(d), _code(td), C.byref(cs["electrons"]), C.byref(cs["positrons"]), C.byref(cs["photons"]),
            (_d * 3)(*e), (_d * 3)(*b), float(dt), seed, step, float(photon_min_energy), int(bool(push)), ev)
        for k in cs:
            pops[k].n = int(cs[k].n)
        self._check(rc)
        return tuple(int(v) for v in ev)


class Species:
    """device structure of arrays with room for `capacity` entries, the first n in use (picsarqed_species_arrays)"""

    def __init__(self, capacity, dtype, tau_dtype, id_base, device="cuda"):
        self.p = [torch.zeros(capacity, dtype=dtype, device=device) for _ in range(3)]
        self.tau = torch.zeros(capacity, dtype=tau_dtype, device=device)
        self.n = 0
        self.capacity = capacity
        self.id_base = id_base

    def _c(self):
        return _CSpecies(self.p[0].data_ptr(), self.p[1].data_ptr(), self.p[2].data_ptr(), self.tau.data_ptr(), self.n,
                         self.capacity, self.id_base)
