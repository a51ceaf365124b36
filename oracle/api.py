"""numpy/ctypes wrappers around libpicsarqed_oracle.so.  Test infrastructure only.

Argument marshalling only: every number is computed by ``picsarqed_oracle.cpp``.
"""
import ctypes as C
from dataclasses import dataclass

import numpy as np

from .build import build

__all__ = [
    "lib", "num_threads", "TableParams", "Tables", "build_tables", "build_bw_rows", "build_qs_rows",
    "bessel_k_scaled", "bessel_ik_scaled", "bw_lnT", "bw_T_scaled", "bw_cdf", "bw_f_scaled",
    "qs_G", "qs_cdf", "qs_s_over_xi", "qs_first_moment", "erber_T", "schwinger_field",
    "rate_prefactor", "selftest_gk15", "philox4x32_10", "uniform", "chi", "init_optical_depth",
    "rate", "evolve_optical_depth", "generate_photons", "generate_pairs", "qs_sample_xi",
    "bw_sample_xi", "LEPTON", "PHOTON", "F32", "F64",
]

LEPTON, PHOTON = 0, 1
F32, F64 = 0, 1

_lib = None
_dp = C.POINTER(C.c_double)
_u64p = C.POINTER(C.c_uint64)
_i64p = C.POINTER(C.c_int64)
_u32p = C.POINTER(C.c_uint32)


class _CTables(C.Structure):
    _fields_ = [
        ("qs_chi_min", C.c_double), ("qs_chi_max", C.c_double), ("qs_n_chi", C.c_int),
        ("qs_xi_min", C.c_double), ("qs_n_xi", C.c_int),
        ("bw_chi_min", C.c_double), ("bw_chi_max", C.c_double), ("bw_n_chi", C.c_int),
        ("bw_n_xi", C.c_int),
        ("lnG", _dp), ("qs_lnP", _dp), ("lnT", _dp), ("bw_P", _dp),
        ("read_fp32", C.c_int),
        ("qs_n_chi_2d", C.c_int), ("bw_n_chi_2d", C.c_int),   # rows of the 2D tables (0: as the 1D tables)
        ("chi_event_min", C.c_double),                        # no event below this chi (0: off)
    ]


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        d, i, i64, u64 = C.c_double, C.c_int, C.c_int64, C.c_uint64
        tp = C.POINTER(_CTables)

        def sig(name, res, *args):
            f = getattr(L, name)
            f.restype = res
            f.argtypes = list(args)

        sig("orc_num_threads", i)
        sig("orc_selftest_gk15", d)
        sig("orc_schwinger_field", d)
        sig("orc_rate_prefactor", d)
        for n in ("orc_bessel_k_scaled", "orc_bessel_ik_scaled", "orc_bw_f_scaled", "orc_bw_cdf",
                  "orc_qs_s_over_xi", "orc_qs_cdf"):
            sig(n, d, d, d)
        for n in ("orc_bw_lnT", "orc_bw_T_scaled", "orc_qs_G", "orc_qs_first_moment", "orc_erber_T"):
            sig(n, d, d)
        sig("orc_build_lnT", None, d, d, i, _dp)
        sig("orc_build_lnG", None, d, d, i, _dp)
        sig("orc_build_bw_cdf_rows", None, d, d, i, i, i, i, _dp, _dp)
        sig("orc_build_qs_cdf_rows", None, d, d, i, d, i, i, i, _dp, _dp)
        sig("orc_philox4x32_10", None, _u32p, _u32p, _u32p)
        sig("orc_uniform", d, u64, u64, u64, i, i, i, i)
        sig("orc_chi", None, i, i64, *([_dp] * 10))
        sig("orc_init_optical_depth", None, i, i, i64, u64, _u64p, _dp)
        sig("orc_rate", None, tp, i, i64, *([_dp] * 10))
        sig("orc_evolve_optical_depth", None, tp, i, i, i64, *([_dp] * 9), d, *([_dp] * 6))
        sig("orc_generate_photons", i64, tp, i, i, i64, *([_dp] * 10), u64, u64, _u64p, i64,
            _dp, _dp, _dp, _dp, _i64p, _dp)
        sig("orc_generate_pairs", i64, tp, i, i, i64, *([_dp] * 10), u64, u64, _u64p, i64,
            *([_dp] * 8), _i64p, _dp)
        sig("orc_classical_loss", None, i, i64, *([_dp] * 9), d, d)
        sig("orc_schwinger_prefactor", d)
        sig("orc_schwinger_rate", None, i64, *([_dp] * 7))
        sig("orc_qs_sample_xi", d, tp, d, d)
        sig("orc_bw_sample_xi", d, tp, d, d)
        _lib = L
    return _lib


def num_threads():
    return lib().orc_num_threads()


def _f64(a):
    """contiguous float64 copy/view (fp32 -> fp64 widening is exact)"""
    return np.ascontiguousarray(np.asarray(a), dtype=np.float64)


def _p(a):
    return a.ctypes.data_as(_dp)


# ------------------------------------------------------------------ definitions (pins)
def selftest_gk15():
    return lib().orc_selftest_gk15()


def schwinger_field():
    return lib().orc_schwinger_field()


def rate_prefactor():
    return lib().orc_rate_prefactor()


def bessel_k_scaled(nu, x):
    return lib().orc_bessel_k_scaled(nu, x)


def bessel_ik_scaled(nu, x):
    return lib().orc_bessel_ik_scaled(nu, x)


def bw_f_scaled(chi, xi):
    return lib().orc_bw_f_scaled(chi, xi)


def bw_lnT(chi):
    return lib().orc_bw_lnT(chi)


def bw_T_scaled(chi):
    return lib().orc_bw_T_scaled(chi)


def bw_cdf(chi, xi):
    return lib().orc_bw_cdf(chi, xi)


def qs_s_over_xi(chi, xi):
    return lib().orc_qs_s_over_xi(chi, xi)


def qs_G(chi):
    return lib().orc_qs_G(chi)


def qs_cdf(chi, xi):
    return lib().orc_qs_cdf(chi, xi)


def qs_first_moment(chi):
    return lib().orc_qs_first_moment(chi)


def erber_T(chi):
    return lib().orc_erber_T(chi)


# ------------------------------------------------------------------ tables
@dataclass
class TableParams:
    qs_chi_min: float = 1e-3
    qs_chi_max: float = 1e3
    qs_n_chi: int = 256
    qs_xi_min: float = 1e-12
    qs_n_xi: int = 256
    bw_chi_min: float = 2e-2
    bw_chi_max: float = 1e3
    bw_n_chi: int = 256
    bw_n_xi: int = 256
    qs_n_chi_2d: int = 0   # rows of the 2D tables when they are on a grid of their own (0: the grid of the 1D table)
    bw_n_chi_2d: int = 0

    def rows_2d(self):
        return (self.qs_n_chi_2d or self.qs_n_chi, self.bw_n_chi_2d or self.bw_n_chi)


class Tables:
    """Table bytes as the runtime half sees them (always fp64 on the wire)."""

    def __init__(self, params, lnG, qs_lnP, lnT, bw_P, read_fp32=False):
        self.params = params
        self.lnG = _f64(lnG)
        self.qs_lnP = _f64(qs_lnP).reshape(params.rows_2d()[0], params.qs_n_xi)
        self.lnT = _f64(lnT)
        self.bw_P = _f64(bw_P).reshape(params.rows_2d()[1], params.bw_n_xi)
        assert self.lnG.shape == (params.qs_n_chi,) and self.lnT.shape == (params.bw_n_chi,)
        self.read_fp32 = bool(read_fp32)
        self.chi_event_min = 0.0

    def with_fp32_reads(self, flag=True):
        t = Tables(self.params, self.lnG, self.qs_lnP, self.lnT, self.bw_P, flag)
        t.chi_event_min = self.chi_event_min
        return t

    def with_chi_event_min(self, chi_min):
        """below chi_min neither process is an event (rate := 0)"""
        t = Tables(self.params, self.lnG, self.qs_lnP, self.lnT, self.bw_P, self.read_fp32)
        t.chi_event_min = float(chi_min)
        return t

    def _c(self):
        p = self.params
        return _CTables(p.qs_chi_min, p.qs_chi_max, p.qs_n_chi, p.qs_xi_min, p.qs_n_xi,
                        p.bw_chi_min, p.bw_chi_max, p.bw_n_chi, p.bw_n_xi,
                        _p(self.lnG), _p(self.qs_lnP), _p(self.lnT), _p(self.bw_P),
                        int(self.read_fp32), p.qs_n_chi_2d, p.bw_n_chi_2d, float(self.chi_event_min))


def build_bw_rows(p, row0, row1, return_half=False):
    out = np.empty((row1 - row0, p.bw_n_xi))
    half = np.empty(row1 - row0)
    lib().orc_build_bw_cdf_rows(p.bw_chi_min, p.bw_chi_max, p.rows_2d()[1], p.bw_n_xi, row0, row1,
                                _p(out), _p(half))
    return (out, half) if return_half else out


def build_qs_rows(p, row0, row1, return_total=False):
    out = np.empty((row1 - row0, p.qs_n_xi))
    tot = np.empty(row1 - row0)
    lib().orc_build_qs_cdf_rows(p.qs_chi_min, p.qs_chi_max, p.rows_2d()[0], p.qs_xi_min, p.qs_n_xi,
                                row0, row1, _p(out), _p(tot))
    return (out, tot) if return_total else out


def build_lnT(p):
    out = np.empty(p.bw_n_chi)
    lib().orc_build_lnT(p.bw_chi_min, p.bw_chi_max, p.bw_n_chi, _p(out))
    return out


def build_lnG(p):
    out = np.empty(p.qs_n_chi)
    lib().orc_build_lnG(p.qs_chi_min, p.qs_chi_max, p.qs_n_chi, _p(out))
    return out


def build_tables(p):
    return Tables(p, build_lnG(p), build_qs_rows(p, 0, p.rows_2d()[0]), build_lnT(p),
                  build_bw_rows(p, 0, p.rows_2d()[1]))


__all__ += ["build_lnT", "build_lnG"]


# ------------------------------------------------------------------ runtime half
def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return tuple(int(v) for v in o)


def uniform(seed, pid, step, purpose, species, pair, dtype):
    return lib().orc_uniform(seed, pid, step, purpose, species, pair, dtype)


def _ids(ids, n):
    if ids is None:
        ids = np.arange(n, dtype=np.uint64)
    ids = np.ascontiguousarray(ids, dtype=np.uint64)
    assert ids.shape == (n,)
    return ids


def chi(species, p, e, b):
    arrs = [_f64(a) for a in (*p, *e, *b)]
    n = arrs[0].size
    out = np.empty(n)
    lib().orc_chi(species, n, *[_p(a) for a in arrs], _p(out))
    return out


def init_optical_depth(species, tau_dtype, n, seed, ids=None):
    ids = _ids(ids, n)
    out = np.empty(n)
    lib().orc_init_optical_depth(species, tau_dtype, n, seed, ids.ctypes.data_as(_u64p), _p(out))
    return out


def rate(tables, species, p, e, b):
    arrs = [_f64(a) for a in (*p, *e, *b)]
    n = arrs[0].size
    out = np.empty(n)
    ct = tables._c()
    lib().orc_rate(C.byref(ct), species, n, *[_p(a) for a in arrs], _p(out))
    return out


def evolve_optical_depth(tables, species, tau_dtype, p, e, b, dt, tau):
    """returns dict(tau, tau_exact, decr, lnval, slope)"""
    arrs = [_f64(a) for a in (*p, *e, *b)]
    tau = _f64(tau)
    n = tau.size
    o = {k: np.empty(n) for k in ("tau", "tau_exact", "decr", "lnval", "slope")}
    ct = tables._c()
    lib().orc_evolve_optical_depth(C.byref(ct), species, tau_dtype, n, *[_p(a) for a in arrs],
                                   float(dt), _p(tau), _p(o["tau"]), _p(o["tau_exact"]),
                                   _p(o["decr"]), _p(o["lnval"]), _p(o["slope"]))
    return o


def generate_photons(tables, dtype, tau_dtype, p, e, b, tau, seed, step, ids=None, capacity=None):
    """returns dict: p (3 arrays, updated), tau (updated), n_fired, ph_p, ph_tau, parent, xi"""
    pp = [_f64(a).copy() for a in p]
    ff = [_f64(a) for a in (*e, *b)]
    tau = _f64(tau).copy()
    n = tau.size
    ids = _ids(ids, n)
    cap = n if capacity is None else int(capacity)
    ph = [np.zeros(cap) for _ in range(4)]
    parent = np.full(cap, -1, dtype=np.int64)
    xi = np.zeros(cap)
    ct = tables._c()
    nf = lib().orc_generate_photons(C.byref(ct), dtype, tau_dtype, n, *[_p(a) for a in pp],
                                    *[_p(a) for a in ff], _p(tau), seed, step,
                                    ids.ctypes.data_as(_u64p), cap, *[_p(a) for a in ph],
                                    parent.ctypes.data_as(_i64p), _p(xi))
    k = min(nf, cap)
    return dict(p=pp, tau=tau, n_fired=int(nf), ph_p=[a[:k] for a in ph[:3]], ph_tau=ph[3][:k],
                parent=parent[:k], xi=xi[:k])


def generate_pairs(tables, dtype, tau_dtype, p, e, b, tau, seed, step, ids=None, capacity=None):
    """returns dict: p, tau (updated), n_fired, el_p, el_tau, po_p, po_tau, parent, xi_el"""
    pp = [_f64(a).copy() for a in p]
    ff = [_f64(a) for a in (*e, *b)]
    tau = _f64(tau).copy()
    n = tau.size
    ids = _ids(ids, n)
    cap = n if capacity is None else int(capacity)
    out = [np.zeros(cap) for _ in range(8)]
    parent = np.full(cap, -1, dtype=np.int64)
    xi = np.zeros(cap)
    ct = tables._c()
    nf = lib().orc_generate_pairs(C.byref(ct), dtype, tau_dtype, n, *[_p(a) for a in pp],
                                  *[_p(a) for a in ff], _p(tau), seed, step,
                                  ids.ctypes.data_as(_u64p), cap, *[_p(a) for a in out],
                                  parent.ctypes.data_as(_i64p), _p(xi))
    k = min(nf, cap)
    return dict(p=pp, tau=tau, n_fired=int(nf), el_p=[a[:k] for a in out[0:3]], el_tau=out[3][:k],
                po_p=[a[:k] for a in out[4:7]], po_tau=out[7][:k], parent=parent[:k], xi_el=xi[:k])


def classical_loss(dtype, p, e, b, dt, chi_min):
    """PAPER.md:340 / DESIGN.md R24: leptons with chi < chi_min lose (2/3)(alpha/tau_C) chi^2 (gamma-1)/gamma dt of kinetic
    energy; returns the three momentum arrays after the step"""
    pp = [_f64(a).copy() for a in p]
    ff = [_f64(a) for a in (*e, *b)]
    lib().orc_classical_loss(dtype, pp[0].size, *[_p(a) for a in pp], *[_p(a) for a in ff], float(dt), float(chi_min))
    return pp


def qs_sample_xi(tables, chi_v, r):
    ct = tables._c()
    return lib().orc_qs_sample_xi(C.byref(ct), chi_v, r)


def bw_sample_xi(tables, chi_v, rp):
    ct = tables._c()
    return lib().orc_bw_sample_xi(C.byref(ct), chi_v, rp)


def schwinger_prefactor():
    return lib().orc_schwinger_prefactor()


def schwinger_rate(e, b):
    """pairs per m^3 per s (eq.19) for fields in units of E_s"""
    arrs = [_f64(a) for a in (*e, *b)]
    n = arrs[0].size
    out = np.empty(n)
    lib().orc_schwinger_rate(n, *[_p(a) for a in arrs], _p(out))
    return out


__all__ += ["schwinger_prefactor", "schwinger_rate", "classical_loss"]
