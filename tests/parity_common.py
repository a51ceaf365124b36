"""Helpers shared by the GPU parity tests: tolerances, the tie
protocol for event flags, host<->device shuttling."""
import numpy as np

LEPTON, PHOTON, F32, F64 = 0, 1, 0, 1
EPS = {np.dtype(np.float64): 2.0 ** -52, np.dtype(np.float32): 2.0 ** -23}
# north star: chi 1e-12 (fp64) / 1e-5 (fp32); optical depth and energies 1e-9 / 1e-5
TOL_CHI = {np.dtype(np.float64): 1e-12, np.dtype(np.float32): 1e-5}
TOL_TAU = {np.dtype(np.float64): 1e-9, np.dtype(np.float32): 1e-5}


def to_dev(arrs, device="cuda"):
    import torch
    return [torch.from_numpy(np.ascontiguousarray(a)).to(device) for a in arrs]


def to_host(tensors):
    return [t.detach().cpu().numpy() for t in tensors]


def code(np_dtype):
    return F64 if np.dtype(np_dtype) == np.float64 else F32


def uncancelled_scale(species, p, e, b):
    """g |e| + |p| |b|: the size of the terms of eq.2 before they cancel"""
    p64 = [np.asarray(a, np.float64) for a in p]
    pn = np.sqrt(sum(a * a for a in p64))
    g = np.sqrt(1 + pn * pn) if species == LEPTON else pn
    en = np.sqrt(sum(np.asarray(a, np.float64) ** 2 for a in e))
    bn = np.sqrt(sum(np.asarray(a, np.float64) ** 2 for a in b))
    return g * en + pn * bn


def assert_chi_close(chi_gpu, chi_orc, species, p, e, b):
    dt = np.dtype(chi_gpu.dtype)
    bound = TOL_CHI[dt] * chi_orc + 8 * EPS[dt] * uncancelled_scale(species, p, e, b)
    err = np.abs(chi_gpu.astype(np.float64) - chi_orc)
    bad = np.nonzero(~(err <= bound))[0]
    assert bad.size == 0, "chi mismatch at %s: gpu %s orc %s" % (bad[:5], chi_gpu[bad[:5]], chi_orc[bad[:5]])
    # how many needed the conditioning term at all
    return int(np.sum(err > TOL_CHI[dt] * chi_orc))


def tie_margin(arith_dtype, tau_old, o, ln_chi):
    """flags of particles with |tau_exact| <= margin are ambiguous (either value accepted):
    margin = eps (|tau_old| + d (16 + 4|L| + 4|slope| (1 + |ln chi|)))"""
    eps = EPS[np.dtype(arith_dtype)]
    lc = np.where(np.isfinite(ln_chi), np.abs(ln_chi), 0.0)
    return eps * (np.abs(tau_old) + o["decr"] * (16 + 4 * np.abs(o["lnval"]) + 4 * np.abs(o["slope"]) * (1 + lc)))


def check_evolve(tau_gpu, tau_old, o, arith_dtype, ln_chi):
    """tau within tolerance of the oracle's exact value; flags equal except ambiguous ones.
    Returns (n_ambiguous, flags_gpu)."""
    tau_gpu = tau_gpu.astype(np.float64)
    tol = max(TOL_TAU[np.dtype(arith_dtype)], 0)
    finite = np.isfinite(tau_old)
    ref = np.abs(tau_old[finite]) + o["decr"][finite]
    err = np.abs(tau_gpu[finite] - o["tau_exact"][finite])
    bad = np.nonzero(~(err <= tol * ref))[0]
    assert bad.size == 0, "tau mismatch (%d): idx %s err %s ref %s" % (bad.size, bad[:5], err[bad[:5]], ref[bad[:5]])
    assert np.all(tau_gpu[~finite] == tau_old[~finite])
    f_gpu, f_orc = tau_gpu < 0, o["tau"] < 0
    amb = np.abs(o["tau_exact"]) <= tie_margin(arith_dtype, tau_old, o, ln_chi)
    diff = (f_gpu != f_orc) & ~amb
    assert not diff.any(), "flag mismatch outside the tie margin at %s" % np.nonzero(diff)[0][:5]
    return int(np.sum(amb & (f_gpu != f_orc))), f_gpu


def rel_err(a, b):
    a = np.asarray(a, np.float64)
    b = np.asarray(b, np.float64)
    den = np.maximum(np.abs(b), 1e-300)
    return np.abs(a - b) / den
