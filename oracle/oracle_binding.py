"""ctypes binding of oracle/liboracle_hydro.so -- TEST INFRASTRUCTURE (see hydro_oracle.c).

All arrays are host numpy float64, C-contiguous, in the state layout a1 documented in
hydro_oracle.c.  This module defines its own parameter struct; it imports nothing from
the CUDA package.
"""
import ctypes as C

import numpy as np

from . import build_oracle


class OracleParams(C.Structure):
    _fields_ = [
        ("ndom", C.c_int32 * 3), ("nbox", C.c_int32 * 3), ("ng", C.c_int32), ("nspec", C.c_int32),
        ("bc_lo", C.c_int32 * 3), ("bc_hi", C.c_int32 * 3),
        ("prob_lo", C.c_double * 3), ("prob_hi", C.c_double * 3),
        ("gamma", C.c_double), ("cfl", C.c_double), ("grav", C.c_double * 3),
        ("small_dens", C.c_double), ("small_pres", C.c_double),
        ("flatten", C.c_int32), ("evolve_eint", C.c_int32),
    ]


def make_params(d: dict) -> OracleParams:
    """d: plain dict with the keys of OracleParams (as workloads.Workload.params)."""
    p = OracleParams()
    for k in ("ndom", "nbox", "bc_lo", "bc_hi"):
        setattr(p, k, (C.c_int32 * 3)(*[int(x) for x in d[k]]))
    for k in ("prob_lo", "prob_hi", "grav"):
        setattr(p, k, (C.c_double * 3)(*[float(x) for x in d[k]]))
    p.ng, p.nspec = int(d["ng"]), int(d["nspec"])
    p.gamma, p.cfl = float(d["gamma"]), float(d["cfl"])
    p.small_dens, p.small_pres = float(d.get("small_dens", 1e-12)), float(d.get("small_pres", 1e-14))
    p.flatten = int(d.get("flatten", 0))
    p.evolve_eint = int(d.get("evolve_eint", 0))
    return p


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build_oracle.build())
        dp = C.POINTER(C.c_double)
        pp = C.POINTER(OracleParams)
        L.oracle_state_doubles.restype = C.c_size_t
        L.oracle_state_doubles.argtypes = [pp]
        L.oracle_fill_ghosts.argtypes = [pp, dp]
        L.oracle_advance_stage.argtypes = [pp, C.c_int, C.c_double, dp, dp]
        L.oracle_estimate_dt.argtypes = [pp, dp, dp]
        L.oracle_conserved_totals.argtypes = [pp, dp, dp]
        L.oracle_step.argtypes = [pp, dp, dp, dp]
        L.oracle_step_fixed_dt.argtypes = [pp, dp, dp, C.c_double]
        L.oracle_cons_to_prim.restype = None
        L.oracle_cons_to_prim.argtypes = [C.c_double, C.c_double, C.c_double, C.c_int, dp, dp]
        L.oracle_ppm_line.restype = None
        L.oracle_ppm_line.argtypes = [dp, C.c_int, dp, dp, dp, dp]
        L.oracle_flatten_line.restype = None
        L.oracle_flatten_line.argtypes = [dp, dp, C.c_int, C.c_double, dp]
        L.oracle_hllc.restype = None
        L.oracle_hllc.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, C.c_int, dp, dp, dp]
        L.oracle_ctu_step.argtypes = [pp, dp, dp, dp]
        L.oracle_ctu_step_fixed_dt.argtypes = [pp, dp, dp, C.c_double]
        L.oracle_ctu_trace.restype = None
        L.oracle_ctu_trace.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, C.c_int, C.c_double, dp, dp, dp, dp, dp]
        L.oracle_fill_from_coarse.argtypes = [pp, dp, pp, dp, C.POINTER(C.c_int32), C.c_int]
        L.oracle_average_down.argtypes = [pp, dp, pp, dp, C.POINTER(C.c_int32), C.c_int]
        L.oracle_max_threads.restype = C.c_int
        L.oracle_set_threads.restype = None
        L.oracle_set_threads.argtypes = [C.c_int]
        _lib = L
    return _lib


def _ptr(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


def state_doubles(p):
    return lib().oracle_state_doubles(C.byref(p))


def fill_ghosts(p, U):
    _check(lib().oracle_fill_ghosts(C.byref(p), _ptr(U)), "fill_ghosts")


def advance_stage(p, stage, dt, U0, U1):
    _check(lib().oracle_advance_stage(C.byref(p), stage, dt, _ptr(U0), _ptr(U1)), "advance_stage")


def estimate_dt(p, U0):
    out = C.c_double(0.0)
    _check(lib().oracle_estimate_dt(C.byref(p), _ptr(U0), C.byref(out)), "estimate_dt")
    return out.value


def estimate_dt_rc(p, U0):
    out = C.c_double(0.0)
    return lib().oracle_estimate_dt(C.byref(p), _ptr(U0), C.byref(out)), out.value


def conserved_totals(p, U):
    out = np.zeros(5 + p.nspec)
    _check(lib().oracle_conserved_totals(C.byref(p), _ptr(U), _ptr(out)), "conserved_totals")
    return out


def step(p, U0, U1):
    out = C.c_double(0.0)
    _check(lib().oracle_step(C.byref(p), _ptr(U0), _ptr(U1), C.byref(out)), "step")
    return out.value


def step_fixed_dt(p, U0, U1, dt):
    _check(lib().oracle_step_fixed_dt(C.byref(p), _ptr(U0), _ptr(U1), dt), "step_fixed_dt")


def cons_to_prim(gamma, small_dens, small_pres, nspec, Uc):
    Uc = np.ascontiguousarray(Uc, dtype=np.float64)
    q = np.zeros(5 + nspec)
    lib().oracle_cons_to_prim(gamma, small_dens, small_pres, nspec, _ptr(Uc), _ptr(q))
    return q


def ppm_line(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    n = a.size
    s, e, aL, aR = (np.zeros(n) for _ in range(4))
    lib().oracle_ppm_line(_ptr(a), n, _ptr(s), _ptr(e), _ptr(aL), _ptr(aR))
    return s, e, aL, aR


def flatten_line(pr, un, small_pres=1e-14):
    pr = np.ascontiguousarray(pr, dtype=np.float64)
    un = np.ascontiguousarray(un, dtype=np.float64)
    flat = np.zeros(pr.size)
    lib().oracle_flatten_line(_ptr(pr), _ptr(un), pr.size, small_pres, _ptr(flat))
    return flat


def hllc(direction, gamma, qL, qR, small_dens=1e-12, small_pres=1e-14):
    qL = np.ascontiguousarray(qL, dtype=np.float64)
    qR = np.ascontiguousarray(qR, dtype=np.float64)
    nspec = qL.size - 5
    F = np.zeros(5 + nspec)
    lib().oracle_hllc(direction, gamma, small_dens, small_pres, nspec, _ptr(qL), _ptr(qR), _ptr(F))
    return F


def max_threads():
    return lib().oracle_max_threads()


def set_threads(n: int):
    lib().oracle_set_threads(int(n))


def ctu_step(p, U0, U1):
    """One CTU step (O12) of U0 in place; returns dt."""
    dt = C.c_double(0.0)
    _check(lib().oracle_ctu_step(C.byref(p), _ptr(U0), _ptr(U1), C.byref(dt)), "ctu_step")
    return dt.value


def ctu_step_fixed_dt(p, U0, U1, dt):
    _check(lib().oracle_ctu_step_fixed_dt(C.byref(p), _ptr(U0), _ptr(U1), dt), "ctu_step_fixed_dt")


def ctu_trace(d, gamma, small_dens, small_pres, dtdx, a, aL, aR):
    """Traced face states (qm, qp) of one zone (readings C2-C5)."""
    a, aL, aR = (np.ascontiguousarray(x, dtype=np.float64) for x in (a, aL, aR))
    qm, qp = np.zeros_like(a), np.zeros_like(a)
    lib().oracle_ctu_trace(d, gamma, small_dens, small_pres, a.size - 5, dtdx, _ptr(a), _ptr(aL), _ptr(aR), _ptr(qm), _ptr(qp))
    return qm, qp


def fill_from_coarse(pf, Uf, pc, Uc, lo, ratio):
    """O13: fine ghost zones across EXTERNAL faces from the coarse level (conservative linear interpolation)."""
    lo3 = (C.c_int32 * 3)(*[int(x) for x in lo])
    _check(lib().oracle_fill_from_coarse(C.byref(pf), _ptr(Uf), C.byref(pc), _ptr(Uc), lo3, int(ratio)), "fill_from_coarse")


def average_down(pc, Uc, pf, Uf, lo, ratio):
    """O13 restriction: coarse valid zones under the patch <- mean of their fine children."""
    lo3 = (C.c_int32 * 3)(*[int(x) for x in lo])
    _check(lib().oracle_average_down(C.byref(pc), _ptr(Uc), C.byref(pf), _ptr(Uf), lo3, int(ratio)), "average_down")
