"""ctypes wrapper around oracle/libia_oracle.so (the C++ CPU oracle, ia_oracle.cpp).

TEST INFRASTRUCTURE ONLY: importable from tests/, ``__graft_entry__.smoke()`` and bench.py's
``cpu_baseline`` / ``--impl reference`` legs.  Argument marshalling only -- every number comes out
of the C++ code.  Builds the library with g++ on first use if it is missing or stale.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "ia_oracle.cpp"
_HDR = _HERE / "ia_oracle.h"
_LIB = _HERE / "libia_oracle.so"

CXXFLAGS = ["-std=c++17", "-O2", "-ffp-contract=off", "-Wall", "-Wextra", "-shared", "-fPIC", "-pthread"]


def build(force: bool = False) -> Path:
    """Compile the oracle (plain g++, no fast-math, no FP contraction)."""
    stale = (not _LIB.exists()) or _LIB.stat().st_mtime < max(_SRC.stat().st_mtime, _HDR.stat().st_mtime)
    if force or stale:
        tmp = _LIB.with_suffix(f".{os.getpid()}.tmp")
        subprocess.run(["g++", *CXXFLAGS, "-o", str(tmp), str(_SRC)], check=True, cwd=str(_HERE))
        os.replace(tmp, _LIB)
    return _LIB


class OracleParams(C.Structure):
    _fields_ = [("m_ion_u", C.c_double), ("m_atom_u", C.c_double), ("alpha_au", C.c_double),
                ("a", C.c_double * 3), ("q", C.c_double * 3), ("omega_rf_au", C.c_double),
                ("De_K", C.c_double), ("r0_a0", C.c_double), ("rtol", C.c_double), ("atol", C.c_double),
                ("t_max_rf", C.c_double), ("h_max_rf", C.c_double), ("r_coll_a0", C.c_double),
                ("max_steps", C.c_uint64)]


class OracleDerived(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("m_i", "m_a", "C4", "C8", "De", "r_e", "Omega", "T_rf", "thr",
                                          "h_max", "h_min", "t_max", "r0", "r_coll")]


class OracleOutcome(C.Structure):
    _fields_ = [("ke_ion", C.c_double), ("t_dwell", C.c_double), ("t_life", C.c_double),
                ("va_f", C.c_double * 3),
                ("n_coll", C.c_uint32), ("n_tp", C.c_uint32), ("steps_acc", C.c_uint32),
                ("steps_rej", C.c_uint32), ("n_loc", C.c_uint32), ("status", C.c_int32),
                ("y_final", C.c_double * 12), ("t_first", C.c_double), ("t_last", C.c_double),
                ("h_first", C.c_double), ("h_last", C.c_double)]


OUTCOME_DTYPE = np.dtype([("ke_ion", "<f8"), ("t_dwell", "<f8"), ("t_life", "<f8"), ("va_f", "<f8", (3,)),
                          ("n_coll", "<u4"), ("n_tp", "<u4"), ("steps_acc", "<u4"), ("steps_rej", "<u4"),
                          ("n_loc", "<u4"), ("status", "<i4"), ("y_final", "<f8", (12,)),
                          ("t_first", "<f8"), ("t_last", "<f8"), ("h_first", "<f8"), ("h_last", "<f8")])
assert OUTCOME_DTYPE.itemsize == C.sizeof(OracleOutcome)


class OracleGen(C.Structure):
    _fields_ = [("mode", C.c_int32), ("domain", C.c_int32), ("phase_mode", C.c_int32),
                ("n_theta", C.c_uint32), ("n_phi", C.c_uint32), ("phase0", C.c_double),
                ("E_min_uK", C.c_double), ("E_max_uK", C.c_double),
                ("seed", C.c_uint64), ("cell", C.c_uint32), ("first_index", C.c_uint64),
                ("T_atom_uK", C.c_double), ("T_ion_uK", C.c_double)]


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        dp = C.POINTER(C.c_double)
        L.oracle_derive.argtypes = [C.POINTER(OracleParams), C.POINTER(OracleDerived)]
        L.oracle_potential.argtypes = [C.POINTER(OracleParams), C.c_double]
        L.oracle_potential.restype = C.c_double
        L.oracle_rhs.argtypes = [C.POINTER(OracleParams), C.c_double, C.c_double, dp, dp]
        L.oracle_rhs.restype = None
        L.oracle_step.argtypes = [C.POINTER(OracleParams), C.c_double, C.c_double, dp, C.c_double, dp, dp]
        L.oracle_step.restype = None
        L.oracle_err_norm.argtypes = [C.POINTER(OracleParams), dp, dp, dp]
        L.oracle_err_norm.restype = C.c_double
        L.oracle_trace.argtypes = [C.POINTER(OracleParams), dp, C.c_double, C.c_double, C.c_uint32, dp]
        L.oracle_trace.restype = None
        L.oracle_run.argtypes = [C.POINTER(OracleParams), dp, C.c_double, C.POINTER(OracleOutcome), dp,
                                 C.c_uint64, C.POINTER(C.c_uint64)]
        L.oracle_philox4x32_10.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
        L.oracle_philox4x32_10.restype = None
        L.oracle_u53.argtypes = [C.c_uint32, C.c_uint32]
        L.oracle_u53.restype = C.c_double
        L.oracle_generate.argtypes = [C.POINTER(OracleParams), C.POINTER(OracleGen), C.c_uint64, dp, dp, dp]
        L.oracle_run_generated.argtypes = [C.POINTER(OracleParams), C.POINTER(OracleGen),
                                           C.POINTER(C.c_uint64), C.c_uint64, C.c_uint64, C.c_void_p, C.c_int]
        L.oracle_run_explicit.argtypes = [C.POINTER(OracleParams), dp, dp, C.c_uint64, C.c_void_p, C.c_int]
        L.oracle_tableau.argtypes = [dp, dp, dp, dp]
        L.oracle_tableau.restype = None
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def to_params(p) -> OracleParams:
    """p: ia_inputs.Params (or any object with the same attribute names)."""
    return OracleParams(p.m_ion_u, p.m_atom_u, p.alpha_au, (C.c_double * 3)(*p.a), (C.c_double * 3)(*p.q),
                        p.omega_rf_au, p.De_K, p.r0_a0, p.rtol, p.atol, p.t_max_rf, p.h_max_rf,
                        p.r_coll_a0, int(p.max_steps))


def to_gen(l) -> OracleGen:
    """l: ia_inputs.Launch."""
    return OracleGen(l.mode, l.domain, l.phase_mode, l.n_theta, l.n_phi, l.phase0, l.E_min_uK, l.E_max_uK,
                     l.seed, l.cell, l.first_index, float(getattr(l, "T_atom_uK", 0.0)),
                     float(getattr(l, "T_ion_uK", 0.0)))


def derive(p) -> dict:
    d = OracleDerived()
    lib().oracle_derive(C.byref(to_params(p)), C.byref(d))
    return {n: getattr(d, n) for n, _ in OracleDerived._fields_}


def potential(p, r: float) -> float:
    return lib().oracle_potential(C.byref(to_params(p)), float(r))


def rhs(p, t_frac: float, phase: float, y) -> np.ndarray:
    y = np.ascontiguousarray(y, dtype=np.float64)
    f = np.empty(12)
    lib().oracle_rhs(C.byref(to_params(p)), t_frac, phase, _dp(y), _dp(f))
    return f


def step(p, t_frac: float, phase: float, y, h: float):
    y = np.ascontiguousarray(y, dtype=np.float64)
    ynew, e = np.empty(12), np.empty(12)
    lib().oracle_step(C.byref(to_params(p)), t_frac, phase, _dp(y), h, _dp(ynew), _dp(e))
    return ynew, e


def err_norm(p, y, ynew, e) -> float:
    y, ynew, e = (np.ascontiguousarray(v, dtype=np.float64) for v in (y, ynew, e))
    return lib().oracle_err_norm(C.byref(to_params(p)), _dp(y), _dp(ynew), _dp(e))


def trace(p, y0, phase: float, h: float, nsteps: int) -> np.ndarray:
    y0 = np.ascontiguousarray(y0, dtype=np.float64)
    st = np.empty((nsteps + 1, 13))
    lib().oracle_trace(C.byref(to_params(p)), _dp(y0), phase, h, nsteps, _dp(st))
    return st


def run(p, y0, phase: float = 0.0, path_cap: int = 0):
    """One adaptive trajectory.  Returns (outcome record as numpy scalar, path[(t,y)] or None)."""
    y0 = np.ascontiguousarray(y0, dtype=np.float64)
    out = np.zeros(1, dtype=OUTCOME_DTYPE)
    path = np.empty((path_cap, 13)) if path_cap else None
    n = C.c_uint64(0)
    rc = lib().oracle_run(C.byref(to_params(p)), _dp(y0), phase,
                          C.cast(out.ctypes.data, C.POINTER(OracleOutcome)),
                          _dp(path) if path is not None else None, path_cap, C.byref(n))
    if rc != 0:
        raise RuntimeError("oracle_run failed")
    return out[0], (path[: n.value] if path is not None else None)


def philox4x32_10(ctr, key) -> np.ndarray:
    c = (C.c_uint32 * 4)(*[int(x) for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) for x in key])
    o = (C.c_uint32 * 4)()
    lib().oracle_philox4x32_10(c, k, o)
    return np.array(list(o), dtype=np.uint32)


def u53(w_even: int, w_odd: int) -> float:
    return lib().oracle_u53(int(w_even), int(w_odd))


def generate(p, launch, indices) -> tuple:
    """ICs of local indices: (y0[n,12], phase[n], E_au[n])."""
    indices = np.asarray(indices, dtype=np.uint64).reshape(-1)
    pp, g = to_params(p), to_gen(launch)
    y0 = np.empty((len(indices), 12))
    ph = np.empty(len(indices))
    E = np.empty(len(indices))
    for n, idx in enumerate(indices):
        a, b = C.c_double(), C.c_double()
        rc = lib().oracle_generate(C.byref(pp), C.byref(g), int(idx), _dp(y0[n]), C.byref(a), C.byref(b))
        if rc != 0:
            raise RuntimeError("oracle_generate failed")
        ph[n], E[n] = a.value, b.value
    return y0, ph, E


def run_generated(p, launch, indices=None, first: int = 0, count: int | None = None, nthreads: int = 1) -> np.ndarray:
    pp, g = to_params(p), to_gen(launch)
    if indices is not None:
        indices = np.ascontiguousarray(indices, dtype=np.uint64).reshape(-1)
        count = len(indices)
        iptr = indices.ctypes.data_as(C.POINTER(C.c_uint64))
    else:
        iptr = None
        if count is None:
            count = launch.n - first
    outs = np.zeros(count, dtype=OUTCOME_DTYPE)
    rc = lib().oracle_run_generated(C.byref(pp), C.byref(g), iptr, first, count, outs.ctypes.data, nthreads)
    if rc != 0:
        raise RuntimeError("oracle_run_generated failed")
    return outs


def run_explicit(p, y0, phase, nthreads: int = 1) -> np.ndarray:
    y0 = np.ascontiguousarray(y0, dtype=np.float64).reshape(-1, 12)
    phase = np.ascontiguousarray(np.broadcast_to(np.asarray(phase, dtype=np.float64), (len(y0),)))
    outs = np.zeros(len(y0), dtype=OUTCOME_DTYPE)
    rc = lib().oracle_run_explicit(C.byref(to_params(p)), _dp(y0), _dp(phase), len(y0), outs.ctypes.data, nthreads)
    if rc != 0:
        raise RuntimeError("oracle_run_explicit failed")
    return outs


def tableau():
    c, a, b, bh = np.empty(7), np.empty(49), np.empty(7), np.empty(7)
    lib().oracle_tableau(_dp(c), _dp(a), _dp(b), _dp(bh))
    return c, a.reshape(7, 7), b, bh


# ---- reductions over the outcomes of an ensemble (plain numpy, the definitions written out) -------------

def life_bins(t_life, n_coll, T_rf: float, nbins: int = 64) -> np.ndarray:
    """Histogram of complex lifetimes (Fig. 2; reading R17): over trajectories with
    n_coll >= 2, bin = clamp(ilogb(((q q)(q q))) + 8, 0, nbins-1) with q = t_life / T_rf, every product rounded
    to double -- quarter-octave bins, bin b holding 2^((b-8)/4) <= q < 2^((b-7)/4)."""
    t_life = np.asarray(t_life, dtype=np.float64)
    sel = np.asarray(n_coll) >= 2
    q = t_life[sel] / np.float64(T_rf)
    q2 = q * q
    q4 = q2 * q2
    _, ex = np.frexp(q4)                      # q4 = m 2^ex with 0.5 <= m < 1, so ilogb(q4) = ex - 1
    e = np.where(q4 > 0.0, ex - 1, -1023)
    b = np.clip(e + 8, 0, nbins - 1).astype(np.int64)
    return np.bincount(b, minlength=nbins).astype(np.uint64)


def survival(t_life, n_coll, times) -> np.ndarray:
    """Fraction of complexes (n_coll >= 2) still alive after each of `times` (Fig. 2)."""
    t = np.asarray(t_life, dtype=np.float64)[np.asarray(n_coll) >= 2]
    if len(t) == 0:
        return np.zeros(len(times))
    return np.array([(t > x).mean() for x in np.asarray(times, dtype=np.float64)])
