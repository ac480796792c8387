"""ORACLE — TEST INFRASTRUCTURE ONLY (ctypes view of oracle/pic_oracle.cpp).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this.  It shares no code with paper_1111_5295_b200 and imports
nothing from it.  Marshalling only: every formula lives in pic_oracle.cpp, each with
its PAPER.md citation.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pic_oracle.cpp")
# PIC_ORACLE_SANITIZE=1 (tests/test_oracle_sanitized.py): the same source built with
# AddressSanitizer + UndefinedBehaviorSanitizer as libpic_oracle_san.so.  Loader switch only --
# the arithmetic is pic_oracle.cpp's either way; the process must then run under
# LD_PRELOAD=<libasan.so> (the ASan runtime has to be the first library of the process).
_SANITIZE = os.environ.get("PIC_ORACLE_SANITIZE", "0") == "1"
_LIB = os.path.join(_HERE, "libpic_oracle_san.so" if _SANITIZE else "libpic_oracle.so")
_OPT = (["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined",
         "-fno-sanitize-recover=all"] if _SANITIZE else ["-O2"])


def build(force=False):
    """Compile pic_oracle.cpp -> libpic_oracle.so (g++ -O2, serial, no FMA contraction)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    cmd = ["g++"] + _OPT + ["-std=c++17", "-ffp-contract=off", "-fPIC", "-shared", "-Wall",
                            "-o", _LIB, _SRC]
    subprocess.run(cmd, check=True)
    return _LIB


class Params(C.Structure):
    _fields_ = [("eps_a", C.c_double), ("eps_r", C.c_double), ("kappa_max", C.c_double),
                ("tol", C.c_double), ("max_substeps", C.c_int32), ("cn_mode", C.c_int32),
                ("picard_max", C.c_int32), ("pad_", C.c_int32)]


class Stats(C.Structure):
    _fields_ = [(k, C.c_int64) for k in
                ("n_sub", "n_cross", "n_picard_it", "n_picard_cap", "n_kappa_cap",
                 "n_substep_cap", "n_neg_disc", "n_clamped_tau")]

    def as_dict(self):
        return {k: int(getattr(self, k)) for k, _ in self._fields_}


class Substep(C.Structure):
    _fields_ = [("dtau_est", C.c_double), ("dtau", C.c_double), ("s0", C.c_double),
                ("v0", C.c_double), ("s1", C.c_double), ("v1", C.c_double), ("a", C.c_double),
                ("aprime", C.c_double), ("a_mid", C.c_double), ("cell", C.c_int32),
                ("crossed", C.c_int32)]


PICARD, DIRECT = 0, 1


def make_params(eps_a=1e-8, eps_r=0.02, kappa_max=0.5, tol=1e-10, max_substeps=1 << 20,
                cn_mode=PICARD, picard_max=100):
    return Params(eps_a, eps_r, kappa_max, tol, max_substeps, cn_mode, picard_max, 0)


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_estimate_dtau.restype = C.c_double
        _lib.oracle_estimate_dtau.argtypes = [C.c_double] * 5
        _lib.oracle_trace_particle.restype = C.c_int64
    return _lib


def _p(a, ct):
    return None if a is None else a.ctypes.data_as(C.POINTER(ct))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def bin_particles(n_cells, length, x):
    x = _f64(x)
    cell = np.empty(x.size, np.int32)
    s = np.empty(x.size, np.float64)
    lib().oracle_bin(C.c_int32(n_cells), C.c_double(length), C.c_int64(x.size),
                     _p(x, C.c_double), _p(cell, C.c_int32), _p(s, C.c_double))
    return cell, s


def move_accumulate(n_cells, length, q_over_m, w_q, cell0, s0, v0, E_n, E_np1, dt,
                    params=None, J=None, stats=None, want_state=True):
    """One species through O1-O9.  Returns dict(cell, s, v, k, n_sub, n_cross, J, stats).

    J (raw, un-normalised) and stats accumulate when passed in."""
    params = params or make_params()
    cell0 = np.ascontiguousarray(cell0, dtype=np.int32)
    s0, v0, E_n, E_np1 = _f64(s0), _f64(v0), _f64(E_n), _f64(E_np1)
    n = cell0.size
    assert s0.size == n and v0.size == n and E_n.size == n_cells and E_np1.size == n_cells
    if J is None:
        J = np.zeros(n_cells, np.float64)
    if stats is None:
        stats = Stats()
    out = {}
    if want_state:
        out = dict(cell=np.empty(n, np.int32), s=np.empty(n), v=np.empty(n),
                   k=np.empty(n, np.int32), n_sub=np.empty(n, np.uint32),
                   n_cross=np.empty(n, np.uint32))
    rc = lib().oracle_move_accumulate(
        C.c_int32(n_cells), C.c_double(length), C.c_double(q_over_m), C.c_double(w_q),
        C.c_int64(n), _p(cell0, C.c_int32), _p(s0, C.c_double), _p(v0, C.c_double),
        _p(E_n, C.c_double), _p(E_np1, C.c_double), C.c_double(dt), C.byref(params),
        _p(out.get("cell"), C.c_int32), _p(out.get("s"), C.c_double),
        _p(out.get("v"), C.c_double), _p(out.get("k"), C.c_int32),
        _p(out.get("n_sub"), C.c_uint32), _p(out.get("n_cross"), C.c_uint32),
        _p(J, C.c_double), C.byref(stats))
    if rc != 0:
        raise ValueError(f"oracle_move_accumulate failed: {rc}")
    out["J"] = J
    out["stats"] = stats
    return out


def trace_particle(n_cells, length, q_over_m, w_q, cell0, s0, v0, E_n, E_np1, dt,
                   params=None, cap=1 << 16):
    """One particle with a record per sub-step.  Returns (records, final dict)."""
    params = params or make_params()
    E_n, E_np1 = _f64(E_n), _f64(E_np1)
    rec = (Substep * cap)()
    c1, k = C.c_int32(), C.c_int32()
    s1, v1 = C.c_double(), C.c_double()
    J = np.zeros(n_cells)
    nrec = lib().oracle_trace_particle(
        C.c_int32(n_cells), C.c_double(length), C.c_double(q_over_m), C.c_double(w_q),
        C.c_int32(int(cell0)), C.c_double(float(s0)), C.c_double(float(v0)),
        _p(E_n, C.c_double), _p(E_np1, C.c_double), C.c_double(dt), C.byref(params), rec,
        C.c_int64(cap), C.byref(c1), C.byref(s1), C.byref(v1), C.byref(k), _p(J, C.c_double))
    if nrec < 0:
        raise ValueError("oracle_trace_particle failed")
    recs = [rec[i] for i in range(nrec)]
    return recs, dict(cell=c1.value, s=s1.value, v=v1.value, k=k.value, J=J)


def estimate_dtau(a, aprime, v, eps_a, eps_r):
    return lib().oracle_estimate_dtau(a, aprime, v, eps_a, eps_r)


def jbar_from_J(n_cells, length, dt, J):
    J = _f64(J)
    out = np.empty(n_cells)
    lib().oracle_jbar(C.c_int32(n_cells), C.c_double(length), C.c_double(dt), _p(J, C.c_double),
                      _p(out, C.c_double))
    return out


def residual(E_n, E_np1, dt, jbar):
    E_n, E_np1, jbar = _f64(E_n), _f64(E_np1), _f64(jbar)
    out = np.empty(E_n.size)
    lib().oracle_residual(C.c_int32(E_n.size), _p(E_n, C.c_double), _p(E_np1, C.c_double),
                          C.c_double(dt), _p(jbar, C.c_double), _p(out, C.c_double))
    return out


def rho(n_cells, length, w_q, cell, s, rho=None):
    cell = np.ascontiguousarray(cell, dtype=np.int32)
    s = _f64(s)
    if rho is None:
        rho = np.zeros(n_cells)
    lib().oracle_rho(C.c_int32(n_cells), C.c_double(length), C.c_double(w_q),
                     C.c_int64(cell.size), _p(cell, C.c_int32), _p(s, C.c_double),
                     _p(rho, C.c_double))
    return rho
