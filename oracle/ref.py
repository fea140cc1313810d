"""ctypes binding of the oracle library (``oracle/liblrmd_ref.so``).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only ``tests/``, ``__graft_entry__.smoke()``
and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this.
It imports nothing from the CUDA package and holds no arithmetic of its own —
argument marshalling only; every number comes from ``lrmd_ref.cpp``.

All arrays are host numpy fp64, C-contiguous.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HMF, RING, GRAV2D = 0, 1, 2

_HERE = os.path.dirname(os.path.abspath(__file__))
_lib = None

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int64)


def _load():
    global _lib
    if _lib is not None:
        return _lib
    import importlib.util
    spec = importlib.util.spec_from_file_location("_lrmd_ref_build", os.path.join(_HERE, "build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    path = mod.build()
    lib = C.CDLL(path)
    lib.lrmd_ref_coefficients.argtypes = [_dp]
    lib.lrmd_ref_coefficients.restype = None
    lib.lrmd_ref_forces.argtypes = [C.c_int, C.c_int64, C.c_double, _dp, _dp, _dp, _dp, C.c_int, C.c_int]
    lib.lrmd_ref_forces_rows.argtypes = [C.c_int, C.c_int64, C.c_double, _dp, _dp, _ip, C.c_int64,
                                         _dp, _dp, C.c_int, C.c_int]
    lib.lrmd_ref_abs_force_sums.argtypes = [C.c_int, C.c_int64, C.c_double, _dp, _dp, _ip, C.c_int64,
                                            _dp, _dp, _dp, _dp, C.c_int, C.c_int]
    lib.lrmd_ref_energy.argtypes = [C.c_int, C.c_int64, C.c_double, _dp, _dp, _dp, _dp, _dp, _dp,
                                    C.c_int, C.c_int]
    lib.lrmd_ref_step.argtypes = [C.c_int, C.c_int64, C.c_double, _dp, _dp, _dp, _dp, _dp, _dp,
                                  C.c_int, C.c_int64, C.c_double, C.c_int, C.c_int]
    lib.lrmd_ref_max_threads.argtypes = []
    for f in (lib.lrmd_ref_forces, lib.lrmd_ref_forces_rows, lib.lrmd_ref_abs_force_sums,
              lib.lrmd_ref_energy, lib.lrmd_ref_step, lib.lrmd_ref_max_threads):
        f.restype = C.c_int
    _lib = lib
    return lib


def _a(x):
    """fp64 C-contiguous view (copy only if needed) or None."""
    if x is None:
        return None
    return np.ascontiguousarray(x, dtype=np.float64)


def _p(x):
    return None if x is None else x.ctypes.data_as(_dp)


def _chk(rc, what):
    if rc != 0:
        raise ValueError(f"oracle {what}: invalid arguments (rc={rc})")


def max_threads() -> int:
    return int(_load().lrmd_ref_max_threads())


def coefficients():
    """(B0, B1, D0, D1), reading G4."""
    out = np.zeros(4)
    _load().lrmd_ref_coefficients(_p(out))
    return tuple(float(v) for v in out)


def forces(model, eps, q0, q1=None, form=0, nthreads=0):
    """Forces on all particles; returns f (HMF/RING) or (fx, fy) (GRAV2D)."""
    q0 = _a(q0); q1 = _a(q1)
    N = q0.shape[0]
    f0 = np.empty(N); f1 = np.empty(N) if model == GRAV2D else None
    _chk(_load().lrmd_ref_forces(model, N, float(eps), _p(q0), _p(q1), _p(f0), _p(f1), form, nthreads), "forces")
    return (f0, f1) if model == GRAV2D else f0


def forces_rows(model, eps, q0, q1, rows, form=0, nthreads=0, with_abs=False):
    """Forces on the sampled rows (each against all N).  with_abs: also A_i = sum_j |f_ij|.

    Returns (f0, f1_or_None) or (f0, f1_or_None, A0, A1_or_None).
    """
    q0 = _a(q0); q1 = _a(q1)
    N = q0.shape[0]
    rows = np.ascontiguousarray(rows, dtype=np.int64)
    R = rows.shape[0]
    two = model == GRAV2D
    f0 = np.empty(R); f1 = np.empty(R) if two else None
    rp = rows.ctypes.data_as(_ip)
    if not with_abs:
        _chk(_load().lrmd_ref_forces_rows(model, N, float(eps), _p(q0), _p(q1), rp, R, _p(f0), _p(f1),
                                          form, nthreads), "forces_rows")
        return f0, f1
    A0 = np.empty(R); A1 = np.empty(R) if two else None
    _chk(_load().lrmd_ref_abs_force_sums(model, N, float(eps), _p(q0), _p(q1), rp, R, _p(f0), _p(f1),
                                         _p(A0), _p(A1), form, nthreads), "abs_force_sums")
    return f0, f1, A0, A1


def forces_abs(model, eps, q0, q1=None, form=0, nthreads=0):
    """All rows: (f0, f1_or_None, A0, A1_or_None)."""
    q0 = _a(q0); q1 = _a(q1)
    N = q0.shape[0]
    two = model == GRAV2D
    f0 = np.empty(N); f1 = np.empty(N) if two else None
    A0 = np.empty(N); A1 = np.empty(N) if two else None
    _chk(_load().lrmd_ref_abs_force_sums(model, N, float(eps), _p(q0), _p(q1), None, 0, _p(f0), _p(f1),
                                         _p(A0), _p(A1), form, nthreads), "abs_force_sums")
    return f0, f1, A0, A1


def energy(model, eps, q0, q1, p0, p1, form=0, nthreads=0):
    """Returns (out4, out_abs): out4 = (K, V, a, b); out_abs = (sum|K terms|, sum|V terms|)."""
    q0 = _a(q0); q1 = _a(q1); p0 = _a(p0); p1 = _a(p1)
    N = q0.shape[0]
    out4 = np.zeros(4); out_abs = np.zeros(2)
    _chk(_load().lrmd_ref_energy(model, N, float(eps), _p(q0), _p(q1), _p(p0), _p(p1), _p(out4), _p(out_abs),
                                 form, nthreads), "energy")
    return out4, out_abs


def step(model, eps, q0, q1, p0, p1, n, dt, f0=None, f1=None, force_valid=False, form=0, nthreads=0):
    """n steps IN PLACE on the given fp64 C-contiguous arrays.  Returns the force arrays (f0, f1)."""
    for x in (q0, q1, p0, p1, f0, f1):
        if x is not None:
            assert x.dtype == np.float64 and x.flags.c_contiguous and x.flags.writeable
    N = q0.shape[0]
    two = model == GRAV2D
    if f0 is None:
        f0 = np.zeros(N); force_valid = False
    if two and f1 is None:
        f1 = np.zeros(N); force_valid = False
    _chk(_load().lrmd_ref_step(model, N, float(eps), _p(q0), _p(q1), _p(p0), _p(p1), _p(f0), _p(f1),
                               1 if force_valid else 0, int(n), float(dt), form, nthreads), "step")
    return f0, f1
