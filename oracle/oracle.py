"""ctypes front end of the CPU oracle (oracle/demons_oracle.c) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from the CUDA package.  Arrays: volumes are float32
numpy arrays of shape (nz, ny, nx); fields are float32 (3, nz, ny, nx).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "liboracle_demons.so")
_SRC = os.path.join(_HERE, "demons_oracle.c")
_HDR = os.path.join(_HERE, "demons_oracle.h")

PASSIVE, EVOLVED_PASSIVE, ACTIVE, DOUBLE, ADJUSTED_DOUBLE, INVERSE_CONSISTENT = range(6)


def build(force: bool = False) -> str:
    """gcc -O2, single-threaded, no fast-math.  Rebuilds when the source is newer than the library."""
    stale = (not os.path.exists(_LIB_PATH)
             or os.path.getmtime(_LIB_PATH) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR)))
    if force or stale:
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-Wall", "-Wextra",
                               "-o", _LIB_PATH, _SRC, "-lm"])
    return _LIB_PATH


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.oracle_final_ssd.restype = ctypes.c_double
        _lib.oracle_cc.restype = ctypes.c_double
        _lib.oracle_gauss_taps.restype = ctypes.c_int
        _lib.oracle_register.restype = ctypes.c_int
    return _lib


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p) if a is not None else None


def _dims_of(vol_shape):
    nz, ny, nx = vol_shape[-3:]
    return (ctypes.c_int * 3)(nx, ny, nz)


def gradient(I):
    I = _f32(I)
    g = np.empty((3,) + I.shape, dtype=np.float32)
    lib().oracle_gradient(_ptr(I), _dims_of(I.shape), _ptr(g))
    return g


def warp(I, u):
    I, u = _f32(I), _f32(u)
    out = np.empty_like(I)
    lib().oracle_warp(_ptr(I), _ptr(u), _dims_of(I.shape), _ptr(out))
    return out


def force_voxel(variant, alpha, d, gS=None, gM0=None, gMw=None, gSw=None):
    def v(g):
        return (ctypes.c_double * 3)(*(g if g is not None else (0.0, 0.0, 0.0)))
    F = (ctypes.c_double * 3)()
    lib().oracle_force_voxel(ctypes.c_int(variant), ctypes.c_double(alpha), ctypes.c_double(d),
                             v(gS), v(gM0), v(gMw), v(gSw), F)
    return np.array(list(F))


def gauss_taps(sigma):
    w = np.zeros(64, dtype=np.float32)
    R = lib().oracle_gauss_taps(ctypes.c_double(sigma), _ptr(w), 64)
    assert R >= 0
    return w[:R + 1].copy()


def smooth(field, sigma):
    """field: (ncomp, nz, ny, nx) or (nz, ny, nx)."""
    f = _f32(field)
    ncomp = 1 if f.ndim == 3 else f.shape[0]
    out = np.empty_like(f)
    lib().oracle_smooth(_ptr(f), _ptr(out), _dims_of(f.shape), ctypes.c_int(ncomp), ctypes.c_double(sigma))
    return out


def coarse_shape(shape):
    nz, ny, nx = shape[-3:]
    return ((nz + 1) // 2, (ny + 1) // 2, (nx + 1) // 2)


def restrict(fine):
    fine = _f32(fine)
    coarse = np.empty(coarse_shape(fine.shape), dtype=np.float32)
    lib().oracle_restrict(_ptr(fine), _dims_of(fine.shape), _ptr(coarse))
    return coarse


def prolong(uc, fine_shape):
    uc = _f32(uc)
    uf = np.empty((3,) + tuple(fine_shape[-3:]), dtype=np.float32)
    lib().oracle_prolong(_ptr(uc), _dims_of(uc.shape), _dims_of(uf.shape), _ptr(uf))
    return uf


def warp_force(variant, alpha, S, M, u, ub=None, gS=None, gM0=None):
    """One un-smoothed update.  Fixed gradients are computed here when the variant needs them
    and they are not supplied.  Returns (u_out, ub_out or None, metrics[3])."""
    S, M, u = _f32(S), _f32(M), _f32(u)
    if variant in (PASSIVE, EVOLVED_PASSIVE, DOUBLE, ADJUSTED_DOUBLE) and gS is None:
        gS = gradient(S)
    if variant == EVOLVED_PASSIVE and gM0 is None:
        gM0 = gradient(M)
    ic = variant == INVERSE_CONSISTENT
    ub = _f32(ub) if ic else None
    u_out = np.empty_like(u)
    ub_out = np.empty_like(u) if ic else None
    m = np.zeros(3, dtype=np.float64)
    lib().oracle_warp_force(ctypes.c_int(variant), ctypes.c_double(alpha), _dims_of(S.shape), _ptr(S), _ptr(M),
                            _ptr(gS), _ptr(gM0), _ptr(u), _ptr(u_out), _ptr(ub), _ptr(ub_out), _ptr(m))
    return u_out, ub_out, m


def register(variant, alpha, sigma, S, M, iters, u0=None, ub0=None, eps=0.0):
    """Full registration.  iters: list per level, coarse -> fine.  Returns dict(u, ub, stats, iters_done)."""
    S, M = _f32(S), _f32(M)
    levels = len(iters)
    u = np.zeros((3,) + S.shape, dtype=np.float32) if u0 is None else _f32(u0).copy()
    ic = variant == INVERSE_CONSISTENT
    ub = None
    if ic:
        ub = np.zeros((3,) + S.shape, dtype=np.float32) if ub0 is None else _f32(ub0).copy()
    stats = np.zeros((int(sum(iters)), 3), dtype=np.float64)
    done = (ctypes.c_int * levels)()
    it = (ctypes.c_int * levels)(*[int(i) for i in iters])
    rc = lib().oracle_register(ctypes.c_int(variant), ctypes.c_double(alpha), ctypes.c_double(sigma),
                               _dims_of(S.shape), _ptr(S), _ptr(M), _ptr(u), _ptr(ub), ctypes.c_int(levels), it,
                               ctypes.c_double(eps), _ptr(stats), done)
    if rc != 0:
        raise ValueError("oracle_register: bad arguments")
    return {"u": u, "ub": ub, "stats": stats, "iters_done": list(done)}


def final_ssd(variant, S, M, u, ub=None):
    S, M, u = _f32(S), _f32(M), _f32(u)
    ub = _f32(ub) if ub is not None else None
    return float(lib().oracle_final_ssd(ctypes.c_int(variant), _dims_of(S.shape), _ptr(S), _ptr(M), _ptr(u), _ptr(ub)))


def ic_error(uf, ub):
    uf, ub = _f32(uf), _f32(ub)
    mean, mx = ctypes.c_double(), ctypes.c_double()
    lib().oracle_ic_error(_ptr(uf), _ptr(ub), _dims_of(uf.shape), ctypes.byref(mean), ctypes.byref(mx))
    return mean.value, mx.value


def cc(variant, S, M, u, ub=None):
    S, M, u = _f32(S), _f32(M), _f32(u)
    ub = _f32(ub) if ub is not None else None
    return float(lib().oracle_cc(ctypes.c_int(variant), _dims_of(S.shape), _ptr(S), _ptr(M), _ptr(u), _ptr(ub)))


def point_error(u, spacing, points, expect):
    u, points, expect = _f32(u), _f32(points), _f32(expect)
    n = points.shape[0]
    err = np.empty(n, dtype=np.float64)
    sp = (ctypes.c_double * 3)(*[float(v) for v in spacing])
    lib().oracle_point_error(_ptr(u), _dims_of(u.shape), sp, ctypes.c_int(n), _ptr(points), _ptr(expect), _ptr(err))
    return err


if __name__ == "__main__":
    print(build(force=True))
