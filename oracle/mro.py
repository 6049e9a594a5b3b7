"""ctypes binding of the CPU oracle ``oracle/mro.c`` (TEST INFRASTRUCTURE -- not part of the product path).

Only tests/, ``__graft_entry__.smoke()`` and bench.py's ``cpu_baseline`` / ``--impl reference`` legs may import
this module.  All arrays are float64, C-contiguous, shape ``(3, nz, ny, nx)`` (scalars: ``(nz, ny, nx)``).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_lib = C.CDLL(_build.build())

_i3 = C.c_int * 3
_d3 = C.c_double * 3
_dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_vp = C.c_void_p

_lib.mro_set_threads.argtypes = [C.c_int]
_lib.mro_get_threads.restype = C.c_int
_lib.mro_max_threads.restype = C.c_int
_lib.mro_reference_grid.argtypes = [_i3, _d3, _d3, _dp]
_lib.mro_jacobian.argtypes = [_i3, _d3, _d3, _dp, _vp, _vp]
_lib.mro_push_forward.argtypes = [_i3, _d3, _d3, _dp, _dp, _dp, _vp]
_lib.mro_curl_mimetic.argtypes = [_i3, _dp, _dp, _dp]
_lib.mro_curl_direct.argtypes = [_i3, _d3, _d3, _dp, _dp, _dp]
_lib.mro_fields.argtypes = [_i3, _d3, _d3, _dp, _dp, C.c_double, C.c_int, _vp, _vp, _vp, _vp]
_lib.mro_step.argtypes = [_i3, _d3, _d3, _dp, _dp, C.c_double, C.c_double, C.c_longlong, C.c_int]
_lib.mro_diagnostics.argtypes = [_i3, _d3, _d3, _dp, _dp, C.c_int, C.c_double * 4]

MIMETIC, DIRECT = 0, 1


class NumericError(ArithmeticError):
    """det(F) <= 0, a non-finite value, or a singular matrix of normals."""


def set_threads(t: int) -> None:
    _lib.mro_set_threads(int(t))


def get_threads() -> int:
    return _lib.mro_get_threads()


def max_threads() -> int:
    return _lib.mro_max_threads()


def _g(n, lo, hi):
    return _i3(*[int(v) for v in n]), _d3(*[float(v) for v in lo]), _d3(*[float(v) for v in hi])


def _shape(n):
    return (3, int(n[2]), int(n[1]), int(n[0]))


def _arr(a, n, lead=3):
    a = np.ascontiguousarray(a, dtype=np.float64)
    want = _shape(n) if lead == 3 else _shape(n)[1:]
    if a.shape != want:
        raise ValueError("expected shape %r, got %r" % (want, a.shape))
    return a


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _check(rc, strict=True):
    if rc == 5 and strict:
        raise NumericError("oracle: numeric failure")
    if rc not in (0, 5):
        raise ValueError("oracle: bad argument (rc=%d)" % rc)
    return rc


def reference_grid(n, lo, hi):
    X = np.empty(_shape(n))
    _check(_lib.mro_reference_grid(*_g(n, lo, hi), X))
    return X


def jacobian(n, lo, hi, x, strict=True):
    """O1/O2: returns (F, det) with F[c, a] = dx_c/dX_a of shape (3,3,nz,ny,nx)."""
    x = _arr(x, n)
    F = np.empty((3, 3) + _shape(n)[1:])
    det = np.empty(_shape(n)[1:])
    _check(_lib.mro_jacobian(*_g(n, lo, hi), x, _ptr(F), _ptr(det)), strict)
    return F, det


def push_forward(n, lo, hi, x, B0, strict=True):
    """O3: returns (B, det)."""
    x, B0 = _arr(x, n), _arr(B0, n)
    B = np.empty(_shape(n))
    det = np.empty(_shape(n)[1:])
    _check(_lib.mro_push_forward(*_g(n, lo, hi), x, B0, B, _ptr(det)), strict)
    return B, det


def curl_mimetic(n, x, B, strict=True):
    """O4m on given nodal x and B (Eqs. 2.3-2.7 literally); J = 0 on boundary nodes."""
    x, B = _arr(x, n), _arr(B, n)
    J = np.empty(_shape(n))
    _check(_lib.mro_curl_mimetic(_i3(*[int(v) for v in n]), x, B, J), strict)
    return J


def curl_direct(n, lo, hi, x, B0, strict=True):
    """O4d from x and B0; J = 0 on boundary nodes."""
    x, B0 = _arr(x, n), _arr(B0, n)
    J = np.empty(_shape(n))
    _check(_lib.mro_curl_direct(*_g(n, lo, hi), x, B0, J), strict)
    return J


def fields(n, lo, hi, x, B0, gamma=1.0, op=MIMETIC, strict=True):
    """Returns (B, J, u, det) of the state x."""
    x, B0 = _arr(x, n), _arr(B0, n)
    B, J, u = np.empty(_shape(n)), np.empty(_shape(n)), np.empty(_shape(n))
    det = np.empty(_shape(n)[1:])
    _check(_lib.mro_fields(*_g(n, lo, hi), x, B0, float(gamma), int(op), _ptr(B), _ptr(J), _ptr(u), _ptr(det)), strict)
    return B, J, u, det


def step(n, lo, hi, x, B0, dt, nsteps=1, gamma=1.0, op=MIMETIC, strict=True):
    """O6: returns a new array holding x after ``nsteps`` forward-Euler steps."""
    x = _arr(x, n).copy()
    B0 = _arr(B0, n)
    _check(_lib.mro_step(*_g(n, lo, hi), x, B0, float(gamma), float(dt), int(nsteps), int(op)), strict)
    return x


def diagnostics(n, lo, hi, x, B0, op=MIMETIC, strict=True):
    """O7: dict(energy, max_jxb, xi, min_det)."""
    x, B0 = _arr(x, n), _arr(B0, n)
    out = (C.c_double * 4)()
    _check(_lib.mro_diagnostics(*_g(n, lo, hi), x, B0, int(op), out), strict)
    return {"energy": out[0], "max_jxb": out[1], "xi": out[2], "min_det": out[3]}
