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

_lib.mro_set_bc.argtypes = [_i3]
_lib.mro_curl_mimetic_dom.argtypes = [_i3, _vp, _vp, _dp, _dp, _dp]
_RHS = C.CFUNCTYPE(C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_void_p)
_lib.mro_cash_karp_trial.argtypes = [C.c_longlong, _dp, C.c_double, _RHS, C.c_void_p, _vp, _vp, C.POINTER(C.c_double), _dp]
_lib.mro_step_control.argtypes = [C.c_double, C.c_double, C.c_double, C.POINTER(C.c_double)]
_lib.mro_step_adaptive.argtypes = [_i3, _d3, _d3, _dp, _dp, C.c_double, C.c_int, C.c_double, C.c_double, C.POINTER(C.c_double),
                                   C.POINTER(C.c_double), C.c_longlong, C.c_longlong * 2, _vp, C.c_longlong]
_lib.mro_convexity.argtypes = [_i3, _d3, _d3, _dp, _vp, C.POINTER(C.c_longlong)]
_lib.mro_eps_star.argtypes = [_i3, _d3, _d3, _dp, _dp, C.c_int, C.c_int, C.c_int, C.c_double, _vp, C.POINTER(C.c_double)]
_lib.mro_sigma.argtypes = [_i3, _d3, _d3, _dp, _dp, _dp, _dp, C.POINTER(C.c_double), C.POINTER(C.c_double)]

MIMETIC, DIRECT = 0, 1
LINE_TIED, PERIODIC = 0, 1


class _bc:
    """Boundary type per logical axis for the calls inside the ``with`` block (0 line-tied, 1 periodic; Eqs. 2.12-2.14)."""

    def __init__(self, bc):
        self.bc = tuple(int(b) for b in (bc or (0, 0, 0)))

    def __enter__(self):
        _lib.mro_set_bc(_i3(*self.bc))

    def __exit__(self, *a):
        _lib.mro_set_bc(_i3(0, 0, 0))


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


def jacobian(n, lo, hi, x, strict=True, bc=None):
    """O1/O2: returns (F, det) with F[c, a] = dx_c/dX_a of shape (3,3,nz,ny,nx)."""
    x = _arr(x, n)
    F = np.empty((3, 3) + _shape(n)[1:])
    det = np.empty(_shape(n)[1:])
    with _bc(bc):
        _check(_lib.mro_jacobian(*_g(n, lo, hi), x, _ptr(F), _ptr(det)), strict)
    return F, det


def push_forward(n, lo, hi, x, B0, strict=True, bc=None):
    """O3: returns (B, det)."""
    x, B0 = _arr(x, n), _arr(B0, n)
    B = np.empty(_shape(n))
    det = np.empty(_shape(n)[1:])
    with _bc(bc):
        _check(_lib.mro_push_forward(*_g(n, lo, hi), x, B0, B, _ptr(det)), strict)
    return B, det


def curl_mimetic(n, x, B, strict=True, lo=None, hi=None, bc=None):
    """O4m on given nodal x and B (Eqs. 2.3-2.7 literally); J = 0 on boundary nodes.  A periodic axis needs lo/hi
    (the ghost positions are shifted by the period, Eqs. 2.12/2.13)."""
    x, B = _arr(x, n), _arr(B, n)
    J = np.empty(_shape(n))
    with _bc(bc):
        if lo is None:
            _check(_lib.mro_curl_mimetic(_i3(*[int(v) for v in n]), x, B, J), strict)
        else:
            gi, glo, ghi = _g(n, lo, hi)
            _check(_lib.mro_curl_mimetic_dom(gi, C.cast(glo, C.c_void_p), C.cast(ghi, C.c_void_p), x, B, J), strict)
    return J


def curl_direct(n, lo, hi, x, B0, strict=True, bc=None):
    """O4d from x and B0; J = 0 on boundary nodes."""
    x, B0 = _arr(x, n), _arr(B0, n)
    J = np.empty(_shape(n))
    with _bc(bc):
        _check(_lib.mro_curl_direct(*_g(n, lo, hi), x, B0, J), strict)
    return J


def fields(n, lo, hi, x, B0, gamma=1.0, op=MIMETIC, strict=True, bc=None):
    """Returns (B, J, u, det) of the state x."""
    x, B0 = _arr(x, n), _arr(B0, n)
    B, J, u = np.empty(_shape(n)), np.empty(_shape(n)), np.empty(_shape(n))
    det = np.empty(_shape(n)[1:])
    with _bc(bc):
        _check(_lib.mro_fields(*_g(n, lo, hi), x, B0, float(gamma), int(op), _ptr(B), _ptr(J), _ptr(u), _ptr(det)), strict)
    return B, J, u, det


def step(n, lo, hi, x, B0, dt, nsteps=1, gamma=1.0, op=MIMETIC, strict=True, bc=None):
    """O6: returns a new array holding x after ``nsteps`` forward-Euler steps."""
    x = _arr(x, n).copy()
    B0 = _arr(B0, n)
    with _bc(bc):
        _check(_lib.mro_step(*_g(n, lo, hi), x, B0, float(gamma), float(dt), int(nsteps), int(op)), strict)
    return x


def diagnostics(n, lo, hi, x, B0, op=MIMETIC, strict=True, bc=None):
    """O7: dict(energy, max_jxb, xi, min_det)."""
    x, B0 = _arr(x, n), _arr(B0, n)
    out = (C.c_double * 4)()
    with _bc(bc):
        _check(_lib.mro_diagnostics(*_g(n, lo, hi), x, B0, int(op), out), strict)
    return {"energy": out[0], "max_jxb": out[1], "xi": out[2], "min_det": out[3]}


# ---- section 2.4: adaptive Cash-Karp RK5(4) ---------------------------------------------------------------------

def cash_karp_trial(y, dt, f):
    """One trial step for the autonomous system y' = f(y) (numpy in, numpy out): returns (y5, y4, Lambda)."""
    y = np.ascontiguousarray(y, dtype=np.float64).ravel()
    m = y.size

    def cb(yp, dp, _):
        yy = np.ctypeslib.as_array(yp, shape=(m,))
        np.ctypeslib.as_array(dp, shape=(m,))[:] = f(yy.copy())
        return 0

    y5, y4, work, lam = np.empty(m), np.empty(m), np.empty(7 * m), C.c_double()
    _check(_lib.mro_cash_karp_trial(m, y, float(dt), _RHS(cb), None, _ptr(y5), _ptr(y4), C.byref(lam), work))
    return y5, y4, lam.value


def step_control(dt, lam, lam0):
    """Eq. 2.11 and the accept/reject rule: returns (accepted, dt_next)."""
    out = C.c_double()
    ok = _lib.mro_step_control(float(dt), float(lam), float(lam0), C.byref(out))
    return bool(ok), out.value


def step_adaptive(n, lo, hi, x, B0, t_end, lam0, dt, t=0.0, gamma=1.0, op=MIMETIC, max_trials=100000, strict=True, bc=None):
    """Integrate to t_end: returns (x, t, dt_next, (accepted, rejected), trace[trials, 4] = t, dt tried, Lambda, accepted)."""
    x = _arr(x, n).copy()
    B0 = _arr(B0, n)
    tt, dd = C.c_double(float(t)), C.c_double(float(dt))
    counts = (C.c_longlong * 2)()
    trace = np.zeros((int(max_trials), 4))
    with _bc(bc):
        rc = _lib.mro_step_adaptive(*_g(n, lo, hi), x, B0, float(gamma), int(op), float(t_end), float(lam0), C.byref(tt), C.byref(dd),
                                    int(max_trials), counts, _ptr(trace), int(max_trials))
    if rc == 7:
        raise RuntimeError("oracle: max_trials exhausted")
    _check(rc, strict)
    return x, tt.value, dd.value, (counts[0], counts[1]), trace[: counts[0] + counts[1]]


# ---- section 3.2: convexity, eps*, sigma ------------------------------------------------------------------------

def convexity(n, lo, hi, x, bc=None):
    """Eqs. 3.10-3.11: returns (kappa[nz, ny, nx] of +1/-1, number of nodes with kappa = -1)."""
    x = _arr(x, n)
    kap = np.empty(_shape(n)[1:], dtype=np.int32)
    cnt = C.c_longlong()
    with _bc(bc):
        _check(_lib.mro_convexity(*_g(n, lo, hi), x, kap.ctypes.data_as(C.c_void_p), C.byref(cnt)))
    return kap, cnt.value


def eps_star(n, lo, hi, x, B0, ic, jc, a_r, op=MIMETIC, strict=True, bc=None):
    """Eqs. 3.5-3.7 on the grid line (ic, jc, .): returns (alpha*[nz], eps*)."""
    x, B0 = _arr(x, n), _arr(B0, n)
    al = np.empty(int(n[2]))
    e = C.c_double()
    with _bc(bc):
        _check(_lib.mro_eps_star(*_g(n, lo, hi), x, B0, int(op), int(ic), int(jc), float(a_r), _ptr(al), C.byref(e)), strict)
    return al, e.value


def sigma(n, lo, hi, x, B0, x_ref, B_ref, strict=True, bc=None):
    """Eqs. 3.8-3.9: returns (sigma_x, sigma_B)."""
    x, B0, x_ref, B_ref = _arr(x, n), _arr(B0, n), _arr(x_ref, n), _arr(B_ref, n)
    sx, sb = C.c_double(), C.c_double()
    with _bc(bc):
        _check(_lib.mro_sigma(*_g(n, lo, hi), x, B0, x_ref, B_ref, C.byref(sx), C.byref(sb)), strict)
    return sx.value, sb.value
