"""ctypes binding of oracle/liboracle.so (TEST INFRASTRUCTURE, NOT PRODUCT).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It shares nothing with paper_2402_05240_b200.
"""
import ctypes
import os
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
if _HERE not in sys.path:
    sys.path.insert(0, _HERE)
import build as _build  # noqa: E402  (oracle/build.py)

_lib = None
_dp = ctypes.POINTER(ctypes.c_double)
_d = ctypes.c_double


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = ctypes.CDLL(path)
        L.oracle_init.argtypes = [ctypes.c_int] * 3 + [_d, ctypes.c_int]
        L.oracle_set_boundary.argtypes = [ctypes.c_int, ctypes.c_int]
        L.oracle_set_domain.argtypes = [_d, _d, _d]
        L.oracle_set_state.argtypes = [_dp] * 8
        L.oracle_get_state.argtypes = [_dp] * 8
        L.oracle_get_half_state.argtypes = [_dp] * 8
        L.oracle_compute_dt.argtypes = [_d, _dp]
        L.oracle_step.argtypes = [_d]
        L.oracle_max_divb.argtypes = [_dp]
        L.oracle_get_flux.argtypes = [ctypes.c_int, ctypes.c_int, _dp]
        L.oracle_hlld.argtypes = [_d, _dp, _dp, _d, _dp]
        L.oracle_hlld.restype = None
        L.oracle_eigensystem.argtypes = [_d, _dp, _d, _dp, _dp, _dp]
        L.oracle_eigensystem.restype = None
        L.oracle_plmc.argtypes = [_d, _dp, _dp, _dp, _d, _dp, _dp]
        L.oracle_plmc.restype = None
        L.oracle_ppmc.argtypes = [_d, _dp, _d, _dp, _dp]
        L.oracle_plmp.argtypes = [_dp, _dp, _dp, _dp, _dp]
        L.oracle_ppmp.argtypes = [_dp, _dp, _dp]
        L.oracle_ppmc.restype = None
        L.oracle_ppm_scalar.argtypes = [_dp, _dp, _dp]
        L.oracle_ppm_scalar.restype = None
        L.oracle_ct_edge.argtypes = [_d] * 12
        L.oracle_ct_edge.restype = _d
        L.oracle_fast_speed.argtypes = [_d] * 6
        L.oracle_fast_speed.restype = _d
        L.oracle_phys_flux.argtypes = [_d, _dp, _d, _dp]
        L.oracle_phys_flux.restype = None
        L.oracle_num_threads.restype = ctypes.c_int
        L.oracle_set_guards.argtypes = [ctypes.c_int, ctypes.c_int]
        L.oracle_set_guards.restype = None
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(_dp)


def _vec(x, n):
    a = np.ascontiguousarray(np.asarray(x, dtype=np.float64).reshape(n))
    return a


# ---- unit-level entry points -------------------------------------------------
def hlld(gamma, WL, WR, bx):
    WL = _vec(WL, 7); WR = _vec(WR, 7); F = np.empty(7)
    lib().oracle_hlld(gamma, _p(WL), _p(WR), float(bx), _p(F))
    return F


def phys_flux(gamma, W, bx):
    W = _vec(W, 7); F = np.empty(7)
    lib().oracle_phys_flux(gamma, _p(W), float(bx), _p(F))
    return F


def eigensystem(gamma, W, bx):
    W = _vec(W, 7)
    lam = np.empty(7); L = np.empty(49); R = np.empty(49)
    lib().oracle_eigensystem(gamma, _p(W), float(bx), _p(lam), _p(L), _p(R))
    return lam, L.reshape(7, 7), R.reshape(7, 7)


def plmc(gamma, Wm, W0, Wp, bx0):
    Wm = _vec(Wm, 7); W0 = _vec(W0, 7); Wp = _vec(Wp, 7)
    lo = np.empty(7); hi = np.empty(7)
    lib().oracle_plmc(gamma, _p(Wm), _p(W0), _p(Wp), float(bx0), _p(lo), _p(hi))
    return lo, hi


def ppmc(gamma, Ws, bx0):
    Ws = _vec(Ws, 35)
    lo = np.empty(7); hi = np.empty(7)
    lib().oracle_ppmc(gamma, _p(Ws), float(bx0), _p(lo), _p(hi))
    return lo, hi


def plmp(Wm, W0, Wp):
    Wm = _vec(Wm, 7); W0 = _vec(W0, 7); Wp = _vec(Wp, 7)
    lo = np.empty(7); hi = np.empty(7)
    lib().oracle_plmp(_p(Wm), _p(W0), _p(Wp), _p(lo), _p(hi))
    return lo, hi


def ppmp(Ws):
    Ws = _vec(Ws, 35)
    lo = np.empty(7); hi = np.empty(7)
    lib().oracle_ppmp(_p(Ws), _p(lo), _p(hi))
    return lo, hi


def ppm_scalar(q):
    q = _vec(q, 5)
    lo = ctypes.c_double(); hi = ctypes.c_double()
    lib().oracle_ppm_scalar(_p(q), ctypes.byref(lo), ctypes.byref(hi))
    return lo.value, hi.value


def ct_edge(*args):
    assert len(args) == 12
    return lib().oracle_ct_edge(*[float(a) for a in args])


def fast_speed(gamma, rho, P, bn, bt1, bt2):
    return lib().oracle_fast_speed(gamma, rho, P, bn, bt1, bt2)


def set_guards(r6=True, r7=True):
    """Pin support only: switch the round-off guards of readings R6 / R7 (both on by default)."""
    lib().oracle_set_guards(int(bool(r6)), int(bool(r7)))


def num_threads():
    return lib().oracle_num_threads()


# ---- grid driver ---------------------------------------------------------------
FIELDS = ("rho", "mx", "my", "mz", "E", "bx", "by", "bz")


def field_shapes(nx, ny, nz):
    """numpy shapes (k, j, i) of the 8 host arrays of the C ABI (i fastest)."""
    s = {f: (nz, ny, nx) for f in FIELDS[:5]}
    s["bx"] = (nz, ny, nx + 1)
    s["by"] = (nz, ny + 1, nx)
    s["bz"] = (nz + 1, ny, nx)
    return s


class Oracle:
    """One global grid inside liboracle.so (same call sequence as the product ABI)."""

    def __init__(self, nx, ny, nz, gamma, recon, bc=(0, 0, 0), domain=(1.0, 1.0, 1.0)):
        self.n = (nx, ny, nz)
        rc = lib().oracle_init(nx, ny, nz, float(gamma), int(recon))
        if rc:
            raise RuntimeError("oracle_init failed: %d" % rc)
        if tuple(domain) != (1.0, 1.0, 1.0):
            if lib().oracle_set_domain(*[float(x) for x in domain]):
                raise RuntimeError("oracle_set_domain failed")
        for a, kind in enumerate(bc):
            lib().oracle_set_boundary(a, int(kind))

    def set_state(self, state):
        arrs = [np.ascontiguousarray(state[f], dtype=np.float64) for f in FIELDS]
        sh = field_shapes(*self.n)
        for f, a in zip(FIELDS, arrs):
            assert a.shape == sh[f], (f, a.shape, sh[f])
        rc = lib().oracle_set_state(*[_p(a) for a in arrs])
        if rc:
            raise RuntimeError("oracle_set_state failed: %d" % rc)

    def _get(self, fn):
        sh = field_shapes(*self.n)
        out = {f: np.empty(sh[f]) for f in FIELDS}
        rc = fn(*[_p(out[f]) for f in FIELDS])
        if rc:
            raise RuntimeError("oracle get failed: %d" % rc)
        return out

    def get_state(self):
        return self._get(lib().oracle_get_state)

    def get_half_state(self):
        return self._get(lib().oracle_get_half_state)

    def compute_dt(self, cfl):
        dt = ctypes.c_double()
        rc = lib().oracle_compute_dt(float(cfl), ctypes.byref(dt))
        if rc:
            raise RuntimeError("oracle_compute_dt failed: %d" % rc)
        return dt.value

    def step(self, dt):
        rc = lib().oracle_step(float(dt))
        if rc:
            raise RuntimeError("oracle_step failed: %d" % rc)

    def get_flux(self, axis, comp):
        nx, ny, nz = self.n
        out = np.empty((nz, ny, nx))
        rc = lib().oracle_get_flux(int(axis), int(comp), _p(out))
        if rc:
            raise RuntimeError("oracle_get_flux failed: %d" % rc)
        return out

    def max_divb(self):
        v = ctypes.c_double()
        lib().oracle_max_divb(ctypes.byref(v))
        return v.value

    def close(self):
        lib().oracle_finalize()
