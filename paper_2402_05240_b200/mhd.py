"""Thin ctypes binding of libmhd.so (include/mhd.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; PyTorch is used for
device memory (the workspace tensor, device-resident input/output tensors) and streams.
There is no CPU fallback: importing this module raises if the library is missing, and every
call raises MhdError on a non-zero return code.
"""
import ctypes
import os

import numpy as np

from .inputs import FIELDS, field_shapes

_HERE = os.path.dirname(os.path.abspath(__file__))
# MHD_LIBRARY overrides the in-tree build (e.g. to compare two builds of the same ABI)
LIB_PATH = os.environ.get("MHD_LIBRARY") or os.path.join(_HERE, "libmhd.so")

RECON_PCM, RECON_PLMC, RECON_PPMC, RECON_PLMP, RECON_PPMP = 0, 1, 2, 3, 4
BC_PERIODIC, BC_OUTFLOW = 0, 1

_dp = ctypes.POINTER(ctypes.c_double)
_vp = ctypes.c_void_p


class MhdError(RuntimeError):
    pass


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            "%s not found: build it with `python -m paper_2402_05240_b200.build` "
            "(there is no CPU fallback)" % LIB_PATH)
    L = ctypes.CDLL(LIB_PATH)
    L.mhd_workspace_bytes.argtypes = [ctypes.c_int] * 4
    L.mhd_workspace_bytes.restype = ctypes.c_size_t
    L.mhd_init.argtypes = [ctypes.c_int] * 3 + [ctypes.c_double, ctypes.c_int]
    L.mhd_init_workspace.argtypes = [ctypes.c_int] * 3 + [ctypes.c_double, ctypes.c_int, _vp, ctypes.c_size_t]
    L.mhd_set_boundary.argtypes = [ctypes.c_int, ctypes.c_int]
    L.mhd_set_stream.argtypes = [_vp]
    L.mhd_set_domain.argtypes = [ctypes.c_double] * 3
    L.mhd_set_state.argtypes = [_dp] * 8
    L.mhd_set_state_device.argtypes = [_vp] * 8
    L.mhd_compute_dt.argtypes = [ctypes.c_double, _dp]
    L.mhd_step.argtypes = [ctypes.c_double]
    L.mhd_advance.argtypes = [ctypes.c_int, ctypes.c_double, _dp]
    L.mhd_get_state.argtypes = [_dp] * 8
    L.mhd_get_state_device.argtypes = [_vp] * 8
    L.mhd_get_half_state.argtypes = [_dp] * 8
    L.mhd_max_divb.argtypes = [_dp]
    L.mhd_get_flux.argtypes = [ctypes.c_int, ctypes.c_int, _dp]
    L.mhd_measure_peaks.argtypes = [_dp, _dp, ctypes.c_double]
    L.mhd_measure_peaks.restype = ctypes.c_int
    L.mhd_step_profile.argtypes = [ctypes.c_double, ctypes.c_int, _dp, ctypes.POINTER(ctypes.c_char_p),
                                   ctypes.POINTER(ctypes.c_int)]
    L.mhd_step_profile.restype = ctypes.c_int
    L.mhd_advance_profile.argtypes = [ctypes.c_int, ctypes.c_double, ctypes.c_int, _dp, ctypes.POINTER(ctypes.c_char_p),
                                      ctypes.POINTER(ctypes.c_int)]
    L.mhd_advance_profile.restype = ctypes.c_int
    L.mhd_unit_hlld.argtypes = [ctypes.c_int, ctypes.c_double, _dp, _dp, _dp, _dp]
    L.mhd_unit_reconstruct.argtypes = [ctypes.c_int, ctypes.c_double, ctypes.c_int, _dp, _dp, _dp, _dp]
    L.mhd_unit_ct_edge.argtypes = [ctypes.c_int, _dp, _dp]
    L.mhd_unit_math.argtypes = [ctypes.c_int, ctypes.c_int, _dp, _dp]
    L.mhd_debug_guard_errors.argtypes = [ctypes.POINTER(ctypes.c_longlong)]
    L.mhd_debug_guard_errors.restype = ctypes.c_int
    L.mhd_launch_count.restype = ctypes.c_longlong
    L.mhd_last_error.restype = ctypes.c_char_p
    L.mhd_max_divb_noalloc.argtypes = [ctypes.c_int] * 3 + [ctypes.c_double] * 3 + [_vp] * 5
    L.mhd_max_divb_noalloc.restype = ctypes.c_int
    L.mhd_noalloc_last_error.restype = ctypes.c_char_p
    for name in ("mhd_init", "mhd_init_workspace", "mhd_set_boundary", "mhd_set_domain", "mhd_set_stream", "mhd_set_state",
                 "mhd_set_state_device", "mhd_compute_dt", "mhd_step", "mhd_advance", "mhd_get_state",
                 "mhd_get_state_device", "mhd_get_half_state", "mhd_max_divb", "mhd_synchronize",
                 "mhd_finalize", "mhd_get_flux", "mhd_unit_hlld", "mhd_unit_reconstruct", "mhd_unit_ct_edge", "mhd_unit_math"):
        getattr(L, name).restype = ctypes.c_int
    return L


_lib = _load()


def lib():
    return _lib


def _check(rc):
    if rc != 0:
        raise MhdError("libmhd error %d: %s" % (rc, _lib.mhd_last_error().decode()))


def _hp(a):
    return a.ctypes.data_as(_dp)


NOALLOC_MAX_CELLS = 256 * 65536   # MHD_NOALLOC_MAX_CELLS of include/mhd.h


def max_divb_noalloc(n, d, bx, by, bz, out, stream=None):
    """mhd_max_divb_noalloc: max |div B| of dense DEVICE face arrays (torch tensors, ABI layout) into the
    one-element device tensor `out`, on `stream` (a torch.cuda.Stream; None = legacy default stream).
    Allocates nothing and does not synchronise; needs no Mhd context.  n = (nx, ny, nz), d = (dx, dy, dz)."""
    rc = _lib.mhd_max_divb_noalloc(int(n[0]), int(n[1]), int(n[2]), float(d[0]), float(d[1]), float(d[2]),
                                   _vp(bx.data_ptr()), _vp(by.data_ptr()), _vp(bz.data_ptr()), _vp(out.data_ptr()),
                                   _vp(stream.cuda_stream if stream is not None else 0))
    if rc != 0:
        raise MhdError("libmhd error %d: %s" % (rc, _lib.mhd_noalloc_last_error().decode()))


def measure_peaks(seconds=0.0):
    """(fp64 DFMA TFLOP/s, HBM copy GB/s) measured on the current device."""
    tf, bw = ctypes.c_double(), ctypes.c_double()
    _check(_lib.mhd_measure_peaks(ctypes.byref(tf), ctypes.byref(bw), float(seconds)))
    return tf.value, bw.value


def unit_hlld(gamma, WL, WR, bx):
    """n HLLD solves on the device: WL, WR (n,7), bx (n,) -> F (n,7)."""
    WL = np.ascontiguousarray(WL, dtype=np.float64).reshape(-1, 7)
    WR = np.ascontiguousarray(WR, dtype=np.float64).reshape(-1, 7)
    bx = np.ascontiguousarray(bx, dtype=np.float64).reshape(-1)
    n = WL.shape[0]
    if WR.shape[0] != n or bx.shape[0] != n:
        raise MhdError("unit_hlld: inconsistent lengths")
    F = np.empty((n, 7))
    _check(_lib.mhd_unit_hlld(n, float(gamma), _hp(WL), _hp(WR), _hp(bx), _hp(F)))
    return F


def unit_reconstruct(gamma, recon, Ws, bn0):
    """n reconstructions on the device: Ws (n, 2*recon+1, 7), bn0 (n,) -> (Wlo, Whi), (n,7) each."""
    radius = 1 if recon in (RECON_PLMC, RECON_PLMP) else 2
    Ws = np.ascontiguousarray(Ws, dtype=np.float64).reshape(-1, 2 * radius + 1, 7)
    bn0 = np.ascontiguousarray(bn0, dtype=np.float64).reshape(-1)
    n = Ws.shape[0]
    if bn0.shape[0] != n:
        raise MhdError("unit_reconstruct: inconsistent lengths")
    lo, hi = np.empty((n, 7)), np.empty((n, 7))
    _check(_lib.mhd_unit_reconstruct(n, float(gamma), int(recon), _hp(Ws), _hp(bn0), _hp(lo), _hp(hi)))
    return lo, hi


def unit_ct_edge(in12):
    """n CT edge fields on the device: in12 (n,12) in the argument order of mhd_unit_ct_edge."""
    in12 = np.ascontiguousarray(in12, dtype=np.float64).reshape(-1, 12)
    out = np.empty(in12.shape[0])
    _check(_lib.mhd_unit_ct_edge(in12.shape[0], _hp(in12), _hp(out)))
    return out


def unit_math(op, x):
    """The kernels' rcp (op 0), rsqrt (op 1), sqrt (op 2) on the device."""
    x = np.ascontiguousarray(x, dtype=np.float64).reshape(-1)
    y = np.empty_like(x)
    _check(_lib.mhd_unit_math(x.shape[0], int(op), _hp(x), _hp(y)))
    return y


class Mhd:
    """The single global context of libmhd.so, same call sequence as the C ABI."""

    def __init__(self, nx, ny, nz, gamma, recon=RECON_PLMC, bc=(0, 0, 0), use_torch_workspace=True,
                 stream=None, domain=(1.0, 1.0, 1.0)):
        import torch
        if not torch.cuda.is_available():
            raise MhdError("no CUDA device: the VL+CT step has no CPU fallback")
        self.n = (nx, ny, nz)
        self.recon = recon
        self._torch = torch
        self._ws = None
        if stream is not None:
            _check(_lib.mhd_set_stream(_vp(stream.cuda_stream)))
        else:
            _check(_lib.mhd_set_stream(None))
        if use_torch_workspace:
            nbytes = _lib.mhd_workspace_bytes(nx, ny, nz, recon)
            if nbytes == 0:
                raise MhdError("bad grid arguments")
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
            ptr = (self._ws.data_ptr() + 255) // 256 * 256
            _check(_lib.mhd_init_workspace(nx, ny, nz, float(gamma), int(recon), _vp(ptr), nbytes))
        else:
            _check(_lib.mhd_init(nx, ny, nz, float(gamma), int(recon)))
        for a, kind in enumerate(bc):
            _check(_lib.mhd_set_boundary(a, int(kind)))
        if tuple(domain) != (1.0, 1.0, 1.0):
            _check(_lib.mhd_set_domain(*[float(x) for x in domain]))

    # ---- host-buffer path -------------------------------------------------------------
    def set_state(self, state):
        sh = field_shapes(*self.n)
        arrs = []
        for f in FIELDS:
            a = np.ascontiguousarray(state[f], dtype=np.float64)
            if a.shape != sh[f]:
                raise MhdError("field %s has shape %s, expected %s" % (f, a.shape, sh[f]))
            arrs.append(a)
        _check(_lib.mhd_set_state(*[_hp(a) for a in arrs]))

    def _get_host(self, fn, out=None):
        sh = field_shapes(*self.n)
        if out is None:
            out = {f: np.empty(sh[f]) for f in FIELDS}
        _check(fn(*[_hp(out[f]) for f in FIELDS]))
        return out

    def get_state(self, out=None):
        return self._get_host(_lib.mhd_get_state, out)

    def get_half_state(self):
        return self._get_host(_lib.mhd_get_half_state)

    # ---- device-buffer path -----------------------------------------------------------
    def set_state_device(self, tensors):
        """tensors: dict of 8 contiguous float64 CUDA tensors in the ABI layout."""
        self._check_dev(tensors)
        _check(_lib.mhd_set_state_device(*[_vp(tensors[f].data_ptr()) for f in FIELDS]))

    def get_state_device(self, tensors):
        self._check_dev(tensors)
        _check(_lib.mhd_get_state_device(*[_vp(tensors[f].data_ptr()) for f in FIELDS]))
        return tensors

    def _check_dev(self, tensors):
        sh = field_shapes(*self.n)
        for f in FIELDS:
            t = tensors[f]
            if (not t.is_cuda or t.dtype != self._torch.float64 or not t.is_contiguous()
                    or tuple(t.shape) != sh[f]):
                raise MhdError("field %s: need a contiguous float64 CUDA tensor of shape %s" % (f, sh[f]))

    # ---- the hot path -----------------------------------------------------------------
    def compute_dt(self, cfl):
        dt = ctypes.c_double()
        _check(_lib.mhd_compute_dt(float(cfl), ctypes.byref(dt)))
        return dt.value

    def step(self, dt):
        _check(_lib.mhd_step(float(dt)))

    def advance(self, n_steps, cfl, want_time=False):
        if want_time:
            t = ctypes.c_double()
            _check(_lib.mhd_advance(int(n_steps), float(cfl), ctypes.byref(t)))
            return t.value
        _check(_lib.mhd_advance(int(n_steps), float(cfl), None))
        return None

    def step_profile(self, dt, max_entries=32):
        """One instrumented {CFL; step}: list of (kernel name, milliseconds)."""
        ms = (ctypes.c_double * max_entries)()
        names = (ctypes.c_char_p * max_entries)()
        n = ctypes.c_int()
        _check(_lib.mhd_step_profile(float(dt), max_entries, ms, names, ctypes.byref(n)))
        return [(names[i].decode(), ms[i]) for i in range(n.value)]

    def advance_profile(self, n_steps, cfl, max_entries=32):
        """n_steps instrumented steps of advance(), back to back: list of (kernel name, mean milliseconds)."""
        ms = (ctypes.c_double * max_entries)()
        names = (ctypes.c_char_p * max_entries)()
        n = ctypes.c_int()
        _check(_lib.mhd_advance_profile(int(n_steps), float(cfl), max_entries, ms, names, ctypes.byref(n)))
        return [(names[i].decode(), ms[i]) for i in range(n.value)]

    def get_flux(self, axis, comp):
        """Corrector flux component on the lower `axis`-faces of the active cells, shape (nz, ny, nx)."""
        out = np.empty((self.n[2], self.n[1], self.n[0]))
        _check(_lib.mhd_get_flux(int(axis), int(comp), _hp(out)))
        return out

    def guard_errors(self):
        """Damaged guard words of a context created with MHD_GUARD=1 (-1: not a guarded context)."""
        n = ctypes.c_longlong()
        _check(_lib.mhd_debug_guard_errors(ctypes.byref(n)))
        return n.value

    def max_divb(self):
        v = ctypes.c_double()
        _check(_lib.mhd_max_divb(ctypes.byref(v)))
        return v.value

    def launch_count(self):
        return int(_lib.mhd_launch_count())

    def synchronize(self):
        _check(_lib.mhd_synchronize())

    def close(self):
        _check(_lib.mhd_finalize())
        self._ws = None
