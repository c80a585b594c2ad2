"""ctypes front end of the CPU oracle (oracle/tnlm_oracle.c).  TEST INFRASTRUCTURE ONLY.

Marshals numpy arrays; every number is computed by the C file.  Citations of the
equations live in tnlm_oracle.c.  Not imported by the product package.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build_oracle import build


class RefParams(C.Structure):
    _fields_ = [("n_phase", C.c_int32), ("nz", C.c_int32), ("ny", C.c_int32), ("nx", C.c_int32),
                ("patch_radius", C.c_int32), ("search_radius", C.c_int32),
                ("h", C.c_double), ("mu", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        pp = C.POINTER(RefParams)
        vp = C.c_void_p
        L.tnlm_ref_weights_f64.argtypes = [pp, vp, vp]
        L.tnlm_ref_weights.argtypes = [pp, vp, vp]
        L.tnlm_ref_nlm_f64.argtypes = [pp, vp, vp, C.c_int, vp]
        L.tnlm_ref_jacobi_step_f64.argtypes = [pp, vp, vp, vp, vp]
        L.tnlm_ref_jacobi_step.argtypes = [pp, vp, vp, vp, vp]
        L.tnlm_ref_sweep_with_weights_f64.argtypes = [pp, vp, vp, vp, vp]
        L.tnlm_ref_jacobi_step_at.argtypes = [pp, vp, vp, vp, C.c_int64, vp, vp]
        L.tnlm_ref_enhance.argtypes = [pp, vp, vp, vp, C.c_int32]
        L.tnlm_ref_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _params(shape, d, M, h, mu):
    P, Z, Y, X = (int(v) for v in shape)
    return RefParams(P, Z, Y, X, int(d), int(M), float(h), float(mu))


def _ptr(a):
    return None if a is None else a.ctypes.data


def _chk(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


def _as(a, dtype):
    if a is None:
        return None
    a = np.ascontiguousarray(a, dtype=dtype)
    assert a.ndim == 4, "stack must be [phase][z][y][x]"
    return a


def n_offsets(M):
    return (2 * M + 1) ** 3


def weights(ref, d, M, h):
    """Normalised weights w[p][s][k][z][y][x] (fp64). fp32 or fp64 ``ref`` accepted."""
    f64 = np.asarray(ref).dtype == np.float64
    ref = _as(ref, np.float64 if f64 else np.float32)
    P, Z, Y, X = ref.shape
    out = np.empty((P, 2, n_offsets(M), Z, Y, X), dtype=np.float64)
    p = _params(ref.shape, d, M, h, 1.0)
    fn = lib().tnlm_ref_weights_f64 if f64 else lib().tnlm_ref_weights
    _chk(fn(C.byref(p), _ptr(ref), _ptr(out)), "weights")
    return out


def nlm_f64(f, ref, d, M, h, direction):
    f = _as(f, np.float64)
    ref = _as(ref, np.float64)
    out = np.empty_like(f)
    p = _params(f.shape, d, M, h, 1.0)
    _chk(lib().tnlm_ref_nlm_f64(C.byref(p), _ptr(f), _ptr(ref), int(direction), _ptr(out)), "nlm")
    return out


def jacobi_step_f64(f, g, d, M, h, mu, ref=None):
    f = _as(f, np.float64)
    g = _as(g, np.float64)
    ref = _as(ref, np.float64)
    out = np.empty_like(f)
    p = _params(f.shape, d, M, h, mu)
    _chk(lib().tnlm_ref_jacobi_step_f64(C.byref(p), _ptr(f), _ptr(g), _ptr(ref), _ptr(out)), "jacobi_step_f64")
    return out


def sweep_with_weights_f64(f, g, w, M, mu):
    """Eq. 8 with given weights w[p][s][k][z][y][x] (fp64)."""
    f = _as(f, np.float64)
    g = _as(g, np.float64)
    w = np.ascontiguousarray(w, dtype=np.float64)
    assert w.shape == (f.shape[0], 2, n_offsets(M)) + f.shape[1:]
    out = np.empty_like(f)
    p = _params(f.shape, 0, M, 1.0, mu)
    _chk(lib().tnlm_ref_sweep_with_weights_f64(C.byref(p), _ptr(f), _ptr(g), _ptr(w), _ptr(out)), "sweep_with_weights")
    return out


def jacobi_step(f, g, d, M, h, mu, ref=None):
    f = _as(f, np.float32)
    g = _as(g, np.float32)
    ref = _as(ref, np.float32)
    out = np.empty_like(f)
    p = _params(f.shape, d, M, h, mu)
    _chk(lib().tnlm_ref_jacobi_step(C.byref(p), _ptr(f), _ptr(g), _ptr(ref), _ptr(out)), "jacobi_step")
    return out


def jacobi_step_at(f, g, d, M, h, mu, idx, ref=None):
    """Eq. 8 at flat output indices ``idx`` (int64) of the [P][Z][Y][X] stack -> fp32."""
    f = _as(f, np.float32)
    g = _as(g, np.float32)
    ref = _as(ref, np.float32)
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    out = np.empty(idx.shape, dtype=np.float32)
    p = _params(f.shape, d, M, h, mu)
    _chk(lib().tnlm_ref_jacobi_step_at(C.byref(p), _ptr(f), _ptr(g), _ptr(ref), idx.size, _ptr(idx), _ptr(out)),
         "jacobi_step_at")
    return out


def enhance(g, d, M, h, mu, n_iter, f_init=None):
    g = _as(g, np.float32)
    f_init = _as(f_init, np.float32)
    out = np.empty_like(g)
    p = _params(g.shape, d, M, h, mu)
    _chk(lib().tnlm_ref_enhance(C.byref(p), _ptr(g), _ptr(f_init), _ptr(out), int(n_iter)), "enhance")
    return out


def num_threads():
    return int(lib().tnlm_ref_num_threads())
