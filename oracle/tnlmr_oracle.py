"""ctypes front end of the TNLM-R oracle (oracle/tnlmr_oracle.c) and the TNLM-R loop.  TEST INFRASTRUCTURE ONLY.

The projector pair and CGLS are computed by the C file (fp64).  The loop of PAPER.md:191-200 is composed here from
those and from the TNLM sweep of oracle/tnlm_oracle.c:

    for k = 1..n_outer:
        g_i^(k) = CGLS(P_i, y_i; start f_i^(k-1), n_cgls iterations)   for every phase      (step 1)
        weights from g^(k)                                                                  (step 2, Eq. 9)
        f^(k)   = one sweep of Eq. 8 with g = g^(k)                                         (step 3)
        f^(k)   = max(f^(k), 0)                                                             (step 4)

Reading R1: the single sweep of step 3 starts from f^(l=0) = g^(k), as TNLM-E starts from g
(PAPER.md:206), so it averages the neighbouring phases of g^(k): sweep(f = g^(k), g = g^(k), ref = g^(k)).
`inner_start="previous"` gives the other reading, sweep(f = f^(k-1), g = g^(k), ref = g^(k)).
Iterates are rounded to fp32 where they cross the C ABI of the product (after CGLS and after the sweep).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import tnlm_oracle as O
from .build_oracle import build_r


class RefGeom(C.Structure):
    _fields_ = [("n_view", C.c_int32), ("nu", C.c_int32), ("nv", C.c_int32),
                ("nz", C.c_int32), ("ny", C.c_int32), ("nx", C.c_int32),
                ("du", C.c_double), ("dv", C.c_double), ("sid", C.c_double), ("sdd", C.c_double), ("voxel", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build_r())
        gp, vp = C.POINTER(RefGeom), C.c_void_p
        L.tnlmr_ref_project.argtypes = [gp, vp, vp, vp]
        L.tnlmr_ref_backproject.argtypes = [gp, vp, vp, vp]
        L.tnlmr_ref_cgls.argtypes = [gp, vp, vp, vp, C.c_int32, vp]
        L.tnlmr_ref_ray.argtypes = [gp, vp, vp, vp, vp, C.c_int32]
        L.tnlmr_ref_ray_endpoints.argtypes = [gp, C.c_double, C.c_int32, C.c_int32, vp, vp]
        L.tnlmr_ref_ray_endpoints.restype = None
        _lib = L
    return _lib


def geom(vol_shape, n_view, nu, nv, du, dv, sid, sdd, voxel):
    nz, ny, nx = (int(v) for v in vol_shape)
    return RefGeom(int(n_view), int(nu), int(nv), nz, ny, nx, float(du), float(dv), float(sid), float(sdd), float(voxel))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def project(g: RefGeom, angles, f):
    """y[view][v][u] = P f for one phase (fp64)."""
    angles, f = _f64(angles), _f64(f)
    assert angles.shape == (g.n_view,) and f.shape == (g.nz, g.ny, g.nx)
    y = np.empty((g.n_view, g.nv, g.nu), dtype=np.float64)
    if lib().tnlmr_ref_project(C.byref(g), angles.ctypes.data, f.ctypes.data, y.ctypes.data):
        raise RuntimeError("oracle project failed")
    return y


def backproject(g: RefGeom, angles, y):
    """f = P^T y for one phase (fp64)."""
    angles, y = _f64(angles), _f64(y)
    assert angles.shape == (g.n_view,) and y.shape == (g.n_view, g.nv, g.nu)
    f = np.empty((g.nz, g.ny, g.nx), dtype=np.float64)
    if lib().tnlmr_ref_backproject(C.byref(g), angles.ctypes.data, y.ctypes.data, f.ctypes.data):
        raise RuntimeError("oracle backproject failed")
    return f


def cgls(g: RefGeom, angles, y, x0, n_iter, residuals=False):
    """n_iter CGLS iterations on ||P x - y||^2 from x0 (fp64); optionally the ||P^T r|| history."""
    angles, y = _f64(angles), _f64(y)
    x = _f64(x0).copy()
    res = np.zeros(int(n_iter) + 1, dtype=np.float64)
    if lib().tnlmr_ref_cgls(C.byref(g), angles.ctypes.data, y.ctypes.data, x.ctypes.data, int(n_iter), res.ctypes.data):
        raise RuntimeError("oracle cgls failed")
    return (x, res) if residuals else x


def ray(g: RefGeom, S, D):
    """(voxel indices, intersection lengths) of the ray from S to D."""
    S, D = _f64(S), _f64(D)
    cap = g.nx + g.ny + g.nz + 8
    vox, ln = np.zeros(cap, dtype=np.int64), np.zeros(cap, dtype=np.float64)
    n = lib().tnlmr_ref_ray(C.byref(g), S.ctypes.data, D.ctypes.data, vox.ctypes.data, ln.ctypes.data, cap)
    if n < 0:
        raise RuntimeError("oracle ray failed")
    return vox[:n], ln[:n]


def ray_endpoints(g: RefGeom, theta, iu, iv):
    S, D = np.zeros(3), np.zeros(3)
    lib().tnlmr_ref_ray_endpoints(C.byref(g), float(theta), int(iu), int(iv), S.ctypes.data, D.ctypes.data)
    return S, D


def reconstruct(g: RefGeom, angles, y, f_init, d, M, h, mu, n_outer, n_cgls, inner_start="g", history=False):
    """TNLM-R.  angles [P][n_view], y [P][n_view][nv][nu], f_init [P][nz][ny][nx] (fp32 in, fp32 out)."""
    angles = _f64(angles)
    y = np.ascontiguousarray(y, dtype=np.float32)
    f = np.ascontiguousarray(f_init, dtype=np.float32).copy()
    P = f.shape[0]
    hist = []
    for _ in range(int(n_outer)):
        gk = np.empty_like(f)
        for i in range(P):                                         # step 1, phase by phase
            gk[i] = cgls(g, angles[i], y[i], f[i], n_cgls).astype(np.float32)
        start = gk if inner_start == "g" else f                    # reading R1
        f = O.jacobi_step(start, gk, d, M, np.float32(h), np.float32(mu), ref=gk)   # steps 2-3
        f = np.maximum(f, np.float32(0.0))                         # step 4
        if history:
            hist.append((gk, f.copy()))
    return (f, hist) if history else f
