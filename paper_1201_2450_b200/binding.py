"""ctypes binding of libtnlm.so: same names as include/tnlm.h, argument marshalling only.

Stacks are torch CUDA tensors of dtype float32 and shape [n_phase][nz][ny][nx] (contiguous);
PyTorch provides device memory and streams, nothing else.  Every function raises TnlmError with
the library's message on a non-zero status.  The library must have been built
(``python -m paper_1201_2450_b200._build`` or ``__graft_entry__.build()``); a missing library is
an error, never a fallback.
"""
from __future__ import annotations

import ctypes as C
import os

VARIANT_AUTO, VARIANT_GENERIC, VARIANT_TILED, VARIANT_PAIRED, VARIANT_PAIRED_TMEM = 0, 1, 2, 3, 4

# every symbol include/tnlm.h declares
EXPORTS = ["tnlm_workspace_bytes", "tnlm_weights_bytes", "tnlm_weights", "tnlm_jacobi_step",
           "tnlm_jacobi_step_variant", "tnlm_enhance", "tnlm_enhance_variant", "tnlm_host_workspace_bytes",
           "tnlm_enhance_host", "tnlm_enhance_host_streams", "tnlm_jacobi_step_slab", "tnlm_jacobi_step_slab_variant", "tnlm_strerror",
           "tnlm_kernel_name", "tnlm_launches_per_sweep", "tnlm_z_tile", "tnlm_probe_fp32", "tnlm_probe_fp32_ffma_count",
           "tnlm_tv_diff", "tnlm_srr", "tnlm_srr_static", "tnlm_cnr",
           "tnlmr_workspace_bytes", "tnlmr_project", "tnlmr_backproject", "tnlmr_cgls", "tnlmr_reconstruct"]


class TnlmParams(C.Structure):
    """Mirror of ``tnlm_params`` (include/tnlm.h)."""
    _fields_ = [("n_phase", C.c_int32), ("nz", C.c_int32), ("ny", C.c_int32), ("nx", C.c_int32),
                ("patch_radius", C.c_int32), ("search_radius", C.c_int32), ("h", C.c_float), ("mu", C.c_float)]

    @classmethod
    def make(cls, shape, patch_radius, search_radius, h, mu):
        P, Z, Y, X = (int(v) for v in shape)
        return cls(P, Z, Y, X, int(patch_radius), int(search_radius), float(h), float(mu))

    @property
    def shape(self):
        return (self.n_phase, self.nz, self.ny, self.nx)


class TnlmError(RuntimeError):
    def __init__(self, code, what):
        self.code = int(code)
        super().__init__(f"{what}: tnlm status {code}: {strerror(code)}")


_LIB = None


def library_path() -> str:
    return os.path.join(os.path.dirname(os.path.abspath(__file__)), "libtnlm.so")


def lib():
    global _LIB
    if _LIB is None:
        path = library_path()
        if not os.path.exists(path):
            raise ImportError(f"{path} is missing: build it with `python -m paper_1201_2450_b200._build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(path)
        pp, vp, i32, sz = C.POINTER(TnlmParams), C.c_void_p, C.c_int32, C.c_size_t
        L.tnlm_workspace_bytes.argtypes = [pp]; L.tnlm_workspace_bytes.restype = sz
        L.tnlm_weights_bytes.argtypes = [pp]; L.tnlm_weights_bytes.restype = sz
        L.tnlm_host_workspace_bytes.argtypes = [pp]; L.tnlm_host_workspace_bytes.restype = sz
        L.tnlm_weights.argtypes = [pp, vp, vp, vp, sz, vp]
        L.tnlm_jacobi_step.argtypes = [pp, vp, vp, vp, vp, vp, sz, vp]
        L.tnlm_jacobi_step_variant.argtypes = [pp, vp, vp, vp, vp, vp, sz, vp, C.c_int]
        L.tnlm_jacobi_step_slab.argtypes = [pp, vp, vp, vp, vp, i32, i32, vp, sz, vp]
        L.tnlm_jacobi_step_slab_variant.argtypes = [pp, vp, vp, vp, vp, i32, i32, vp, sz, vp, C.c_int]
        L.tnlm_enhance.argtypes = [pp, vp, vp, vp, i32, vp, sz, vp]
        L.tnlm_enhance_variant.argtypes = [pp, vp, vp, vp, i32, vp, sz, vp, C.c_int]
        L.tnlm_enhance_host.argtypes = [pp, vp, vp, vp, i32, vp, sz, vp]
        L.tnlm_enhance_host_streams.argtypes = [pp, vp, vp, vp, i32, vp, sz, vp, vp]
        L.tnlm_strerror.argtypes = [C.c_int]; L.tnlm_strerror.restype = C.c_char_p
        L.tnlm_kernel_name.argtypes = [pp]; L.tnlm_kernel_name.restype = C.c_char_p
        L.tnlm_launches_per_sweep.argtypes = [pp]; L.tnlm_launches_per_sweep.restype = i32
        L.tnlm_z_tile.argtypes = [pp]; L.tnlm_z_tile.restype = i32
        gp = C.POINTER(TnlmrGeometry)
        L.tnlmr_workspace_bytes.argtypes = [gp, pp]; L.tnlmr_workspace_bytes.restype = C.c_size_t
        L.tnlmr_project.argtypes = [gp, vp, vp, vp, vp, C.c_size_t, vp]; L.tnlmr_project.restype = C.c_int
        L.tnlmr_backproject.argtypes = [gp, vp, vp, vp, vp, C.c_size_t, vp]; L.tnlmr_backproject.restype = C.c_int
        L.tnlmr_cgls.argtypes = [gp, vp, vp, vp, i32, vp, C.c_size_t, vp]; L.tnlmr_cgls.restype = C.c_int
        L.tnlmr_reconstruct.argtypes = [gp, pp, vp, vp, vp, vp, i32, i32, i32, vp, C.c_size_t, vp]; L.tnlmr_reconstruct.restype = C.c_int
        L.tnlm_tv_diff.argtypes = [pp, vp, vp, vp, vp]
        L.tnlm_srr.argtypes = [pp, vp, vp, vp, vp, vp, sz, vp]
        L.tnlm_srr_static.argtypes = [pp, vp, vp, vp, vp, vp]
        L.tnlm_cnr.argtypes = [pp, vp, i32, C.POINTER(C.c_int32), C.POINTER(C.c_int32), vp, vp]
        L.tnlm_probe_fp32.argtypes = [i32, vp, vp]
        L.tnlm_probe_fp32_ffma_count.argtypes = [i32]; L.tnlm_probe_fp32_ffma_count.restype = C.c_double
        _LIB = L
    return _LIB


def strerror(code) -> str:
    return lib().tnlm_strerror(int(code)).decode()


def _check(rc, what):
    if rc != 0:
        raise TnlmError(rc, what)


def workspace_bytes(p: TnlmParams) -> int:
    return int(lib().tnlm_workspace_bytes(C.byref(p)))


def weights_bytes(p: TnlmParams) -> int:
    return int(lib().tnlm_weights_bytes(C.byref(p)))


def host_workspace_bytes(p: TnlmParams) -> int:
    return int(lib().tnlm_host_workspace_bytes(C.byref(p)))


class TnlmrGeometry(C.Structure):
    """Mirror of ``tnlmr_geometry`` (include/tnlmr.h)."""
    _fields_ = [("n_phase", C.c_int32), ("nz", C.c_int32), ("ny", C.c_int32), ("nx", C.c_int32),
                ("n_view", C.c_int32), ("nv", C.c_int32), ("nu", C.c_int32),
                ("voxel", C.c_float), ("du", C.c_float), ("dv", C.c_float), ("sid", C.c_float), ("sdd", C.c_float)]

    @classmethod
    def make(cls, n_phase, vol_shape, n_view, nv, nu, voxel, du, dv, sid, sdd):
        nz, ny, nx = (int(v) for v in vol_shape)
        return cls(int(n_phase), nz, ny, nx, int(n_view), int(nv), int(nu), float(voxel), float(du), float(dv), float(sid), float(sdd))

    @property
    def vol_shape(self):
        return (self.n_phase, self.nz, self.ny, self.nx)

    @property
    def proj_shape(self):
        return (self.n_phase, self.n_view, self.nv, self.nu)


def _angles(g: TnlmrGeometry, angles):
    import numpy as np
    a = np.ascontiguousarray(angles, dtype=np.float64)
    if a.shape != (g.n_phase, g.n_view):
        raise TypeError(f"angles must have shape {(g.n_phase, g.n_view)}")
    return a


def _dev_like(t, shape, name):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and tuple(t.shape) == tuple(shape)):
        raise TypeError(f"{name} must be a contiguous float32 CUDA tensor of shape {tuple(shape)}")
    return t.data_ptr()


def tnlmr_workspace_bytes(g: TnlmrGeometry, p: TnlmParams = None) -> int:
    return int(lib().tnlmr_workspace_bytes(C.byref(g), None if p is None else C.byref(p)))


def tnlmr_project(g: TnlmrGeometry, angles, f, y=None, stream=None):
    """y = P f for every phase (include/tnlmr.h)."""
    import torch
    a = _angles(g, angles)
    with _Call(stream, f, y) as c:
        if y is None:
            y = torch.empty(g.proj_shape, dtype=torch.float32, device=f.device)
        ws = c.workspace(None, tnlmr_workspace_bytes(g))
        _check(lib().tnlmr_project(C.byref(g), a.ctypes.data, _dev_like(f, g.vol_shape, "f"), _dev_like(y, g.proj_shape, "y"),
                                   ws.data_ptr(), ws.numel(), c.handle), "tnlmr_project")
    return y


def tnlmr_backproject(g: TnlmrGeometry, angles, y, f=None, stream=None):
    """f = P^T y for every phase."""
    import torch
    a = _angles(g, angles)
    with _Call(stream, f, y) as c:
        if f is None:
            f = torch.empty(g.vol_shape, dtype=torch.float32, device=y.device)
        ws = c.workspace(None, tnlmr_workspace_bytes(g))
        _check(lib().tnlmr_backproject(C.byref(g), a.ctypes.data, _dev_like(y, g.proj_shape, "y"), _dev_like(f, g.vol_shape, "f"),
                                       ws.data_ptr(), ws.numel(), c.handle), "tnlmr_backproject")
    return f


def tnlmr_cgls(g: TnlmrGeometry, angles, y, x, n_iter, ws=None, stream=None):
    """n_iter CGLS iterations on ||P x - y||^2 per phase, x updated in place (and returned)."""
    a = _angles(g, angles)
    with _Call(stream, x, y, ws) as c:
        ws = c.workspace(ws, tnlmr_workspace_bytes(g))
        _check(lib().tnlmr_cgls(C.byref(g), a.ctypes.data, _dev_like(y, g.proj_shape, "y"), _dev_like(x, g.vol_shape, "x"), int(n_iter),
                                ws.data_ptr(), ws.numel(), c.handle), "tnlmr_cgls")
    return x


def tnlmr_reconstruct(g: TnlmrGeometry, p: TnlmParams, angles, y, f_init, n_outer, n_cgls, inner_start=0, f_out=None, ws=None,
                      stream=None):
    """TNLM-R: n_outer x {CGLS from f^(k-1); weights from g^(k); one sweep of Eq. 8; clamp}."""
    import torch
    a = _angles(g, angles)
    with _Call(stream, y, f_init, f_out, ws) as c:
        if f_out is None:
            f_out = torch.empty_like(f_init)
        ws = c.workspace(ws, tnlmr_workspace_bytes(g, p))
        _check(lib().tnlmr_reconstruct(C.byref(g), C.byref(p), a.ctypes.data, _dev_like(y, g.proj_shape, "y"),
                                       _dev_like(f_init, g.vol_shape, "f_init"), _dev_like(f_out, g.vol_shape, "f_out"), int(n_outer),
                                       int(n_cgls), int(inner_start), ws.data_ptr(), ws.numel(), c.handle), "tnlmr_reconstruct")
    return f_out


def z_tile(p: TnlmParams) -> int:
    """z-tile period of the sweep kernels for these parameters (include/tnlm.h: tnlm_z_tile)."""
    return int(lib().tnlm_z_tile(C.byref(p)))


def kernel_name(p: TnlmParams) -> str:
    return lib().tnlm_kernel_name(C.byref(p)).decode()


def launches_per_sweep(p: TnlmParams) -> int:
    return int(lib().tnlm_launches_per_sweep(C.byref(p)))


# ---- torch marshalling ------------------------------------------------------------------------
def _dev_ptr(t, p: TnlmParams, name, optional=False):
    if t is None:
        if optional:
            return None
        raise TnlmError(-1, f"{name} is None")
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name} must be a CUDA torch tensor (no CPU path exists)")
    if t.dtype != torch.float32 or not t.is_contiguous() or tuple(t.shape) != p.shape:
        raise TypeError(f"{name} must be contiguous float32 of shape {p.shape}, got {t.dtype} {tuple(t.shape)}")
    return t.data_ptr()


class _Call:
    """Context of one library call: the device all tensors live on is made current (the C ABI works on 'the
    current CUDA device'), the stream handle is resolved on it, and temporaries the binding allocated itself are
    tied to a non-current stream with record_stream so the caching allocator cannot reuse them while work is queued."""

    def __init__(self, stream, *tensors):
        import torch
        for t in tensors:
            if t is not None and not (isinstance(t, torch.Tensor) and t.is_cuda):
                raise TypeError("every tensor argument must be a CUDA torch tensor (no CPU path exists)")
        devs = {t.device for t in tensors if t is not None}
        if len(devs) > 1:
            raise TypeError(f"all tensors of a call must live on one CUDA device, got {sorted(str(d) for d in devs)}")
        self.device = devs.pop() if devs else torch.device("cuda", torch.cuda.current_device())
        self.guard = torch.cuda.device(self.device)
        self.stream_arg = stream
        self.temps = []

    def __enter__(self):
        import torch
        self.guard.__enter__()
        self.stream = torch.cuda.current_stream(self.device) if self.stream_arg is None else self.stream_arg
        return self

    def __exit__(self, *exc):
        import torch
        if self.stream != torch.cuda.current_stream(self.device):
            for t in self.temps:
                t.record_stream(self.stream)
        return self.guard.__exit__(*exc)

    @property
    def handle(self):
        return self.stream.cuda_stream

    def temp(self, *size, dtype):
        import torch
        t = torch.empty(*size, dtype=dtype, device=self.device)
        self.temps.append(t)
        return t

    def workspace(self, ws, need):
        import torch
        if ws is None:
            return self.temp(max(need, 16), dtype=torch.uint8)
        if not ws.is_cuda or ws.dtype != torch.uint8 or ws.device != self.device:
            raise TypeError(f"workspace must be a CUDA uint8 tensor on {self.device}")
        return ws


def tnlm_weights(p: TnlmParams, ref, w_out=None, stream=None):
    """Normalised weights w[p][s][k][z][y][x] of Eq. 3/9 (see include/tnlm.h)."""
    import torch
    n_t = (2 * p.search_radius + 1) ** 3
    with _Call(stream, ref, w_out) as c:
        if w_out is None:
            w_out = torch.empty((p.n_phase, 2, n_t, p.nz, p.ny, p.nx), dtype=torch.float32, device=c.device)
        _check(lib().tnlm_weights(C.byref(p), _dev_ptr(ref, p, "ref"), w_out.data_ptr(), None, 0, c.handle), "tnlm_weights")
    return w_out


def tnlm_jacobi_step(p: TnlmParams, f, g, ref=None, f_out=None, ws=None, stream=None, variant=VARIANT_AUTO):
    """One Gauss-Jacobi sweep of Eq. 8 (see include/tnlm.h)."""
    import torch
    with _Call(stream, f, g, ref, f_out, ws) as c:
        if f_out is None:
            f_out = torch.empty_like(f)
        ws = c.workspace(ws, workspace_bytes(p))
        _check(lib().tnlm_jacobi_step_variant(C.byref(p), _dev_ptr(f, p, "f"), _dev_ptr(g, p, "g"),
                                              _dev_ptr(ref, p, "ref", optional=True), _dev_ptr(f_out, p, "f_out"),
                                              ws.data_ptr(), ws.numel(), c.handle, int(variant)),
               "tnlm_jacobi_step")
    return f_out


def tnlm_jacobi_step_slab(p: TnlmParams, f, g, z_begin, z_end, ref=None, f_out=None, ws=None, stream=None,
                          variant=VARIANT_AUTO):
    import torch
    with _Call(stream, f, g, ref, f_out, ws) as c:
        if f_out is None:
            f_out = torch.empty_like(f)
        ws = c.workspace(ws, workspace_bytes(p))
        _check(lib().tnlm_jacobi_step_slab_variant(C.byref(p), _dev_ptr(f, p, "f"), _dev_ptr(g, p, "g"),
                                                   _dev_ptr(ref, p, "ref", optional=True), _dev_ptr(f_out, p, "f_out"),
                                                   int(z_begin), int(z_end), ws.data_ptr(), ws.numel(),
                                                   c.handle, int(variant)),
               "tnlm_jacobi_step_slab")
    return f_out


def tnlm_enhance(p: TnlmParams, g, n_iter, f_init=None, f_out=None, ws=None, stream=None, variant=VARIANT_AUTO):
    """TNLM-E: n_iter x {weights from f^k; one sweep} (see include/tnlm.h)."""
    import torch
    with _Call(stream, g, f_init, f_out, ws) as c:
        if f_out is None:
            f_out = torch.empty_like(g)
        ws = c.workspace(ws, workspace_bytes(p))
        _check(lib().tnlm_enhance_variant(C.byref(p), _dev_ptr(g, p, "g"), _dev_ptr(f_init, p, "f_init", optional=True),
                                          _dev_ptr(f_out, p, "f_out"), int(n_iter), ws.data_ptr(), ws.numel(),
                                          c.handle, int(variant)),
               "tnlm_enhance")
    return f_out


def tnlm_enhance_host(p: TnlmParams, g_host, n_iter, f_out_host=None, f_init_host=None, dev_ws=None, stream=None,
                      copy_stream=None):
    """End-to-end form with HOST tensors (pinned for asynchronous copies); returns the host result.
    copy_stream: a torch.cuda.Stream for the pipelined copies (default: the library makes one per call)."""
    import torch
    for name, t in (("g_host", g_host), ("f_init_host", f_init_host), ("f_out_host", f_out_host)):
        if t is not None and (t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous()
                              or tuple(t.shape) != p.shape):
            raise TypeError(f"{name} must be a contiguous float32 CPU tensor of shape {p.shape}")
    if f_out_host is None:
        f_out_host = torch.empty(p.shape, dtype=torch.float32, pin_memory=True)
    with _Call(stream, dev_ws) as c:
        dev_ws = c.workspace(dev_ws, host_workspace_bytes(p))
        _check(lib().tnlm_enhance_host_streams(C.byref(p), g_host.data_ptr(),
                                               None if f_init_host is None else f_init_host.data_ptr(),
                                               f_out_host.data_ptr(), int(n_iter), dev_ws.data_ptr(), dev_ws.numel(),
                                               c.handle, None if copy_stream is None else copy_stream.cuda_stream),
               "tnlm_enhance_host")                    # synchronises both streams before returning
    return f_out_host


def probe_fp32(n_iter: int, sink, stream=None) -> float:
    """Enqueue the FFMA probe; returns the number of FFMA lane-operations it executes."""
    with _Call(stream, sink) as c:
        _check(lib().tnlm_probe_fp32(int(n_iter), sink.data_ptr(), c.handle), "tnlm_probe_fp32")
    return float(lib().tnlm_probe_fp32_ffma_count(int(n_iter)))


def tnlm_tv_diff(p: TnlmParams, a, b=None, stream=None):
    """TV(a_p - b_p) per phase (Eq. 10's seminorm; see include/tnlm.h) -> float64 CUDA tensor [n_phase]."""
    import torch
    with _Call(stream, a, b) as c:
        out = torch.empty(p.n_phase, dtype=torch.float64, device=c.device)
        _check(lib().tnlm_tv_diff(C.byref(p), _dev_ptr(a, p, "a"), _dev_ptr(b, p, "b", optional=True), out.data_ptr(),
                                  c.handle), "tnlm_tv_diff")
    return out


def tnlm_srr(p: TnlmParams, f_fdk, f_enh, f_star, stream=None):
    """Streak-reduction ratio of Eq. 10 per phase -> float64 CUDA tensor [n_phase]."""
    import torch
    with _Call(stream, f_fdk, f_enh, f_star) as c:
        out = torch.empty(p.n_phase, dtype=torch.float64, device=c.device)
        ws = c.temp(2 * p.n_phase, dtype=torch.float64)
        _check(lib().tnlm_srr(C.byref(p), _dev_ptr(f_fdk, p, "f_fdk"), _dev_ptr(f_enh, p, "f_enh"),
                              _dev_ptr(f_star, p, "f_star"), out.data_ptr(), ws.data_ptr(), ws.numel() * 8,
                              c.handle), "tnlm_srr")
    return out


SRR_STATIC_MAX_PHASES = 64   # TNLM_SRR_STATIC_MAX_PHASES of include/tnlm.h


def tnlm_srr_static(p: TnlmParams, f_fdk, f_enh, f_star, out=None, stream=None):
    """tnlm_srr without a workspace: the library keeps the scratch in a static device array (n_phase <= 64), so
    the C call allocates nothing.  Pass `out` (float64 CUDA tensor [n_phase]) to keep this wrapper allocation-free
    too.  Calls that overlap on the GPU race on the shared scratch (include/tnlm.h)."""
    import torch
    with _Call(stream, f_fdk, f_enh, f_star, out) as c:
        if out is None:
            out = torch.empty(p.n_phase, dtype=torch.float64, device=c.device)
        elif not out.is_cuda or out.dtype != torch.float64 or not out.is_contiguous() or out.numel() != p.n_phase:
            raise TypeError(f"out must be a contiguous float64 CUDA tensor of {p.n_phase} elements")
        _check(lib().tnlm_srr_static(C.byref(p), _dev_ptr(f_fdk, p, "f_fdk"), _dev_ptr(f_enh, p, "f_enh"),
                                     _dev_ptr(f_star, p, "f_star"), out.data_ptr(), c.handle), "tnlm_srr_static")
    return out


def tnlm_cnr(p: TnlmParams, stack, phase, roi, roi_bg, stream=None):
    """[S, sigma, S_b, sigma_b, CNR] of two half-open boxes (z0, z1, y0, y1, x0, x1) of `phase`."""
    import torch
    r0 = (C.c_int32 * 6)(*[int(v) for v in roi])
    r1 = (C.c_int32 * 6)(*[int(v) for v in roi_bg])
    with _Call(stream, stack) as c:
        out = torch.empty(5, dtype=torch.float64, device=c.device)
        _check(lib().tnlm_cnr(C.byref(p), _dev_ptr(stack, p, "stack"), int(phase), r0, r1, out.data_ptr(),
                              c.handle), "tnlm_cnr")
    return out
