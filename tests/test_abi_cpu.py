"""The C-ABI library loads and exports every symbol include/tnlm.h declares; argument errors are
detected synchronously.  No compute call is made here (this file runs without a GPU)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def T():
    from paper_1201_2450_b200 import _build
    _build.build()
    import paper_1201_2450_b200 as T
    T.lib()
    return T


def declared_symbols():
    """Every function include/*.h declares (tnlm.h: TNLM-E and metrics; tnlmr.h: TNLM-R)."""
    syms = set()
    for name in sorted(os.listdir(os.path.join(ROOT, "include"))):
        if name.endswith(".h"):
            text = open(os.path.join(ROOT, "include", name)).read()
            text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
            syms |= set(re.findall(r"\b(tnlmr?_[a-z0-9_]+)\s*\(", text))
    return sorted(syms)


def test_header_symbols_are_exported(T):
    syms = declared_symbols()
    assert len(syms) >= 14
    for s in syms:
        assert hasattr(T.lib(), s), f"{s} declared in include/*.h but not exported"
    assert sorted(T.EXPORTS) == syms


def test_params_struct_layout(T):
    assert C.sizeof(T.TnlmParams) == 32
    p = T.TnlmParams.make((10, 128, 256, 256), 1, 2, 0.05, 0.5)
    stack = 10 * 128 * 256 * 256 * 4
    assert T.workspace_bytes(p) >= stack
    assert T.weights_bytes(p) == 10 * 2 * 125 * 128 * 256 * 256 * 4
    assert T.host_workspace_bytes(p) >= 4 * stack
    assert T.launches_per_sweep(p) >= 1 and T.kernel_name(p) not in ("", "invalid")


def test_invalid_params_give_zero_sizes(T):
    bad = [((1, 4, 4, 4), 1, 1, 0.1, 1.0), ((2, 0, 4, 4), 1, 1, 0.1, 1.0), ((2, 4, 4, 4), -1, 1, 0.1, 1.0),
           ((2, 4, 4, 4), 1, 1, 0.0, 1.0), ((2, 4, 4, 4), 1, 1, 0.1, float("inf")), ((2, 4, 4, 4), 1, 1, float("nan"), 1.0),
           ((2, 4, 4, 4), 9, 1, 0.1, 1.0), ((2, 4, 4, 4), 1, 9, 0.1, 1.0), ((100, 1024, 1024, 1024), 1, 1, 0.1, 1.0)]
    for args in bad:
        p = T.TnlmParams.make(*args)
        assert T.workspace_bytes(p) == 0 and T.weights_bytes(p) == 0 and T.launches_per_sweep(p) == 0


def _call_step(T, p, f, g, ref, out, ws, ws_bytes):
    return T.lib().tnlm_jacobi_step(C.byref(p), f, g, ref, out, ws, ws_bytes, None)


def test_argument_errors_are_synchronous(T):
    """Fake (never dereferenced) device addresses: every path below returns before any launch."""
    L = T.lib()
    p = T.TnlmParams.make((3, 4, 8, 8), 1, 1, 0.1, 1.0)
    sb = 3 * 4 * 8 * 8 * 4
    wsb = T.workspace_bytes(p)
    A, B, Cc, D, W = 0x10000, 0x20000, 0x30000, 0x40000, 0x50000
    assert L.tnlm_jacobi_step(None, A, B, None, D, W, wsb, None) == -1
    assert _call_step(T, p, None, B, None, D, W, wsb) == -1
    assert _call_step(T, p, A, B, None, None, W, wsb) == -1
    assert _call_step(T, p, A, B, None, A, W, wsb) == -5                      # f_out == f
    assert _call_step(T, p, A, B, None, B + 16, W, wsb) == -5                 # overlaps g
    assert _call_step(T, p, A, B, Cc, Cc + sb - 16, W + 0x10000, wsb) == -5   # overlaps ref
    assert _call_step(T, p, A, B, None, D, None, wsb) == -6
    assert _call_step(T, p, A, B, None, D, W, wsb - 1) == -6
    assert _call_step(T, p, A, B, None, D, W + 4, wsb) == -6                  # misaligned workspace
    assert _call_step(T, p, A + 4, B, None, D, W, wsb) == -6                  # misaligned stack
    assert _call_step(T, p, A, B, None, D, D, wsb) == -5                      # workspace overlaps f_out
    bad = T.TnlmParams.make((1, 4, 8, 8), 1, 1, 0.1, 1.0)
    assert _call_step(T, bad, A, B, None, D, W, wsb) == -2
    bad = T.TnlmParams.make((3, 4, 8, 8), 1, 1, -0.1, 1.0)
    assert _call_step(T, bad, A, B, None, D, W, wsb) == -3
    bad = T.TnlmParams.make((3, 4, 8, 8), 4, 1, 0.1, 1.0)
    assert _call_step(T, bad, A, B, None, D, W, wsb) == -4
    assert L.tnlm_jacobi_step_variant(C.byref(p), A, B, None, D, W, wsb, None, 77) == -4
    assert L.tnlm_enhance(C.byref(p), A, None, D, -1, W, wsb, None) == -3
    assert L.tnlm_enhance(C.byref(p), A, None, A, 2, W, wsb, None) == -5
    assert L.tnlm_enhance(C.byref(p), A, B, B, 2, W, wsb, None) == -5
    assert L.tnlm_enhance(C.byref(p), None, None, D, 2, W, wsb, None) == -1
    assert L.tnlm_jacobi_step_slab(C.byref(p), A, B, None, D, 3, 2, W, wsb, None) == -2
    assert L.tnlm_jacobi_step_slab(C.byref(p), A, B, None, D, 0, 5, W, wsb, None) == -2
    assert L.tnlm_weights(C.byref(p), None, D, None, 0, None) == -1
    assert L.tnlm_enhance_host(C.byref(p), A, None, D, 1, W, 16, None) == -6
    assert L.tnlm_probe_fp32(1, None, None) == -1
    # tnlm_srr_static: argument errors come before any CUDA call, the phase limit has its own code
    big = T.TnlmParams.make((65, 2, 4, 4), 1, 1, 0.1, 1.0)
    assert L.tnlm_srr_static(C.byref(big), A, B, A, D, None) == -8
    assert L.tnlm_srr_static(C.byref(p), A, B, None, D, None) == -1
    assert L.tnlm_srr_static(C.byref(p), A, B, A, D + 4, None) == -6
    for code in range(0, -9, -1):
        assert T.strerror(code) not in ("", "unknown tnlm status")


def test_binding_refuses_cpu_tensors(T):
    import torch
    p = T.TnlmParams.make((2, 2, 4, 4), 1, 1, 0.1, 1.0)
    x = torch.zeros(p.shape)
    with pytest.raises(TypeError):
        T.tnlm_jacobi_step(p, x, x, ws=torch.zeros(16, dtype=torch.uint8))


def test_product_package_does_not_import_oracle():
    """The product path may not route through the oracle (tier rule 3)."""
    pkg = os.path.join(ROOT, "paper_1201_2450_b200")
    banned = ("tnlm_ref_", "libtnlm_oracle", "import oracle", "from oracle", "tnlm_oracle")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                for b in banned:
                    assert b not in text, f"{fn} mentions {b}"


def test_tnlmr_argument_errors_are_synchronous(T):
    """include/tnlmr.h: geometry and pointer errors come back as negative codes without touching a device."""
    g = T.TnlmrGeometry.make(2, (8, 8, 8), 3, 6, 6, 1.0, 1.5, 1.5, 30.0, 45.0)
    p = T.TnlmParams.make((2, 8, 8, 8), 1, 1, 0.1, 0.5)
    assert T.tnlmr_workspace_bytes(g) > 0 and T.tnlmr_workspace_bytes(g, p) > T.tnlmr_workspace_bytes(g)
    assert T.tnlmr_workspace_bytes(g, T.TnlmParams.make((3, 8, 8, 8), 1, 1, 0.1, 0.5)) == 0          # stack shapes differ
    bad = T.TnlmrGeometry.make(2, (8, 8, 8), 3, 6, 6, 1.0, 1.5, 1.5, 4.0, 45.0)                      # source inside the volume
    assert T.tnlmr_workspace_bytes(bad) == 0
    L = T.lib()
    ang = (C.c_double * 6)(*[0.1 * k for k in range(6)])
    fake = 0x1000
    assert L.tnlmr_project(C.byref(g), ang, None, fake, fake, 1 << 20, None) == -1                   # NULL volume
    assert L.tnlmr_project(C.byref(bad), ang, fake, fake, fake, 1 << 20, None) == -3                 # bad geometry
    assert L.tnlmr_cgls(C.byref(g), ang, fake, 0x100000, -1, 0x200000, 1 << 30, None) == -3          # negative iteration count
    assert L.tnlmr_cgls(C.byref(g), ang, fake, 0x100000, 1, 0x200000, 16, None) == -6                # workspace too small
    assert L.tnlmr_reconstruct(C.byref(g), C.byref(p), ang, fake, 0x100000, 0x100000, 1, 1, 0, 0x4000000, 1 << 30, None) == -5   # f_out aliases f_init
    assert L.tnlmr_reconstruct(C.byref(g), C.byref(p), ang, fake, 0x100000, 0x200000, 1, 1, 7, 0x4000000, 1 << 30, None) == -3   # bad inner_start
