"""Parity of the TNLM-R path (include/tnlmr.h) with its oracle (oracle/tnlmr_oracle.py), through the C ABI.

Tolerances.  The projector pair keeps the plane-crossing parameters in fp64 and rounds each
intersection length to fp32 once, so a length carries 6e-8 of relative error; the forward projection sums ~10^2 of them
in fp32, the transpose and the dot products of CGLS add a few hundred to a million fp32 terms with atomics (order not
fixed).  Bars: projector and back-projector max|d| <= 2e-5 max|.| and relative L2 <= 1e-5 (measured 6e-7 / 2e-6);
CGLS and the TNLM-R loop the north-star bar of the sweep itself, max|d| <= 1e-4 of the dynamic range and relative
L2 <= 1e-5 (measured 7e-7 / 6e-7 after 8 CGLS iterations: fp32 storage of x, r, s, p, q against the fp64 oracle).
"""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from tnlm_inputs import projections as PJ   # noqa: E402

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def T():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a GPU")
    import paper_1201_2450_b200 as T_
    T_.lib()
    return T_


@pytest.fixture(scope="module")
def R():
    from oracle import tnlmr_oracle as R_
    R_.lib()
    return R_


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def geoms(T, R, P, vol, n_view, nv, nu, voxel, du, dv, sid, sdd):
    """The same geometry for both sides: tnlmr_geometry carries fp32 lengths, so the oracle gets the fp32-rounded values."""
    voxel, du, dv, sid, sdd = (float(np.float32(v)) for v in (voxel, du, dv, sid, sdd))
    return (T.TnlmrGeometry.make(P, vol, n_view, nv, nu, voxel, du, dv, sid, sdd),
            R.geom(vol, n_view, nu, nv, du, dv, sid, sdd, voxel))


def rel(got, want):
    got, want = np.asarray(got, dtype=np.float64), np.asarray(want, dtype=np.float64)
    return np.abs(got - want).max() / max(np.abs(want).max(), 1e-30), np.linalg.norm(got - want) / max(np.linalg.norm(want), 1e-30)


# A ray that runs exactly inside a grid plane (central detector column / row at an axis-aligned view of an even-sized
# volume) has its length attributed to either of the two voxels it separates: both are Siddon's answer.  The cases
# keep such measure-zero rays out (even detector extent where the volume extent is even) and still hold axis-aligned
# views, i.e. rays parallel to grid planes.
CASES = [
    # P, volume (nz, ny, nx), views, nv, nu, voxel, du, dv, sid, sdd
    (2, (12, 20, 28), 5, 18, 24, 0.8, 1.3, 1.1, 60.0, 95.0),          # ragged, off-square
    (3, (33, 32, 32), 4, 40, 48, 0.8, 1.0, 1.0, 100.0, 153.6),        # paper-like magnification
    (1, (1, 9, 9), 7, 1, 30, 1.0, 0.9, 2.0, 20.0, 33.0),              # a single slice and detector row (fan beam)
    (2, (16, 16, 16), 3, 64, 64, 1.0, 0.2, 0.2, 40.0, 60.0),          # detector much finer than the voxels
]


@pytest.mark.parametrize("case", CASES)
def test_projector_pair_matches_the_oracle(T, R, case):
    P, vol, n_view, nv, nu = case[:5]
    g, rg = geoms(T, R, *case)
    rng = np.random.default_rng(4)
    ang = rng.uniform(0, 2 * np.pi, (P, n_view))
    ang[0, 0] = 0.0                                       # axis-aligned view: rays parallel to grid planes
    if n_view > 1:
        ang[0, 1] = np.pi / 2
    f = rng.random((P,) + vol).astype(np.float32)
    y = rng.standard_normal((P, n_view, nv, nu)).astype(np.float32)
    got_y = T.tnlmr_project(g, ang, dev(f)).cpu().numpy()
    got_f = T.tnlmr_backproject(g, ang, dev(y)).cpu().numpy()
    for i in range(P):
        m, l2 = rel(got_y[i], R.project(rg, ang[i], f[i]))
        assert m <= 2e-5 and l2 <= 1e-5, f"project phase {i}: {m:.2e} {l2:.2e}"
        m, l2 = rel(got_f[i], R.backproject(rg, ang[i], y[i]))
        assert m <= 2e-5 and l2 <= 1e-5, f"backproject phase {i}: {m:.2e} {l2:.2e}"
    # adjointness of the GPU pair itself, in fp64 on the host
    lhs = (got_y.astype(np.float64) * y).sum()
    rhs = (got_f.astype(np.float64) * f).sum()
    assert abs(lhs - rhs) <= 1e-5 * max(abs(lhs), 1.0)


def test_projection_misses_and_edges(T, R):
    # a detector far wider than the volume's shadow: most rays miss; constant volume -> chord of the box
    g, rg = geoms(T, R, 1, (6, 8, 10), 3, 31, 41, 0.7, 1.5, 1.5, 40.0, 70.0)
    ang = np.array([[0.3, 2.0, 4.4]])
    got = T.tnlmr_project(g, ang, dev(np.full((1, 6, 8, 10), 2.5))).cpu().numpy()[0]
    want = R.project(rg, ang[0], np.full((6, 8, 10), 2.5))
    assert (want == 0).sum() > want.size // 3
    assert np.abs(got - want).max() <= 2e-5 * want.max()
    assert (got[want == 0] == 0).all()


@pytest.mark.parametrize("n_iter", [0, 1, 4])
def test_cgls_matches_the_oracle(T, R, n_iter):
    P, vol = 2, (10, 14, 14)
    g, rg = geoms(T, R, P, vol, 6, 18, 20, 1.0, 1.2, 1.2, 50.0, 80.0)
    rng = np.random.default_rng(6)
    ang = PJ.phase_angles(P, 6)
    x0 = rng.random((P,) + vol).astype(np.float32)
    y = (5 * rng.random((P, 6, 18, 20))).astype(np.float32)
    got = T.tnlmr_cgls(g, ang, dev(y), dev(x0), n_iter).cpu().numpy()
    span = float(x0.max() - x0.min())
    for i in range(P):
        want = R.cgls(rg, ang[i], y[i], x0[i], n_iter)
        if n_iter == 0:
            assert np.array_equal(got[i], x0[i])
        else:
            d = np.abs(got[i] - want).max()
            l2 = np.linalg.norm(got[i] - want) / np.linalg.norm(want)
            assert d <= 1e-4 * max(span, float(np.abs(want).max())) and l2 <= 1e-5, f"{d:.2e} {l2:.2e}"


@pytest.mark.parametrize("inner_start", [0, 1])
def test_tnlmr_loop_matches_the_oracle(T, R, inner_start):
    # a small phantom study: analytic projections of the moving-tumour thorax, few views per phase, start from zero
    P = 4
    geom = PJ.paper_geometry(24, 6, 40)
    ang, y, clean = PJ.make_projection_stack(geom, P, noise=0.01, seed=3)
    g, rg = geoms(T, R, P, geom.vol_shape, geom.n_view, geom.nv, geom.nu, geom.voxel, geom.du, geom.dv, geom.sid, geom.sdd)
    d, M, h, mu, n_outer, n_cgls = 1, 2, 0.05, 0.5, 3, 3
    p = T.TnlmParams.make((P,) + geom.vol_shape, d, M, h, mu)
    f0 = np.zeros((P,) + geom.vol_shape, dtype=np.float32)
    got = T.tnlmr_reconstruct(g, p, ang, dev(y), dev(f0), n_outer, n_cgls, inner_start=inner_start).cpu().numpy()
    want = R.reconstruct(rg, ang, y, f0, d, M, h, mu, n_outer, n_cgls, inner_start="g" if inner_start == 0 else "previous")
    span = float(want.max() - want.min())
    dmax = np.abs(got - want).max()
    l2 = np.linalg.norm(got - want) / np.linalg.norm(want)
    assert got.min() >= 0.0
    assert dmax <= 1e-4 * span and l2 <= 1e-5, f"{dmax / span:.2e} {l2:.2e}"
    # n_outer = 0 copies the start
    same = T.tnlmr_reconstruct(g, p, ang, dev(y), dev(clean), 0, n_cgls).cpu().numpy()
    assert np.array_equal(same, clean)
    # reading R1: the reconstruction ends closer to the phantom than the same number of CGLS iterations alone (the
    # temporal regulariser suppresses the few-view streaks, the direction of PAPER.md:327).  The other reading averages
    # f^(k-1), which from a zero start (no FDK here) shrinks the first iterates, so it is only held to parity.
    if inner_start == 0:
        only_cgls = T.tnlmr_cgls(g, ang, dev(y), dev(f0), n_outer * n_cgls).cpu().numpy()
        assert np.linalg.norm(got - clean) < np.linalg.norm(only_cgls - clean)


def test_projector_pair_at_the_papers_geometry(T, R):
    """One phase at PAPER.md:245's size (128^3 voxels of 0.2 cm, 30 views, 512 x 512 pixels, 100 / 153.6 cm): the launch
    shape bench.py --tnlmr times, every ray and every voxel against the oracle."""
    geom = PJ.paper_geometry(128, 30, 512)
    g, rg = geoms(T, R, 1, geom.vol_shape, geom.n_view, geom.nv, geom.nu, geom.voxel, geom.du, geom.dv, geom.sid, geom.sdd)
    rng = np.random.default_rng(12)
    ang = PJ.phase_angles(10, 30)[3:4]
    f = rng.random((1,) + geom.vol_shape).astype(np.float32)
    y = rng.standard_normal((1, 30, 512, 512)).astype(np.float32)
    m, l2 = rel(T.tnlmr_project(g, ang, dev(f)).cpu().numpy()[0], R.project(rg, ang[0], f[0]))
    assert m <= 2e-5 and l2 <= 1e-5, f"project: {m:.2e} {l2:.2e}"
    m, l2 = rel(T.tnlmr_backproject(g, ang, dev(y)).cpu().numpy()[0], R.backproject(rg, ang[0], y[0]))
    assert m <= 2e-5 and l2 <= 1e-5, f"backproject: {m:.2e} {l2:.2e}"
