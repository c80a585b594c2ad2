"""Pins of the TNLM-R oracle (oracle/tnlmr_oracle.c, oracle/tnlmr_oracle.py): projector pair, CGLS, the loop.

Every check is against something other than the oracle's own formula: hand-computed rays, a brute-force sampling of a
ray through the grid, the chord of a ray with a box / an ellipsoid in closed form, perspective magnification of a point,
the adjoint identity, dense linear algebra (numpy.linalg.lstsq / pinv) on a matrix assembled column by column.
"""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from tnlm_inputs import projections as PJ   # noqa: E402


@pytest.fixture(scope="module")
def R():
    from oracle import tnlmr_oracle as R_
    R_.lib()
    return R_


def test_axis_aligned_central_ray_by_hand(R):
    # odd grid and odd detector: the central ray at angle 0 runs along -x through the centres of row (iy, iz) = (2, 1)
    g = R.geom((3, 5, 4), 1, 3, 3, 1.0, 1.0, 50.0, 80.0, 0.5)
    S, D = R.ray_endpoints(g, 0.0, 1, 1)
    assert np.allclose(S, [50, 0, 0]) and np.allclose(D, [-30, 0, 0])
    vox, ln = R.ray(g, S, D)
    want = sorted(((1 * 5 + 2) * 4 + ix) for ix in range(4))
    assert sorted(vox.tolist()) == want
    assert np.allclose(ln, 0.5, rtol=0, atol=1e-12)


def test_diagonal_ray_by_hand(R):
    # 4 x 4 x 1 grid of unit voxels spanning [-2, 2]^2: the diagonal crosses voxels (0,0) .. (3,3), sqrt(2) in each
    g = R.geom((1, 4, 4), 1, 1, 1, 1.0, 1.0, 10.0, 20.0, 1.0)
    vox, ln = R.ray(g, [-3.0, -3.0, 0.1], [3.0, 3.0, 0.1])
    assert sorted(vox.tolist()) == [0, 5, 10, 15]
    assert np.allclose(ln, np.sqrt(2.0), atol=1e-12)
    # a ray that misses the grid, and one parallel to a face just outside it
    assert len(R.ray(g, [-3.0, 5.0, 0.0], [3.0, 5.5, 0.0])[0]) == 0
    assert len(R.ray(g, [-3.0, 2.0, 0.0], [3.0, 2.0, 0.0])[0]) == 0


def test_ray_lengths_against_brute_force_sampling(R):
    # intersection length with a voxel = measure of the ray's points inside it: sample the ray densely
    rng = np.random.default_rng(3)
    g = R.geom((5, 6, 7), 1, 1, 1, 1.0, 1.0, 10.0, 20.0, 0.8)
    n = np.array([7, 6, 5])
    lo = -0.5 * n * 0.8
    for _ in range(12):
        S = rng.uniform(-1, 1, 3) * 2 + np.array([9.0, 0, 0]) * rng.choice([-1, 1])
        D = -S + rng.uniform(-1.5, 1.5, 3)
        vox, ln = R.ray(g, S, D)
        m = 400001
        t = (np.arange(m) + 0.5) / m
        pts = S[None, :] + t[:, None] * (D - S)[None, :]
        idx = np.floor((pts - lo) / 0.8).astype(int)
        inside = np.all((idx >= 0) & (idx < n), axis=1)
        flat = (idx[inside, 2] * 6 + idx[inside, 1]) * 7 + idx[inside, 0]
        cnt = np.bincount(flat, minlength=5 * 6 * 7) * (np.linalg.norm(D - S) / m)
        got = np.zeros(5 * 6 * 7)
        np.add.at(got, vox, ln)
        assert np.abs(got - cnt).max() < 3e-4
        assert len(set(vox.tolist())) == len(vox)          # a convex voxel is crossed once


def _box_chord(S, D, half):
    d = D - S
    with np.errstate(divide="ignore", invalid="ignore"):
        a0, a1 = (-half - S) / d, (half - S) / d
    lo, hi = np.minimum(a0, a1), np.maximum(a0, a1)
    amin, amax = max(0.0, np.nanmax(lo)), min(1.0, np.nanmin(hi))
    return max(0.0, amax - amin) * np.linalg.norm(d)


def test_projection_of_a_constant_volume_is_the_chord_of_the_box(R):
    g = R.geom((6, 8, 10), 3, 9, 7, 1.1, 0.9, 40.0, 70.0, 0.7)
    ang = np.array([0.3, 2.0, 4.4])
    y = R.project(g, ang, np.full((6, 8, 10), 2.5))
    half = 0.5 * 0.7 * np.array([10, 8, 6])
    for k, th in enumerate(ang):
        for iv in range(7):
            for iu in range(9):
                S, D = R.ray_endpoints(g, th, iu, iv)
                assert abs(y[k, iv, iu] - 2.5 * _box_chord(S, D, half)) < 1e-10


def test_geometry_point_magnification(R):
    # a single bright voxel projects to the pixel that perspective geometry predicts:
    # depth s = sid - p.e_r, u = sdd (p.e_u) / s, v = sdd p_z / s with e_r = (cos t, sin t, 0), e_u = (-sin t, cos t, 0)
    g = R.geom((17, 17, 17), 4, 41, 41, 0.5, 0.5, 30.0, 50.0, 0.5)
    ang = np.array([0.0, 0.9, 2.2, 5.0])
    f = np.zeros((17, 17, 17))
    iz, iy, ix = 11, 4, 13
    f[iz, iy, ix] = 1.0
    p = (np.array([ix, iy, iz]) - 8.0) * 0.5
    y = R.project(g, ang, f)
    for k, th in enumerate(ang):
        e_r, e_u = np.array([np.cos(th), np.sin(th), 0]), np.array([-np.sin(th), np.cos(th), 0])
        s = 30.0 - p @ e_r
        u, v = 50.0 * (p @ e_u) / s, 50.0 * p[2] / s
        iv, iu = np.unravel_index(np.argmax(y[k]), y[k].shape)
        assert abs((iu - 20) * 0.5 - u) <= 0.5 and abs((iv - 20) * 0.5 - v) <= 0.5


def test_projection_of_an_ellipsoid_approaches_its_analytic_chord(R):
    # discretised P of the voxelised phantom vs the closed-form line integral: agreement to the voxelisation error
    geom = PJ.ConeGeometry((48, 48, 48), 25.6 / 48, 2, 24, 24, 40.96 / 24, 40.96 / 24, 100.0, 153.6)
    ell = [((1.0, -2.0, 0.5), (7.0, 5.0, 6.0), 1.0)]
    ang = np.array([0.4, 2.9])
    g = R.geom(geom.vol_shape, 2, 24, 24, geom.du, geom.dv, geom.sid, geom.sdd, geom.voxel)
    y = R.project(g, ang, PJ.voxelise(geom, ell))
    ya = PJ.analytic_projections(geom, ang, ell)
    core = ya > 0.5 * ya.max()                     # away from the grazing rays, where a binary voxelisation is coarse
    assert core.sum() > 50 and (np.abs(y - ya)[core] < 2.0 * geom.voxel).all()   # a chord is off by about a voxel per end
    assert abs(y.sum() - ya.sum()) < 0.02 * ya.sum()


@pytest.mark.parametrize("shape,nview,nu,nv", [((4, 5, 6), 3, 7, 5), ((8, 8, 8), 2, 12, 12), ((1, 9, 9), 4, 16, 1)])
def test_backprojector_is_the_adjoint(R, shape, nview, nu, nv):
    rng = np.random.default_rng(5)
    g = R.geom(shape, nview, nu, nv, 1.3, 1.7, 25.0, 41.0, 0.9)
    ang = rng.uniform(0, 2 * np.pi, nview)
    f, y = rng.standard_normal(shape), rng.standard_normal((nview, nv, nu))
    lhs, rhs = (R.project(g, ang, f) * y).sum(), (f * R.backproject(g, ang, y)).sum()
    assert abs(lhs - rhs) <= 1e-12 * max(abs(lhs), 1.0)


def _dense(R, g, ang):
    nvox = g.nz * g.ny * g.nx
    A = np.zeros((g.n_view * g.nv * g.nu, nvox))
    for j in range(nvox):
        e = np.zeros(nvox)
        e[j] = 1.0
        A[:, j] = R.project(g, ang, e.reshape(g.nz, g.ny, g.nx)).ravel()
    return A


def test_cgls_converges_to_the_minimum_norm_least_squares_solution(R):
    rng = np.random.default_rng(9)
    g = R.geom((3, 3, 3), 2, 5, 4, 1.5, 1.5, 20.0, 32.0, 1.0)
    ang = np.array([0.2, 1.9])
    A = _dense(R, g, ang)
    y = rng.standard_normal(A.shape[0])
    yv = y.reshape(2, 4, 5)
    # from zero: the minimum-norm least-squares solution (numpy.linalg.lstsq); with a start x0: x0 + pinv(A)(y - A x0)
    x, res = R.cgls(g, ang, yv, np.zeros((3, 3, 3)), 80, residuals=True)
    want = np.linalg.lstsq(A, y, rcond=None)[0]
    assert np.abs(x.ravel() - want).max() < 1e-8 * max(1.0, np.abs(want).max())
    assert res[-1] < 1e-9 * res[0]
    x0 = rng.standard_normal((3, 3, 3))
    x1 = R.cgls(g, ang, yv, x0, 80)
    want1 = x0.ravel() + np.linalg.pinv(A) @ (y - A @ x0.ravel())
    assert np.abs(x1.ravel() - want1).max() < 1e-8 * max(1.0, np.abs(want1).max())


def test_cgls_iterates_minimise_over_the_krylov_subspace(R):
    # the k-th CGLS iterate from 0 minimises ||A x - y|| over span{A^T y, (A^T A) A^T y, ...}: solve that small problem densely
    rng = np.random.default_rng(10)
    g = R.geom((2, 4, 4), 3, 6, 3, 1.2, 1.2, 18.0, 30.0, 1.0)
    ang = np.array([0.1, 2.3, 4.1])
    A = _dense(R, g, ang)
    y = rng.standard_normal(A.shape[0])
    K = [A.T @ y]
    prev_r = np.inf
    for k in range(1, 6):
        x = R.cgls(g, ang, y.reshape(3, 3, 6), np.zeros((2, 4, 4)), k).ravel()
        B = np.stack(K, axis=1)
        c = np.linalg.lstsq(A @ B, y, rcond=None)[0]
        assert np.abs(x - B @ c).max() < 1e-9 * np.abs(x).max()
        r = np.linalg.norm(A @ x - y)
        assert r <= prev_r + 1e-12
        prev_r = r
        K.append(A.T @ (A @ K[-1]))
    # zero iterations leave the start untouched; the residual history starts at ||A^T (y - A x0)||
    x0 = rng.standard_normal((2, 4, 4))
    xz, res = R.cgls(g, ang, y.reshape(3, 3, 6), x0, 0, residuals=True)
    assert np.array_equal(xz, x0) and abs(res[0] - np.linalg.norm(A.T @ (y - A @ x0.ravel()))) < 1e-10


def test_tnlmr_loop_structure(R):
    from oracle import tnlm_oracle as O
    rng = np.random.default_rng(2)
    P, shape = 3, (4, 6, 6)
    g = R.geom(shape, 2, 8, 6, 1.4, 1.4, 30.0, 45.0, 1.0)
    ang = PJ.phase_angles(P, 2)
    y = rng.random((P, 2, 6, 8)).astype(np.float32)
    f0 = (rng.random((P,) + shape) - 0.3).astype(np.float32)
    d, M, h, mu = 1, 1, 0.4, 0.8
    # n_cgls = 0: step 1 returns f^(k-1), so an outer iteration is clamp(sweep(f, f, ref = f))
    got = R.reconstruct(g, ang, y, f0, d, M, h, mu, 1, 0)
    want = np.maximum(O.jacobi_step(f0, f0, d, M, np.float32(h), np.float32(mu)), 0)
    assert np.array_equal(got, want) and got.min() >= 0
    # two outer iterations = one after the other; the history exposes g^(k)
    f2, hist = R.reconstruct(g, ang, y, f0, d, M, h, mu, 2, 2, history=True)
    f1 = R.reconstruct(g, ang, y, f0, d, M, h, mu, 1, 2)
    assert np.array_equal(hist[0][1], f1) and np.array_equal(R.reconstruct(g, ang, y, f1, d, M, h, mu, 1, 2), f2)
    # the data term acts: g^(1) fits the projections better than the start does
    r0 = sum(np.linalg.norm(R.project(g, ang[i], f0[i]) - y[i]) for i in range(P))
    r1 = sum(np.linalg.norm(R.project(g, ang[i], hist[0][0][i]) - y[i]) for i in range(P))
    assert r1 < r0
    # the two readings of the inner start differ (so the flag is live) but share g^(1)
    alt, hist_alt = R.reconstruct(g, ang, y, f0, d, M, h, mu, 1, 2, inner_start="previous", history=True)
    assert np.array_equal(hist_alt[0][0], hist[0][0]) and not np.array_equal(alt, f1)


def test_projection_inputs_module():
    geom = PJ.paper_geometry(16, 3, 20)
    ang, y, vols = PJ.make_projection_stack(geom, 4, noise=0.0, seed=1)
    assert ang.shape == (4, 3) and y.shape == (4, 3, 20, 20) and vols.shape == (4, 16, 16, 16)
    allang = np.sort(ang.ravel())
    assert np.allclose(np.diff(allang), 2 * np.pi / 12)                    # 12 views equally spaced, dealt in turn
    assert np.allclose(np.diff(ang, axis=1), 2 * np.pi / 3)                # each phase: equally spaced in a full turn
    assert y.min() >= 0 and y.max() > 1.0 and vols.max() <= 1.01
    assert not np.array_equal(vols[0], vols[2])                            # the tumour moves
