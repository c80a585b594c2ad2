"""Pins for the CPU oracle (oracle/tnlm_oracle.c): every check compares the oracle with
something OTHER than itself -- a closed form, a library routine, a dense linear solve, a
brute-force evaluation over all voxel pairs, or an invariant the paper states.

Citations are PAPER.md lines (arxiv/paper_1201_2450); readings P1..P15 are DESIGN.md's.
"""
import itertools

import numpy as np
import pytest
from numpy.lib.stride_tricks import sliding_window_view

from tnlm_inputs import CONFIGS, make_stack, random_stack

RNG = np.random.default_rng(1234)


def rand64(shape, seed):
    return np.random.default_rng(seed).random(shape)


def offsets(M):
    r = range(-M, M + 1)
    return list(itertools.product(r, r, r))  # (tz, ty, tx), raster order == k index


# --------------------------------------------------------------------------- brute force
def brute_force_nlm(f, ref, d, M, h, direction):
    """Eq. 3 + bracket of Eq. 8 evaluated over ALL voxel pairs of the edge-padded volumes.

    Independent route: np.pad(mode='edge') realises reading P4, sliding_window_view extracts
    the cubes, a dense pair matrix holds ||p_i(x)-p_j(y)||^2, candidates outside the search
    window get weight zero, rows are normalised (reading P1).
    """
    P, Z, Y, X = f.shape
    R = M + d
    out = np.zeros_like(f)
    for i in range(P):
        j = (i + direction) % P
        ri = np.pad(ref[i], R, mode="edge")
        rj = np.pad(ref[j], R, mode="edge")
        fj = np.pad(f[j], M, mode="edge")
        e = 2 * d + 1
        # cubes centred at every voxel of the volume padded by M  -> index (z+M, y+M, x+M)
        ci = sliding_window_view(ri, (e, e, e)).reshape(Z + 2 * M, Y + 2 * M, X + 2 * M, -1)
        cj = sliding_window_view(rj, (e, e, e)).reshape(Z + 2 * M, Y + 2 * M, X + 2 * M, -1)
        centres_i = [(z, y, x) for z in range(Z) for y in range(Y) for x in range(X)]
        cand = [(z, y, x) for z in range(-M, Z + M) for y in range(-M, Y + M) for x in range(-M, X + M)]
        A = np.stack([ci[z + M, y + M, x + M] for (z, y, x) in centres_i])          # [Nx, e^3]
        B = np.stack([cj[z + M, y + M, x + M] for (z, y, x) in cand])               # [Ny, e^3]
        D = ((A[:, None, :] - B[None, :, :]) ** 2).sum(-1)                           # all pairs
        ca = np.array(centres_i)[:, None, :]
        cb = np.array(cand)[None, :, :]
        inside = (np.abs(ca - cb).max(-1) <= M)
        Dm = np.where(inside, D, np.inf)
        U = np.exp(-(Dm - Dm.min(1, keepdims=True)) / (2 * h * h))
        W = U / U.sum(1, keepdims=True)
        fy = np.array([fj[z + M, y + M, x + M] for (z, y, x) in cand])
        out[i] = (W @ fy).reshape(Z, Y, X)
    return out


@pytest.mark.parametrize("d,M,P", [(1, 1, 3), (0, 1, 2), (1, 2, 3), (2, 1, 3)])
def test_brute_force_all_pairs(oracle, d, M, P):
    shape = (P, 3, 4, 5)
    f = rand64(shape, 1)
    ref = rand64(shape, 2)
    g = rand64(shape, 3)
    h, mu = 0.3, 0.7
    for direction in (+1, -1):
        want = brute_force_nlm(f, ref, d, M, h, direction)
        got = oracle.nlm_f64(f, ref, d, M, h, direction)
        np.testing.assert_allclose(got, want, rtol=0, atol=1e-13)
    want = mu / (2 + mu) * g + (brute_force_nlm(f, ref, d, M, h, 1) + brute_force_nlm(f, ref, d, M, h, -1)) / (2 + mu)
    got = oracle.jacobi_step_f64(f, g, d, M, h, mu, ref=ref)
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-13)


def test_brute_force_small_h_needs_shift(oracle):
    """With D/2h^2 in the hundreds an unshifted exp gives 0/0; reading P3 must hold."""
    shape = (3, 3, 4, 4)
    f = rand64(shape, 5)
    h = 0.02                      # D ~ 27*0.17 -> D/2h^2 ~ 5000
    want = brute_force_nlm(f, f, 1, 1, h, 1)
    got = oracle.nlm_f64(f, f, 1, 1, h, 1)
    assert np.isfinite(got).all()
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-13)


# --------------------------------------------------------------------------- closed forms
@pytest.mark.parametrize("d,h", [(0, 0.1), (1, 0.05), (2, 3.0)])
def test_M0_closed_form(oracle, d, h):
    """M=0: the only candidate is y=x, w=1 -> sweep = (mu g_i + f_{i+1} + f_{i-1})/(2+mu)."""
    shape = (5, 3, 4, 6)
    f, g = rand64(shape, 10), rand64(shape, 11)
    mu = 0.4
    want = (mu * g + np.roll(f, -1, axis=0) + np.roll(f, 1, axis=0)) / (2 + mu)
    got = oracle.jacobi_step_f64(f, g, d, 0, h, mu)
    np.testing.assert_allclose(got, want, rtol=0, atol=2e-16 * 4)


@pytest.mark.parametrize("M", [1, 2, 3])
def test_h_infinite_is_uniform_filter(oracle, M):
    """h -> inf: w = 1/n_t, NLM_s = box mean of f_j with replicated edges (scipy routine)."""
    from scipy.ndimage import uniform_filter
    shape = (3, 5, 6, 7)
    f = rand64(shape, 20)
    ref = rand64(shape, 21)
    for direction in (1, -1):
        got = oracle.nlm_f64(f, ref, 1, M, 1e7, direction)
        for i in range(shape[0]):
            want = uniform_filter(f[(i + direction) % shape[0]], size=2 * M + 1, mode="nearest")
            np.testing.assert_allclose(got[i], want, rtol=0, atol=1e-12)


def test_M0_fixed_point_dft_closed_form(oracle):
    """M=0 fixed point: f^(k) = mu g^(k) / (2 + mu - 2 cos(2 pi k / P)) along the phase axis."""
    shape = (7, 2, 3, 3)
    g = rand64(shape, 30)
    mu = 0.9
    f = g.copy()
    for _ in range(400):
        f = oracle.jacobi_step_f64(f, g, 1, 0, 0.1, mu)
    k = np.arange(shape[0])
    denom = (2 + mu - 2 * np.cos(2 * np.pi * k / shape[0]))[:, None, None, None]
    want = np.fft.ifft(mu * np.fft.fft(g, axis=0) / denom, axis=0).real
    np.testing.assert_allclose(f, want, rtol=0, atol=1e-12)


# --------------------------------------------------------------------------- invariants
def test_constant_stack_is_fixed_point(oracle):
    c = np.float32(0.3125)
    g = np.full((4, 5, 6, 7), c, dtype=np.float32)
    out = oracle.jacobi_step(g, g, 1, 2, np.float32(0.05), np.float32(0.5))
    # convex combination of equal values; exact up to the rounding of mu/(2+mu)+2/(2+mu)
    np.testing.assert_allclose(out, g, rtol=0, atol=1e-7)
    out64 = oracle.jacobi_step_f64(g.astype(np.float64), g.astype(np.float64), 1, 2, 0.05, 0.5)
    np.testing.assert_allclose(out64, float(c), rtol=0, atol=1e-15)   # 125 weights of 1/125: rounding only


def test_weights_nonnegative_normalised(oracle):
    ref = random_stack((3, 4, 5, 6), 40)
    w = oracle.weights(ref, 1, 2, np.float32(0.05))
    assert w.shape == (3, 2, 125, 4, 5, 6)
    assert (w >= 0).all()
    np.testing.assert_allclose(w.sum(axis=2), 1.0, rtol=0, atol=1e-14)
    # shifted form: the best candidate has u = 1, so max_k w = 1/Z >= 1/n_t
    assert (w.max(axis=2) >= 1.0 / 125 - 1e-15).all()


def test_mutual_weight_symmetry_cross_ratio(oracle):
    """the un-normalised weight of the pair (x in i, y in j) is common to both.

    The normalisers differ, so compare cross-ratios in which they cancel:
    w_ij(x,y) w_ij(x',y') / (w_ij(x,y') w_ij(x',y))  ==  same expression from phase j's side.
    """
    M, d, h = 1, 1, 0.4
    P, Z, Y, X = 3, 5, 5, 6
    ref = rand64((P, Z, Y, X), 50)
    w = oracle.weights(ref, d, M, h)
    offs = offsets(M)
    kidx = {t: k for k, t in enumerate(offs)}

    def wij(i, s, x, y):     # weight of candidate y (in phase i+s) for voxel x of phase i
        t = tuple(np.subtract(y, x))
        return w[i, s, kidx[t], x[0], x[1], x[2]]

    checked = 0
    for i in range(P):
        j = (i + 1) % P
        for z, y, x in itertools.product(range(1, Z - 1), range(1, Y - 1), range(1, X - 2)):
            a, a2 = (z, y, x), (z, y, x + 1)
            b, b2 = (z, y, x), (z, y + 1, x + 1)
            lhs = wij(i, 1, a, b) * wij(i, 1, a2, b2) / (wij(i, 1, a, b2) * wij(i, 1, a2, b))
            rhs = wij(j, 0, b, a) * wij(j, 0, b2, a2) / (wij(j, 0, b2, a) * wij(j, 0, b, a2))
            assert lhs == pytest.approx(rhs, rel=1e-10)
            checked += 1
    assert checked > 50


def test_convex_bounds_over_iterations(oracle):
    c = CONFIGS["config1"].scaled(nz=6, ny=10, nx=12, n_phase=4)
    g = make_stack(c)
    f = g
    for _ in range(4):
        f = oracle.jacobi_step(f, g, 1, 1, np.float32(c.h), np.float32(c.mu))
        assert f.min() >= g.min() - 1e-7 and f.max() <= g.max() + 1e-7


# --------------------------------------------------------------------------- Eq. 7 / linear system
def assemble_W(w, shape, M):
    """Dense [(P V) x (P V)] matrix of the bracket of Eq. 8 with clamped candidate columns."""
    P, Z, Y, X = shape
    V = Z * Y * X
    W = np.zeros((P * V, P * V))
    offs = offsets(M)
    for i in range(P):
        for s, dirn in ((0, -1), (1, 1)):
            j = (i + dirn) % P
            for z, y, x in itertools.product(range(Z), range(Y), range(X)):
                row = i * V + (z * Y + y) * X + x
                for k, (tz, ty, tx) in enumerate(offs):
                    cz, cy, cx = np.clip(z + tz, 0, Z - 1), np.clip(y + ty, 0, Y - 1), np.clip(x + tx, 0, X - 1)
                    W[row, j * V + (cz * Y + cy) * X + cx] += w[i, s, k, z, y, x]
    return W


@pytest.mark.parametrize("P", [2, 3, 4])
def test_frozen_weight_fixed_point_is_linear_solve(oracle, P):
    """Eq. 7: with weights frozen the sweep is Jacobi on [(2+mu) I - W] f = mu g
    and 'converges for any mu > 0'.  P=2 counts the single neighbour twice."""
    shape = (P, 2, 3, 4)
    M, d, h, mu = 1, 1, 0.35, 0.6
    ref, g = rand64(shape, 60), rand64(shape, 61)
    w = oracle.weights(ref, d, M, h)
    W = assemble_W(w, shape, M)
    np.testing.assert_allclose(W.sum(1), 2.0, atol=1e-13)
    n = W.shape[0]
    want = np.linalg.solve((2 + mu) * np.eye(n) - W, mu * g.reshape(-1)).reshape(shape)
    f = g.copy()
    prev_err = None
    for it in range(120):
        f = oracle.jacobi_step_f64(f, g, d, M, h, mu, ref=ref)
        err = np.abs(f - want).max()
        if prev_err is not None and prev_err > 1e-12:
            assert err <= prev_err * (2 / (2 + mu)) + 1e-15    # contraction from the row sums
        prev_err = err
    np.testing.assert_allclose(f, want, rtol=0, atol=1e-12)


def test_jacobi_step_equals_weights_then_sweep(oracle):
    shape = (3, 3, 4, 5)
    f, g, ref = rand64(shape, 70), rand64(shape, 71), rand64(shape, 72)
    w = oracle.weights(ref, 1, 1, 0.3)
    a = oracle.sweep_with_weights_f64(f, g, w, 1, 0.8)
    b = oracle.jacobi_step_f64(f, g, 1, 1, 0.3, 0.8, ref=ref)
    np.testing.assert_allclose(a, b, rtol=0, atol=1e-15)


# --------------------------------------------------------------------------- Eq. 6 / energy
def test_eq6_per_voxel_local_energy(oracle):
    """Eq. 6 is the derivative of the per-voxel local energy
    e(t) = mu/2 (t-g)^2 + 1/2 sum_s sum_y w (t - f_{i+s}(y))^2 and vanishes at the Eq. 8 value."""
    shape = (3, 3, 3, 4)
    M, d, h, mu = 1, 1, 0.3, 0.5
    f, g = rand64(shape, 80), rand64(shape, 81)
    w = oracle.weights(f, d, M, h)
    new = oracle.jacobi_step_f64(f, g, d, M, h, mu)
    nlm = {s: oracle.nlm_f64(f, f, d, M, h, s) for s in (1, -1)}
    offs = offsets(M)
    P, Z, Y, X = shape

    def e(i, z, y, x, t):
        tot = 0.5 * mu * (t - g[i, z, y, x]) ** 2
        for s, dirn in ((0, -1), (1, 1)):
            fj = f[(i + dirn) % P]
            for k, (tz, ty, tx) in enumerate(offs):
                v = fj[np.clip(z + tz, 0, Z - 1), np.clip(y + ty, 0, Y - 1), np.clip(x + tx, 0, X - 1)]
                tot += 0.5 * w[i, s, k, z, y, x] * (t - v) ** 2
        return tot

    eps = 1e-5
    for (i, z, y, x) in [(0, 0, 0, 0), (1, 1, 2, 3), (2, 2, 1, 0), (1, 0, 2, 2)]:
        t0 = f[i, z, y, x]
        fd = (e(i, z, y, x, t0 + eps) - e(i, z, y, x, t0 - eps)) / (2 * eps)
        eq6 = mu * (t0 - g[i, z, y, x]) + 2 * t0 - nlm[1][i, z, y, x] - nlm[-1][i, z, y, x]
        assert fd == pytest.approx(eq6, abs=1e-8)
        t1 = new[i, z, y, x]
        fd1 = (e(i, z, y, x, t1 + eps) - e(i, z, y, x, t1 - eps)) / (2 * eps)
        assert abs(fd1) < 1e-8


def _sinkhorn_symmetric_weights(shape, M, seed):
    """Symmetric non-negative coupling between neighbouring phases, in-window and in-volume
    only, balanced to row sums 2 -- the setting in which Eq. 6 is exactly grad E (reading P14)."""
    P, Z, Y, X = shape
    V = Z * Y * X
    rng = np.random.default_rng(seed)
    S = np.zeros((P * V, P * V))
    offs = offsets(M)
    for i in range(P):
        j = (i + 1) % P
        for z, y, x in itertools.product(range(Z), range(Y), range(X)):
            for (tz, ty, tx) in offs:
                zz, yy, xx = z + tz, y + ty, x + tx
                if 0 <= zz < Z and 0 <= yy < Y and 0 <= xx < X:
                    a, b = i * V + (z * Y + y) * X + x, j * V + (zz * Y + yy) * X + xx
                    S[a, b] = S[b, a] = rng.random() + 0.1
    r = np.ones(P * V)
    for _ in range(2000):
        r = np.sqrt(r * 2.0 / (S @ r))          # symmetric Sinkhorn: diag(r) S diag(r) 1 = 2
    Wg = r[:, None] * S * r[None, :]
    assert np.allclose(Wg.sum(1), 2.0, atol=1e-10) and np.allclose(Wg, Wg.T)
    w = np.zeros((P, 2, len(offs), Z, Y, X))
    for i in range(P):
        for s, dirn in ((0, -1), (1, 1)):
            j = (i + dirn) % P
            for z, y, x in itertools.product(range(Z), range(Y), range(X)):
                for k, (tz, ty, tx) in enumerate(offs):
                    zz, yy, xx = z + tz, y + ty, x + tx
                    if 0 <= zz < Z and 0 <= yy < Y and 0 <= xx < X:
                        w[i, s, k, z, y, x] = Wg[i * V + (z * Y + y) * X + x, j * V + (zz * Y + yy) * X + xx]
    return Wg, w


def _energy(f, g, Wg, mu, shape):
    """E = mu/2 sum_i ||f_i - g_i||^2 + 1/2 sum_i J[f_i, f_{i+1}]   (Eq. 4 with Eq. 2)."""
    P, Z, Y, X = shape
    V = Z * Y * X
    v = f.reshape(-1)
    E = 0.5 * mu * ((f - g) ** 2).sum()
    for i in range(P):
        j = (i + 1) % P
        blk = Wg[i * V:(i + 1) * V, j * V:(j + 1) * V]
        diff = v[i * V:(i + 1) * V, None] - v[None, j * V:(j + 1) * V]
        E += 0.5 * (blk * diff ** 2).sum()
    return E


def test_energy_gradient_and_descent_on_symmetric_weights(oracle):
    """On balanced symmetric weights (P>=3) Eq. 6 is the exact gradient of Eq. 4, the
    Gauss-Jacobi sweep of Eq. 8 decreases E monotonically and converges to the minimiser."""
    shape = (3, 2, 3, 3)
    M, mu = 1, 0.7
    Wg, w = _sinkhorn_symmetric_weights(shape, M, 90)
    f, g = rand64(shape, 91), rand64(shape, 92)
    # finite-difference gradient of the literal energy vs Eq. 6
    eq6 = (mu * (f - g) + 2 * f).reshape(-1) - Wg @ f.reshape(-1)
    eps = 1e-6
    for idx in (0, 7, 23, 40, 53):
        fp, fm = f.reshape(-1).copy(), f.reshape(-1).copy()
        fp[idx] += eps
        fm[idx] -= eps
        fd = (_energy(fp.reshape(shape), g, Wg, mu, shape) - _energy(fm.reshape(shape), g, Wg, mu, shape)) / (2 * eps)
        assert fd == pytest.approx(eq6[idx], abs=1e-7)
    # descent + convergence of the oracle's Eq. 8 sweep
    E_prev = _energy(f, g, Wg, mu, shape)
    for _ in range(150):
        f = oracle.sweep_with_weights_f64(f, g, w, M, mu)
        E = _energy(f, g, Wg, mu, shape)
        assert E <= E_prev + 1e-14
        E_prev = E
    n = Wg.shape[0]
    want = np.linalg.solve((2 + mu) * np.eye(n) - Wg, mu * g.reshape(-1)).reshape(shape)
    np.testing.assert_allclose(f, want, rtol=0, atol=1e-12)


def test_energy_decreases_on_config1_frozen_forward_weights(oracle):
    """Empirical (not provable: W is not symmetric, reading P14): with weights frozen at W_k,
    the literal Eq. 4 energy with forward row-normalised weights decreases over a sweep."""
    c = CONFIGS["config1"].scaled(nz=8, ny=12, nx=12, n_phase=5)
    g = make_stack(c).astype(np.float64)
    d, M, h, mu = c.patch_radius, c.search_radius, c.h, c.mu
    P, Z, Y, X = g.shape
    offs = offsets(M)

    def energy(f, w):
        E = 0.5 * mu * ((f - g) ** 2).sum()
        for i in range(P):
            fj = np.pad(f[(i + 1) % P], M, mode="edge")
            for k, (tz, ty, tx) in enumerate(offs):
                cand = fj[M + tz:M + tz + Z, M + ty:M + ty + Y, M + tx:M + tx + X]
                E += 0.5 * (w[i, 1, k] * (f[i] - cand) ** 2).sum()
        return E

    f = g.copy()
    for _ in range(3):
        w = oracle.weights(f, d, M, h)
        f_new = oracle.jacobi_step_f64(f, g, d, M, h, mu)
        assert energy(f_new, w) < energy(f, w)
        f = f_new


# --------------------------------------------------------------------------- the TNLM-E loop
def test_enhance_is_composition_of_steps(oracle):
    c = CONFIGS["config1"].scaled(nz=5, ny=9, nx=11, n_phase=3)
    g = make_stack(c)
    h, mu = np.float32(c.h), np.float32(c.mu)
    f = g.copy()
    for _ in range(3):
        f = oracle.jacobi_step(f, g, 1, 1, h, mu)          # ref = f^k
    out = oracle.enhance(g, 1, 1, h, mu, 3)
    assert np.array_equal(out, f)
    assert np.array_equal(oracle.enhance(g, 1, 1, h, mu, 0), g)         # n_iter = 0 copies
    f1 = oracle.enhance(g, 1, 1, h, mu, 1)
    f3 = oracle.enhance(g, 1, 1, h, mu, 2, f_init=f1)                   # resume keeps the original g
    assert np.array_equal(f3, f)


def test_jacobi_step_at_matches_full_sweep(oracle):
    g = random_stack((3, 5, 7, 9), 100)
    f = random_stack((3, 5, 7, 9), 101)
    h, mu = np.float32(0.2), np.float32(0.5)
    full = oracle.jacobi_step(f, g, 1, 2, h, mu)
    idx = np.random.default_rng(0).integers(0, f.size, 200)
    idx = np.concatenate([idx, [0, f.size - 1]])
    got = oracle.jacobi_step_at(f, g, 1, 2, h, mu, idx)
    assert np.array_equal(got, full.reshape(-1)[idx])
    # with a separate ref (TNLM-R usage)
    ref = random_stack((3, 5, 7, 9), 102)
    full = oracle.jacobi_step(f, g, 1, 1, h, mu, ref=ref)
    got = oracle.jacobi_step_at(f, g, 1, 1, h, mu, idx, ref=ref)
    assert np.array_equal(got, full.reshape(-1)[idx])


def test_fp32_boundary_matches_fp64_path(oracle):
    g = random_stack((3, 4, 5, 6), 110)
    f = random_stack((3, 4, 5, 6), 111)
    a = oracle.jacobi_step(f, g, 1, 1, np.float32(0.2), np.float32(0.5))
    b = oracle.jacobi_step_f64(f.astype(np.float64), g.astype(np.float64), 1, 1,
                               float(np.float32(0.2)), float(np.float32(0.5)))
    assert np.array_equal(a, b.astype(np.float32))


def test_enhancement_denoises_config1(oracle):
    """Sanity, not parity: same direction as PAPER.md:327 (streak/noise energy is removed)."""
    c = CONFIGS["config1"]
    g, clean = make_stack(c), make_stack(c, clean=True)
    f = oracle.enhance(g, c.patch_radius, c.search_radius, np.float32(c.h), np.float32(c.mu), c.n_iter)
    rmse0 = np.sqrt(((g - clean) ** 2).mean())
    rmse1 = np.sqrt(((f - clean) ** 2).mean())
    assert rmse1 < 0.6 * rmse0


# --------------------------------------------------------------------------- finite dependence reach
@pytest.mark.parametrize("d,M,K", [(1, 1, 2), (1, 2, 1), (2, 1, 1)])
def test_trajectory_on_a_crop_equals_full_volume_inside_the_reach(oracle, d, M, K):
    """Eq. 8 reads f and ref only within M+d voxels of x (PAPER.md:176 with the window of PAPER.md:223), so after
    K sweeps a voxel depends on g within K(M+d) voxels.  An enhancement of a cropped stack therefore equals the
    full-volume one, bit for bit, at every voxel further than K(M+d) from a cut face (faces that are faces of the
    volume are not cuts: clamp-to-edge reads the same voxels, reading P4).  The GPU parity tests use this to check
    whole 10-sweep trajectories at config 3 (tests/test_parity_trajectory_gpu.py); a wrong reach would show here as
    a mismatch one voxel inside the claimed region, which is also asserted to exist."""
    shape = (3, 15, 16, 17)
    g = random_stack(shape, 77)
    h, mu = np.float32(0.15), np.float32(0.5)
    full = oracle.enhance(g, d, M, h, mu, K)
    r = K * (M + d)
    # corner crop: z, y, x faces at 0 are volume faces; the upper faces are cuts
    zc, yc, xc = 15, 12, 13
    crop = oracle.enhance(np.ascontiguousarray(g[:, :zc, :yc, :xc]), d, M, h, mu, K)
    np.testing.assert_array_equal(crop[:, :, :yc - r, :xc - r], full[:, :zc, :yc - r, :xc - r])
    # ... and the claim is sharp: within the reach of a cut face the crop does differ somewhere
    assert np.any(crop[:, :, yc - r:, :] != full[:, :zc, yc - r:yc, :xc])
    # interior crop: every face is a cut
    a, b = 2, 14
    crop = oracle.enhance(np.ascontiguousarray(g[:, :, a:b, a:b]), d, M, h, mu, K)
    if b - a > 2 * r:
        np.testing.assert_array_equal(crop[:, :, r:b - a - r, r:b - a - r], full[:, :, a + r:b - r, a + r:b - r])
