"""Parity of the CUDA path (through the C ABI of libtnlm.so) with the CPU oracle, element by
element on the same seeded inputs.  Bar (BASELINE.json north_star):
    max |delta| <= 1e-4 * (max g - min g)    and    ||delta||_2 / ||f_oracle||_2 <= 1e-5   in fp32.
"""
import numpy as np
import pytest

from tnlm_inputs import CONFIGS, make_stack, dynamic_range, random_stack

pytestmark = pytest.mark.gpu

MAX_TOL = 1e-4     # x dynamic range of the input
L2_TOL = 1e-5


@pytest.fixture(scope="module")
def T():
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    import paper_1201_2450_b200 as T
    T.lib()   # fails loudly if libtnlm.so is missing: there is no fallback
    return T


def variants(T, p):
    """Every kernel variant compiled for these parameters (include/tnlm.h: TNLM_VARIANT_*)."""
    out = [T.VARIANT_GENERIC]
    if 1 <= p.search_radius <= 4:
        if p.patch_radius == 1:
            out.append(T.VARIANT_TILED)
        if p.patch_radius in (1, 2):
            out.append(T.VARIANT_PAIRED)
        if p.patch_radius in (1, 2) and 2 <= p.search_radius <= 4:
            out.append(T.VARIANT_PAIRED_TMEM)
    return out


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def assert_parity(got, want, rng_scale, what=""):
    got = np.asarray(got, dtype=np.float64)
    want = np.asarray(want, dtype=np.float64)
    assert np.isfinite(got).all(), f"{what}: non-finite output"
    max_err = np.abs(got - want).max()
    l2 = np.linalg.norm(got - want) / max(np.linalg.norm(want), 1e-300)
    assert max_err <= MAX_TOL * rng_scale, f"{what}: max|d|={max_err:.3e} > {MAX_TOL * rng_scale:.3e}"
    assert l2 <= L2_TOL, f"{what}: rel L2={l2:.3e} > {L2_TOL}"
    return max_err, l2


def params_of(T, cfg, shape=None):
    return T.TnlmParams.make(shape or cfg.shape, cfg.patch_radius, cfg.search_radius, cfg.h, cfg.mu)


# ------------------------------------------------------------------ config 1: full trajectory
def test_config1_full_enhancement(T, oracle):
    cfg = CONFIGS["config1"]
    g = make_stack(cfg)
    p = params_of(T, cfg)
    want = oracle.enhance(g, cfg.patch_radius, cfg.search_radius, np.float32(cfg.h), np.float32(cfg.mu), cfg.n_iter)
    for v in variants(T, p):
        got = T.tnlm_enhance(p, dev(g), cfg.n_iter, variant=v).cpu().numpy()
        assert_parity(got, want, dynamic_range(g), f"config1 variant {v}")


# ------------------------------------------------------------------ config 2 recipe, reduced grid
def test_config2_recipe_reduced_two_sweeps(T, oracle):
    """Thorax recipe of config 2 (d=1, M=2, h=0.05, mu=0.5) on a grid the oracle finishes in
    seconds; extents span several tiles and leave ragged tails in x, y and z."""
    cfg = CONFIGS["config2"].scaled(nz=21, ny=45, nx=70, n_phase=4, tumour_radius=3, si_amplitude=3)
    g = make_stack(cfg)
    p = params_of(T, cfg)
    want = oracle.enhance(g, 1, 2, np.float32(cfg.h), np.float32(cfg.mu), 2)
    for v in variants(T, p):
        got = T.tnlm_enhance(p, dev(g), 2, variant=v).cpu().numpy()
        assert_parity(got, want, dynamic_range(g), f"config2-reduced variant {v}")


# ------------------------------------------------------------------ edge cases
EDGE = [
    # shape,            d, M, h,     mu
    ((2, 1, 1, 1),      1, 1, 0.1,   1.0),    # smallest legal stack, P=2 counts the neighbour twice
    ((2, 3, 4, 5),      1, 2, 0.05,  0.5),    # window larger than the volume
    ((3, 5, 7, 9),      0, 1, 0.1,   1.0),    # d=0: single-voxel patch
    ((3, 5, 7, 9),      1, 0, 0.1,   1.0),    # M=0: closed form (mu g + f+ + f-)/(2+mu)
    ((3, 6, 9, 33),     2, 1, 0.2,   0.3),    # 5^3 patch
    ((3, 9, 11, 37),    1, 3, 0.06,  0.5),    # 7^3 window (config 4's)
    ((3, 9, 10, 35),    2, 2, 0.1,   0.5),
    ((2, 10, 12, 34),   1, 4, 0.1,   2.0),    # 9^3 window
    ((5, 2, 31, 129),   1, 2, 0.05,  0.5),    # flat slab, ragged x
    ((3, 17, 3, 4),     1, 1, 0.02,  0.5),    # tiny h: exponents in the thousands (reading P3)
    ((3, 4, 5, 6),      3, 1, 0.5,   0.5),    # largest compiled patch radius
    ((2, 7, 33, 21),    2, 3, 0.15,  0.5),    # 5^3 patch, 7^3 window
    ((2, 6, 29, 35),    2, 4, 0.15,  0.5),    # 5^3 patch, 9^3 window
    ((3, 13, 57, 18),   2, 2, 0.12,  1.0),    # 5^3 patch over two y-tiles (28 output rows each)
]


@pytest.mark.parametrize("shape,d,M,h,mu", EDGE)
def test_edge_cases_one_sweep(T, oracle, shape, d, M, h, mu):
    f = random_stack(shape, 7)
    g = random_stack(shape, 8)
    p = T.TnlmParams.make(shape, d, M, h, mu)
    want = oracle.jacobi_step(f, g, d, M, np.float32(h), np.float32(mu))
    for v in variants(T, p):
        got = T.tnlm_jacobi_step(p, dev(f), dev(g), variant=v).cpu().numpy()
        assert_parity(got, want, 1.0, f"edge {shape} d={d} M={M} variant {v}")


def moving_block_stack(shape, shift, seed):
    """A bright block (0.6 on 0.1) that moves `shift` voxels per phase along z, y and x, plus weak noise:
    at the block faces the zero offset is a bad match and a shifted candidate is better by far more
    than 2^100 (small h), so the reference exponent set in the first pass must be re-based later."""
    P, Z, Y, X = shape
    rng = np.random.default_rng(seed)
    out = np.full(shape, 0.1, dtype=np.float64)
    for ph in range(P):
        z0, y0, x0 = Z // 4 + shift * ph, Y // 4 + shift * ph, X // 4 + shift * ph
        out[ph, z0:z0 + Z // 3, y0:y0 + Y // 3, x0:x0 + X // 3] = 0.6
    out += 0.01 * rng.standard_normal(shape)
    return out.astype(np.float32)


@pytest.mark.parametrize("M,shape", [(1, (3, 13, 33, 21)), (2, (3, 11, 35, 37)), (3, (3, 10, 31, 19)), (4, (2, 9, 30, 18))])
def test_moving_edges_rebase_path(T, oracle, M, shape):
    g = moving_block_stack(shape, min(M, 2), 11 + M)
    h, mu = 0.05, 0.5   # c2*D ~ 650 at a mismatched block face: far outside the 2^100 guard band, still fp32-resolvable
    p = T.TnlmParams.make(shape, 1, M, h, mu)
    want = oracle.enhance(g, 1, M, np.float32(h), np.float32(mu), 2)
    for v in variants(T, p):
        got = T.tnlm_enhance(p, dev(g), 2, variant=v).cpu().numpy()
        assert_parity(got, want, dynamic_range(g), f"moving block M={M} variant {v}")


@pytest.mark.parametrize("M,shape", [(1, (3, 9, 30, 20)), (2, (3, 10, 33, 22)), (3, (2, 9, 31, 18))])
def test_moving_edges_rebase_path_patch5(T, oracle, M, shape):
    g = moving_block_stack(shape, min(M, 2), 21 + M)
    h, mu = 0.08, 0.5
    p = T.TnlmParams.make(shape, 2, M, h, mu)
    want = oracle.enhance(g, 2, M, np.float32(h), np.float32(mu), 2)
    for v in variants(T, p):
        got = T.tnlm_enhance(p, dev(g), 2, variant=v).cpu().numpy()
        assert_parity(got, want, dynamic_range(g), f"moving block d=2 M={M} variant {v}")


RAGGED = [(2, 7, 29, 15), (2, 5, 30, 16), (2, 4, 31, 17), (2, 13, 61, 47), (3, 6, 1, 50), (3, 1, 64, 2)]


@pytest.mark.parametrize("shape", RAGGED)
def test_ragged_tiles_one_sweep(T, oracle, shape):
    """Extents around the tile sizes of the sweep kernels (30 output rows, 16/32 columns, RZ planes; odd nx
    takes the scalar epilogue)."""
    f, g = random_stack(shape, 21), random_stack(shape, 22)
    for M in (1, 2):
        p = T.TnlmParams.make(shape, 1, M, 0.25, 0.5)
        want = oracle.jacobi_step(f, g, 1, M, np.float32(0.25), np.float32(0.5))
        for v in variants(T, p):
            got = T.tnlm_jacobi_step(p, dev(f), dev(g), variant=v).cpu().numpy()
            assert_parity(got, want, 1.0, f"ragged {shape} M={M} variant {v}")


@pytest.mark.parametrize("d,M,shape", [(1, 1, (3, 9, 33, 41)), (1, 2, (3, 9, 35, 41)), (1, 3, (3, 7, 33, 29)), (1, 4, (2, 6, 31, 21)),
                                       (2, 1, (3, 9, 31, 37)), (2, 2, (3, 7, 30, 35)), (2, 3, (2, 6, 29, 19)), (2, 4, (2, 5, 29, 13))])
def test_separate_ref_stack(T, oracle, d, M, shape):
    """ref != f (weights from one stack, averages of another): every kernel variant that takes a
    separate ref, the packed kernels included (they hold f_j in a candidate tile of its own), against the oracle."""
    f, g, ref = random_stack(shape, 1), random_stack(shape, 2), random_stack(shape, 3)
    h = 0.3 if d == 1 else 0.45
    p = T.TnlmParams.make(shape, d, M, h, 0.5)
    want = oracle.jacobi_step(f, g, d, M, np.float32(h), np.float32(0.5), ref=ref)
    for v in (T.VARIANT_GENERIC, T.VARIANT_PAIRED, T.VARIANT_AUTO):
        got = T.tnlm_jacobi_step(p, dev(f), dev(g), ref=dev(ref), variant=v).cpu().numpy()
        assert_parity(got, want, 1.0, f"separate ref d={d} M={M} variant {v}")
    if T.VARIANT_TILED in variants(T, p):      # the scalar tiled kernel covers ref = f only: an explicit request is refused
        with pytest.raises(T.TnlmError) as e:
            T.tnlm_jacobi_step(p, dev(f), dev(g), ref=dev(ref), variant=T.VARIANT_TILED)
        assert e.value.code == -4


def test_separate_ref_thorax_moving_edges(T, oracle):
    """Separate ref on structured data: weights from a lightly smoothed copy (what a TNLM-R outer iteration would
    pass), values from the noisy stack; slabs of the packed kernel tile the sweep bit for bit there too."""
    import torch
    cfg = CONFIGS["config2"].scaled(nz=13, ny=47, nx=50, n_phase=4, tumour_radius=3, si_amplitude=3)
    g = make_stack(cfg)
    ref = (0.5 * g + 0.25 * np.roll(g, 1, axis=3) + 0.25 * np.roll(g, -1, axis=3)).astype(np.float32)
    for d, M, h in [(1, 2, 0.05), (2, 1, 0.08)]:
        p = T.TnlmParams.make(cfg.shape, d, M, h, cfg.mu)
        want = oracle.jacobi_step(g, g, d, M, np.float32(h), np.float32(cfg.mu), ref=ref)
        got = T.tnlm_jacobi_step(p, dev(g), dev(g), ref=dev(ref), variant=T.VARIANT_PAIRED)
        assert_parity(got.cpu().numpy(), want, dynamic_range(g), f"separate ref thorax d={d} M={M}")
        out = torch.full_like(got, -5.0)
        for (a, b) in [(0, 3), (3, 4), (4, 13)]:
            T.tnlm_jacobi_step_slab(p, dev(g), dev(g), a, b, ref=dev(ref), f_out=out, variant=T.VARIANT_PAIRED)
        assert torch.equal(out, got)


def test_constant_stack_is_fixed_point_and_bounds(T):
    import torch
    shape = (4, 9, 33, 65)
    p = T.TnlmParams.make(shape, 1, 2, 0.05, 0.5)
    c = torch.full(shape, 0.3125, device="cuda")
    g = dev(random_stack(shape, 11))
    for v in variants(T, p):
        out = T.tnlm_jacobi_step(p, c, c, variant=v)
        assert (out - c).abs().max().item() <= 1e-6
        f = T.tnlm_enhance(p, g, 3, variant=v)
        assert f.min().item() >= g.min().item() - 1e-6 and f.max().item() <= g.max().item() + 1e-6


def _patch_distances(ref, d, M):
    """D[p][s][k][z][y][x] of Eq. 3 in numpy fp64 (edge padding = reading P4; s = 0: phase p-1, s = 1: phase p+1;
    k raster over (tz, ty, tx)): sets the scale of the fp32 error of each weight."""
    P, Z, Y, X = ref.shape
    R = M + d
    pad = [np.pad(ref[i].astype(np.float64), R, mode="edge") for i in range(P)]
    e = 2 * d + 1
    out = np.empty((P, 2, (2 * M + 1) ** 3, Z, Y, X))
    for i in range(P):
        for s, j in enumerate(((i - 1) % P, (i + 1) % P)):
            k = 0
            for tz in range(-M, M + 1):
                for ty in range(-M, M + 1):
                    for tx in range(-M, M + 1):
                        a = pad[i][M:M + Z + 2 * d, M:M + Y + 2 * d, M:M + X + 2 * d]
                        b = pad[j][M + tz:M + tz + Z + 2 * d, M + ty:M + ty + Y + 2 * d, M + tx:M + tx + X + 2 * d]
                        sq = (a - b) ** 2
                        out[i, s, k] = np.lib.stride_tricks.sliding_window_view(sq, (e, e, e)).sum(axis=(-1, -2, -3))
                        k += 1
    return out


@pytest.mark.parametrize("shape,d,M,h", [
    ((3, 4, 6, 10), 1, 1, 0.2),
    ((3, 5, 7, 9), 1, 2, 0.05),     # config 2/3's window and h: shifts of several hundred binades
    ((3, 6, 7, 8), 2, 1, 0.1),      # 5^3 patch
    ((2, 4, 9, 11), 1, 1, 0.02),    # tiny h: nearly one-hot weights, only the shifted form survives (reading P3)
    ((3, 3, 5, 6), 0, 3, 0.3),      # single-voxel patch, 7^3 window larger than the volume
])
def test_weights_match_oracle(T, oracle, shape, d, M, h):
    """tnlm_weights against the oracle's normalised weights of Eq. 3/9, every (p, s, k, x).

    Tolerance from the arithmetic: the kernel forms D in fp32 (as the sweep kernels do).  A distance carries an
    absolute error of at most ~8 ulp (sum of (2d+1)^3 squares, then parked as fp32), and w = 2^((Dmin - D) c2) / Z,
    so |dw| <= w ln2 c2 * 8 * 2^-23 * (D + Dmin), plus 2e-6 for the exp2 approximation and the normalising sum.
    D and Dmin come from numpy here (independent of both sides)."""
    ref = random_stack(shape, 21)
    p = T.TnlmParams.make(shape, d, M, h, 1.0)
    want = oracle.weights(ref, d, M, np.float32(h))
    got = T.tnlm_weights(p, dev(ref)).cpu().numpy()
    n_t = (2 * M + 1) ** 3
    assert got.shape == want.shape and (got >= 0).all() and np.isfinite(got).all()
    np.testing.assert_allclose(got.sum(axis=2), 1.0, atol=n_t * 2.0 ** -23 + 1e-6)
    c2 = 1.4426950408889634 / (2.0 * h * h)
    D = _patch_distances(ref, d, M)
    tol = want * np.log(2.0) * c2 * 8 * 2.0 ** -23 * (D + D.min(axis=2, keepdims=True)) + 2e-6
    excess = np.abs(got - want) - tol
    assert excess.max() <= 0, f"weight error exceeds the fp32 bound by {excess.max():.3e}"


def test_weights_feed_the_sweep(T, oracle):
    """The materialised weights reproduce the fused sweep: Eq. 8 evaluated with w_out (oracle's sweep_with_weights)
    equals tnlm_jacobi_step on the same stack."""
    shape = (3, 5, 8, 9)
    f, g = random_stack(shape, 5), random_stack(shape, 6)
    p = T.TnlmParams.make(shape, 1, 2, 0.15, 0.7)
    w = T.tnlm_weights(p, dev(f)).cpu().numpy().astype(np.float64)
    via_w = oracle.sweep_with_weights_f64(f, g, w, 2, 0.7)
    got = T.tnlm_jacobi_step(p, dev(f), dev(g)).cpu().numpy()
    assert_parity(got, via_w, 1.0, "sweep from materialised weights")


# ------------------------------------------------------------------ loop / ABI semantics on the device
def test_enhance_equals_manual_steps_bitwise(T):
    import torch
    cfg = CONFIGS["config1"]
    g = dev(make_stack(cfg))
    p = params_of(T, cfg)
    for v in variants(T, p):
        f = g
        for _ in range(3):
            f = T.tnlm_jacobi_step(p, f, g, variant=v)
        assert torch.equal(T.tnlm_enhance(p, g, 3, variant=v), f)
        assert torch.equal(T.tnlm_enhance(p, g, 0, variant=v), g)
        f1 = T.tnlm_enhance(p, g, 1, variant=v)
        assert torch.equal(T.tnlm_enhance(p, g, 2, f_init=f1, variant=v), f)
        assert torch.equal(T.tnlm_enhance(p, g, 4, variant=v), T.tnlm_jacobi_step(p, f, g, variant=v))


def test_slabs_tile_the_sweep_bitwise(T):
    import torch
    shape = (3, 19, 30, 40)
    f, g = dev(random_stack(shape, 31)), dev(random_stack(shape, 32))
    p = T.TnlmParams.make(shape, 1, 2, 0.1, 0.5)
    for v in variants(T, p):
        full = T.tnlm_jacobi_step(p, f, g, variant=v)
        out = torch.full_like(f, -7.0)
        for (a, b) in [(0, 5), (5, 6), (6, 6), (6, 19)]:
            T.tnlm_jacobi_step_slab(p, f, g, a, b, f_out=out, variant=v)
        assert torch.equal(out, full)


def test_enhance_host_matches_device_path(T):
    import torch
    cfg = CONFIGS["config1"]
    g = make_stack(cfg)
    p = params_of(T, cfg)
    gh = torch.from_numpy(g).pin_memory()
    out_h = T.tnlm_enhance_host(p, gh, cfg.n_iter)
    out_d = T.tnlm_enhance(p, dev(g), cfg.n_iter)
    assert torch.equal(out_h, out_d.cpu())


@pytest.mark.parametrize("nz,n_iter,M,d", [(40, 1, 2, 1), (37, 2, 2, 1), (64, 3, 1, 1), (48, 2, 3, 1), (44, 2, 1, 2),
                                            (32, 2, 4, 2), (130, 2, 2, 1), (121, 1, 2, 1)])
def test_enhance_host_pipelined_slabs_bitwise(T, nz, n_iter, M, d):
    """Volumes of 32+ planes take the pipelined host path (slab-wise H2D / first sweep, last sweep / D2H on a second
    stream): same bits as the device path, pinned or pageable host memory, and the call may be repeated."""
    import torch
    shape = (3, nz, 33, 40)
    g = random_stack(shape, 70 + nz)
    p = T.TnlmParams.make(shape, d, M, 0.3, 0.5)
    want = T.tnlm_enhance(p, dev(g), n_iter).cpu()
    gh = torch.from_numpy(g).pin_memory()
    for _ in range(2):
        assert torch.equal(T.tnlm_enhance_host(p, gh, n_iter), want)
    assert torch.equal(T.tnlm_enhance_host(p, torch.from_numpy(g), n_iter, f_out_host=torch.empty(shape)), want)
    assert torch.equal(T.tnlm_enhance_host(p, gh, n_iter, copy_stream=torch.cuda.Stream()), want)   # caller-owned copy stream


def test_device_error_codes(T):
    import torch
    shape = (3, 4, 8, 8)
    p = T.TnlmParams.make(shape, 1, 1, 0.1, 1.0)
    f = torch.rand(shape, device="cuda")
    with pytest.raises(T.TnlmError) as e:
        T.tnlm_jacobi_step(p, f, f, f_out=f)
    assert e.value.code == -5
    with pytest.raises(T.TnlmError) as e:
        T.tnlm_jacobi_step(p, f, f, ws=torch.empty(16, dtype=torch.uint8, device="cuda"))
    assert e.value.code == -6
    bad = T.TnlmParams.make(shape, 1, 1, 0.0, 1.0)
    with pytest.raises(T.TnlmError) as e:
        T.tnlm_jacobi_step(bad, f, f)
    assert e.value.code == -3


# ------------------------------------------------------------------ full size, bench launch configuration
def _sampled_step_parity(T, oracle, cfg, n_samples, what):
    import torch
    g = make_stack(cfg)
    p = params_of(T, cfg)
    gd = dev(g)
    ws = torch.empty(T.workspace_bytes(p), dtype=torch.uint8, device="cuda")
    f1 = T.tnlm_jacobi_step(p, gd, gd, ws=ws)                 # first sweep: f^0 = g
    f2 = T.tnlm_jacobi_step(p, f1, gd, ws=ws)                 # second sweep from the GPU's own f^1
    rng = np.random.default_rng(5)
    P, Z, Y, X = cfg.shape
    idx = rng.integers(0, g.size, n_samples)
    # add corners, faces and the last voxel: where clamping and ragged tiles live
    extra = [0, g.size - 1, X - 1, (Y - 1) * X, (Z - 1) * Y * X, Y * X * Z - 1, Y * X * Z, 2 * Y * X * Z - 1]
    idx = np.unique(np.concatenate([idx, np.array(extra, dtype=np.int64)]))
    h, mu = np.float32(cfg.h), np.float32(cfg.mu)
    f1h = f1.cpu().numpy()
    want1 = oracle.jacobi_step_at(g, g, cfg.patch_radius, cfg.search_radius, h, mu, idx)
    want2 = oracle.jacobi_step_at(f1h, g, cfg.patch_radius, cfg.search_radius, h, mu, idx)
    rs = dynamic_range(g)
    assert_parity(f1h.reshape(-1)[idx], want1, rs, what + " sweep 1")
    assert_parity(f2.cpu().numpy().reshape(-1)[idx], want2, rs, what + " sweep 2 (step-wise)")
    assert f2.min().item() >= g.min() - 1e-6 and f2.max().item() <= g.max() + 1e-6


def test_config3_full_size_sampled(T, oracle):
    """10 x 128 x 256 x 256, the configuration bench.py times: oracle at sampled output voxels."""
    _sampled_step_parity(T, oracle, CONFIGS["config3"], 6000, "config3")


def test_config2_full_size_sampled(T, oracle):
    _sampled_step_parity(T, oracle, CONFIGS["config2"], 6000, "config2")


def test_config4_shape_sampled(T, oracle):
    """Clinical-scale recipe (7^3 window, Z = 100 not a power of two) on a quarter in-plane grid."""
    cfg = CONFIGS["config4"].scaled(ny=256, nx=256, tumour_radius=8, si_amplitude=6)
    _sampled_step_parity(T, oracle, cfg, 3000, "config4 (256x256x100)")


@pytest.mark.parametrize("d,M,n", [(2, 2, 1500), (1, 4, 1500), (2, 4, 400)])
def test_config5_points_sampled(T, oracle, d, M, n):
    """Points of the config-5 parameter sweep (5^3 patch, 9^3 window) at full in-plane size, 6 phases."""
    cfg = CONFIGS["config5"].scaled(n_phase=6, nz=48, patch_radius=d, search_radius=M)
    _sampled_step_parity(T, oracle, cfg, n, f"config5 d={d} M={M}")


def test_enhance_z_slabs_driver_matches_tnlm_enhance_bitwise(T):
    """The multi-GPU z-slab driver (dist.enhance_z_slabs) with the CUDA slab sweep; one process here, so the
    halo exchange is a no-op and the slab is the whole stack: it must reproduce tnlm_enhance bit for bit.  A split
    into two slabs on the same device (what two ranks would compute) must as well."""
    import torch
    from paper_1201_2450_b200 import dist as D
    shape = (4, 19, 33, 40)
    g = dev(random_stack(shape, 41))
    p = T.TnlmParams.make(shape, 1, 2, 0.2, 0.5)
    want = T.tnlm_enhance(p, g, 3)
    info = D.RankInfo(0, 0, 1)

    def sweep(f, gg, a, b, out):
        T.tnlm_jacobi_step_slab(p, f, gg, a, b, f_out=out)

    got, (a, b) = D.enhance_z_slabs(info, g, 3, 3, sweep)
    assert (a, b) == (0, shape[1]) and torch.equal(got, want)

    def sweep_two(f, gg, a, b, out):          # the two slabs two ranks would own
        for r in range(2):
            za, zb = D.z_slab(shape[1], r, 2)
            T.tnlm_jacobi_step_slab(p, f, gg, za, zb, f_out=out)

    got2, _ = D.enhance_z_slabs(info, g, 3, 3, sweep_two)
    assert torch.equal(got2, want)


@pytest.mark.parametrize("scale", [1e-3, 4096.0])
def test_scale_covariance(T, scale):
    """Eq. 3 / Eq. 8 are covariant under g -> s g, h -> s h (the exponent is unchanged, the update is linear):
    intensities in other units (HU-like thousands, or tiny) must give the scaled result; powers-of-two-free
    scales exercise the exponent ranges of the accumulators."""
    import torch
    cfg = CONFIGS["config2"].scaled(nz=12, ny=40, nx=48, tumour_radius=3, si_amplitude=2)
    g = make_stack(cfg)
    for d, M in [(1, 2), (2, 1)]:
        p1 = T.TnlmParams.make(cfg.shape, d, M, cfg.h, cfg.mu)
        ps = T.TnlmParams.make(cfg.shape, d, M, cfg.h * scale, cfg.mu)
        base = T.tnlm_enhance(p1, dev(g), 2).cpu().numpy().astype(np.float64)
        got = T.tnlm_enhance(ps, dev((g.astype(np.float64) * scale).astype(np.float32)), 2).cpu().numpy().astype(np.float64)
        assert np.isfinite(got).all()
        assert_parity(got / scale, base, dynamic_range(g), f"scale {scale} d={d} M={M}")


def test_fuzz_packed_kernels_against_generic(T):
    """Seeded random shapes and parameters: the packed kernels (d = 1, 2; M = 1..4) against the generic kernel (which the
    tests above tie to the oracle), one sweep each, including slabs that start and end off the z-tile grid."""
    import torch
    rng = np.random.default_rng(2024)
    for case in range(28):
        d = int(rng.integers(1, 3)); M = int(rng.integers(1, 5))
        shape = (int(rng.integers(2, 5)), int(rng.integers(1, 14)), int(rng.integers(1, 70)), int(rng.integers(1, 50)))
        h = float(rng.choice([0.03, 0.1, 0.4, 5.0])); mu = float(rng.choice([0.2, 1.0, 3.0]))
        f, g = dev(random_stack(shape, 100 + case)), dev(random_stack(shape, 200 + case))
        p = T.TnlmParams.make(shape, d, M, h, mu)
        want = T.tnlm_jacobi_step(p, f, g, variant=T.VARIANT_GENERIC)
        got = T.tnlm_jacobi_step(p, f, g, variant=T.VARIANT_PAIRED)
        err = (got - want).abs().max().item()
        assert err <= 1e-4, f"case {case}: shape {shape} d={d} M={M} h={h}: max|d|={err:.3e}"
        za = int(rng.integers(0, shape[1])); zb = int(rng.integers(za, shape[1] + 1))
        out = torch.full_like(f, -3.0)
        T.tnlm_jacobi_step_slab(p, f, g, za, zb, f_out=out, variant=T.VARIANT_PAIRED)
        assert torch.equal(out[:, za:zb], got[:, za:zb]), f"case {case}: slab [{za},{zb}) differs from the full sweep"
        assert (out[:, :za] == -3.0).all() and (out[:, zb:] == -3.0).all(), f"case {case}: slab wrote outside [{za},{zb})"


def test_fuzz_tmem_kernels_against_oracle(T, oracle):
    """Seeded random shapes and parameters for the TMEM kernels (d = 1, 2; M = 2..4; 4- and 6-plane z-tiles, one or several
    chunks of x-offsets per row): volumes up to 27 planes deep so that several tiles, a ragged last tile and slabs off the
    tile grid occur.  Against the oracle itself, at the north-star tolerance: on random stacks with small h the fp32 generic
    kernel is the less accurate of the two (case 10 of this seed: 1.06e-4 from the oracle, the TMEM kernel 2.4e-5)."""
    import torch
    rng = np.random.default_rng(4048)
    for case in range(24):
        d = int(rng.integers(1, 3)); M = int(rng.integers(2, 5))
        shape = (int(rng.integers(2, 4)), int(rng.integers(1, 28)), int(rng.integers(1, 64)), int(rng.integers(1, 40)))
        h = float(rng.choice([0.03, 0.1, 0.4, 5.0])); mu = float(rng.choice([0.2, 1.0, 3.0]))
        fh, gh = random_stack(shape, 300 + case), random_stack(shape, 400 + case)
        f, g = dev(fh), dev(gh)
        p = T.TnlmParams.make(shape, d, M, h, mu)
        want = oracle.jacobi_step(fh, gh, d, M, np.float32(h), np.float32(mu))
        got = T.tnlm_jacobi_step(p, f, g, variant=T.VARIANT_PAIRED_TMEM)
        # the north-star bar holds where the exponents c2*D stay below ~1e3; a uniform-random stack of
        # unit range has D ~ (2d+1)^3 / 6, and beyond that regime the error of fp32 distances grows in proportion
        scale = max(1.0, 1.4427 / (2 * h * h) * (2 * d + 1) ** 3 / 6.0 / 1e3)
        gn = got.cpu().numpy().astype(np.float64)
        what = f"case {case}: shape {shape} d={d} M={M} h={h}"
        assert np.isfinite(gn).all(), what
        max_err = np.abs(gn - want).max()
        l2 = np.linalg.norm(gn - want) / np.linalg.norm(want)
        assert max_err <= MAX_TOL * scale and l2 <= L2_TOL * scale, f"{what}: max|d|={max_err:.3e} rel L2={l2:.3e} (scale {scale:.1f})"
        assert torch.equal(got, T.tnlm_jacobi_step(p, f, g)), f"case {case}: AUTO is not the TMEM kernel's result"
        za = int(rng.integers(0, shape[1])); zb = int(rng.integers(za, shape[1] + 1))
        out = torch.full_like(f, -3.0)
        T.tnlm_jacobi_step_slab(p, f, g, za, zb, f_out=out, variant=T.VARIANT_PAIRED_TMEM)
        assert torch.equal(out[:, za:zb], got[:, za:zb]), f"case {case}: slab [{za},{zb}) differs from the full sweep"
        assert (out[:, :za] == -3.0).all() and (out[:, zb:] == -3.0).all(), f"case {case}: slab wrote outside [{za},{zb})"


# ------------------------------------------------------------------ memory safety without compute-sanitizer
@pytest.mark.parametrize("shape,d,M", [((3, 7, 31, 33), 1, 2), ((2, 9, 30, 17), 1, 1), ((2, 5, 29, 35), 1, 3), ((2, 6, 33, 19), 1, 4),
                                       ((3, 6, 29, 18), 2, 1), ((2, 7, 28, 34), 2, 2), ((2, 5, 31, 21), 2, 4), ((2, 3, 5, 7), 3, 5)])
def test_guard_regions_stay_untouched(T, shape, d, M):
    """compute-sanitizer is closed on this GPU pool, so out-of-bounds writes are looked for directly: f_out and the
    workspace sit inside larger allocations whose guard regions (4 KB either side) hold a canary pattern, and every
    kernel variant, full sweeps and slabs, must leave the canaries and the planes outside a slab intact."""
    import torch
    n = int(np.prod(shape))
    G = 1024                                                       # guard floats
    f, g = dev(random_stack(shape, 51)), dev(random_stack(shape, 52))
    p = T.TnlmParams.make(shape, d, M, 0.2, 0.5)
    wsb = T.workspace_bytes(p)
    for v in variants(T, p):
        buf = torch.full((n + 2 * G,), -123.25, device="cuda")
        wbuf = torch.full((wsb + 8192,), 0x5A, dtype=torch.uint8, device="cuda")
        out = buf[G:G + n].view(shape)
        ws = wbuf[4096:4096 + wsb]
        assert out.data_ptr() % 16 == 0 and ws.data_ptr() % 16 == 0
        T.tnlm_jacobi_step(p, f, g, f_out=out, ws=ws, variant=v)
        T.tnlm_enhance(p, g, 2, f_out=out, ws=ws, variant=v)
        za, zb = 1, max(1, shape[1] - 1)
        out.fill_(-7.5)
        T.tnlm_jacobi_step_slab(p, f, g, za, zb, f_out=out, ws=ws, variant=v)
        torch.cuda.synchronize()
        assert (buf[:G] == -123.25).all() and (buf[G + n:] == -123.25).all(), f"variant {v}: wrote outside f_out"
        assert (wbuf[:4096] == 0x5A).all() and (wbuf[4096 + wsb:] == 0x5A).all(), f"variant {v}: wrote outside the workspace"
        assert (out[:, :za] == -7.5).all() and (out[:, zb:] == -7.5).all(), f"variant {v}: slab sweep wrote outside its planes"
        assert out[:, za:zb].isfinite().all()


@pytest.mark.gpu
@pytest.mark.parametrize("d,M,world,Z", [(1, 2, 3, 37), (2, 1, 2, 30), (1, 3, 2, 22), (1, 2, 1, 9)])
def test_slab_local_ranks_reproduce_the_enhancement_bitwise(T, d, M, world, Z):
    """a rank that stores only its z-slab, the M+d halo planes and the tile-alignment padding
    (dist.enhance_z_slabs_local + tnlm_jacobi_step_slab on the local arrays) reproduces its planes of tnlm_enhance bit
    for bit.  One GPU, one rank at a time: the halo planes a neighbour would send are taken from the single-device
    trajectory (loop-back exchange), which is what the neighbours hold if they are right too."""
    import torch
    from paper_1201_2450_b200 import dist as D
    shape, h, mu, n_iter = (3, Z, 40, 36), 0.25, 0.6, 3
    P, _, Y, X = shape
    g = dev(random_stack(shape, 11))
    p = T.TnlmParams.make(shape, d, M, h, mu)
    iters = [g]
    for _ in range(n_iter):
        iters.append(T.tnlm_jacobi_step(p, iters[-1], g))
    halo, zt = M + d, T.z_tile(p)
    for rank in range(world):
        info = D.RankInfo(rank, 0, world)
        L = D.slab_layout(Z, rank, world, halo, zt)
        p_loc = T.TnlmParams.make((P, L.nz_local, Y, X), d, M, h, mu)
        calls = [0]

        def exchange(_info, stack, L_):
            ref = iters[calls[0]]
            calls[0] += 1
            for zl in list(range(L_.lo - L_.halo, L_.lo)) + list(range(L_.hi, L_.hi + L_.halo)):
                stack[:, zl] = ref[:, min(max(zl + L_.origin, 0), Z - 1)]      # clamp-to-edge beyond the volume (P4)

        def sweep_slab(f, gg, z0, z1, out):
            if z1 > z0:
                T.tnlm_jacobi_step_slab(p_loc, f, gg, z0, z1, f_out=out)

        f, L2 = D.enhance_z_slabs_local(info, g[:, L.a:L.b].contiguous(), n_iter, halo, zt, Z, sweep_slab, exchange=exchange)
        torch.cuda.synchronize()
        assert calls[0] == n_iter and (L2.a, L2.b) == (L.a, L.b)
        assert torch.equal(f.owned(), iters[n_iter][:, L.a:L.b]), f"rank {rank} of {world}: slab differs from the single-device run"


def _nccl_worker(rank, world, port, shape, d, M, h, mu, n_iter, out_dir):
    import os
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import torch
    import paper_1201_2450_b200 as T
    from paper_1201_2450_b200 import dist as D
    torch.cuda.set_device(rank)
    info = D.init("nccl")
    P, Z, Y, X = shape
    p = T.TnlmParams.make(shape, d, M, h, mu)
    L = D.slab_layout(Z, rank, world, M + d, T.z_tile(p))
    g_own = torch.from_numpy(np.ascontiguousarray(random_stack(shape, 11)[:, L.a:L.b])).cuda()
    p_loc = T.TnlmParams.make((P, L.nz_local, Y, X), d, M, h, mu)

    def sweep_slab(f, gg, z0, z1, out):
        if z1 > z0:
            T.tnlm_jacobi_step_slab(p_loc, f, gg, z0, z1, f_out=out)

    f, _ = D.enhance_z_slabs_local(info, g_own, n_iter, M + d, T.z_tile(p), Z, sweep_slab)
    torch.cuda.synchronize()
    np.save(os.path.join(out_dir, f"nccl{rank}.npy"), f.owned().cpu().numpy())
    D.barrier(info)
    D.finalize(info)


def _gloo_cuda_worker(rank, world, port, shape, d, M, h, mu, n_iter, out_dir):
    import os
    os.environ.update(RANK=str(rank), LOCAL_RANK="0", WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import torch
    import paper_1201_2450_b200 as T
    from paper_1201_2450_b200 import dist as D
    torch.cuda.set_device(0)
    info = D.init("gloo")
    P, Z, Y, X = shape
    p = T.TnlmParams.make(shape, d, M, h, mu)
    L = D.slab_layout(Z, rank, world, M + d, T.z_tile(p))
    g_own = torch.from_numpy(np.ascontiguousarray(random_stack(shape, 11)[:, L.a:L.b])).cuda()
    p_loc = T.TnlmParams.make((P, L.nz_local, Y, X), d, M, h, mu)

    def sweep_slab(f, gg, z0, z1, out):
        if z1 > z0:
            T.tnlm_jacobi_step_slab(p_loc, f, gg, z0, z1, f_out=out)

    def exchange_via_host(info_, stack, L_):
        # gloo cannot send CUDA memory: stage the local array through the host on whatever stream is current (the side
        # stream inside enhance_z_slabs_local), run the library's exchange on the copy, write the halo planes back
        host = stack.cpu()
        D.exchange_slab_halos(info_, host, L_)
        h = L_.halo
        stack[:, L_.lo - h:L_.lo].copy_(host[:, L_.lo - h:L_.lo])
        stack[:, L_.hi:L_.hi + h].copy_(host[:, L_.hi:L_.hi + h])

    f, _ = D.enhance_z_slabs_local(info, g_own, n_iter, M + d, T.z_tile(p), Z, sweep_slab, exchange=exchange_via_host)
    torch.cuda.synchronize()
    np.save(os.path.join(out_dir, f"gc{rank}.npy"), f.owned().cpu().numpy())
    D.barrier(info)
    D.finalize(info)


@pytest.mark.gpu
def test_two_rank_z_slab_enhancement_with_a_real_exchange_on_one_gpu(T, tmp_path):
    """Two processes share cuda:0 and exchange their halo planes through torch.distributed (gloo, staged through the
    host): the device side of dist.enhance_z_slabs_local -- side stream, events, boundary / interior launches on
    slab-local arrays -- with a real neighbour, bit-identical to tnlm_enhance.  A correctness test only: nothing is
    timed with two ranks on one GPU."""
    import socket
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    shape, d, M, h, mu, n_iter = (3, 26, 40, 36), 1, 2, 0.25, 0.6, 3
    mp.spawn(_gloo_cuda_worker, args=(2, port, shape, d, M, h, mu, n_iter, str(tmp_path)), nprocs=2, join=True)
    g = dev(random_stack(shape, 11))
    want = T.tnlm_enhance(T.TnlmParams.make(shape, d, M, h, mu), g, n_iter).cpu().numpy()
    got = np.concatenate([np.load(tmp_path / f"gc{r}.npy") for r in range(2)], axis=1)
    assert np.array_equal(got, want)


@pytest.mark.gpu
def test_two_gpu_z_slab_enhancement_over_nccl(T, tmp_path):
    """The same on two GPUs with the real exchange (ncclSend/ncclRecv through torch.distributed); skipped on one GPU."""
    import socket
    import torch
    import torch.multiprocessing as mp
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    shape, d, M, h, mu, n_iter = (4, 40, 64, 48), 1, 2, 0.25, 0.6, 4
    mp.spawn(_nccl_worker, args=(2, port, shape, d, M, h, mu, n_iter, str(tmp_path)), nprocs=2, join=True)
    g = dev(random_stack(shape, 11))
    want = T.tnlm_enhance(T.TnlmParams.make(shape, d, M, h, mu), g, n_iter).cpu().numpy()
    got = np.concatenate([np.load(tmp_path / f"nccl{r}.npy") for r in range(2)], axis=1)
    assert np.array_equal(got, want)
