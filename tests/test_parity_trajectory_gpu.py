"""Parity of the CUDA path with the CPU oracle over whole TNLM-E trajectories and at the real sizes of
BASELINE.json's configs (SURVEY.md section 8(d) "Parity at scale"), through the C ABI, in the launch
configuration bench.py times.  Bar (north_star): max|delta| <= 1e-4 x dynamic range, relative L2 <= 1e-5.

  config 2   full trajectory: oracle.enhance on the whole 10 x 64 x 128 x 128 stack, 5 sweeps, every voxel
  config 3   (a) every sweep's input is the GPU's own iterate (step-wise): sweeps 1, 5 and 10 at >= 1e5 random
                 voxels plus one complete z-plane of every phase (each output voxel is independent given f^k)
             (b) full 10-sweep trajectories of the oracle ALONE on two cropped sub-volumes: a voxel of f^K depends
                 on g only within K(M+d) voxels (Eq. 8 reads f within M+d of x), so inside a
                 crop every voxel further than K(M+d) = 30 from a cut face equals the full-volume trajectory; the
                 10-sweep result bench.py times is compared there with no GPU value fed to the oracle
             (c) the packed kernel against the generic kernel (tied to the oracle by test_parity_gpu.py) over EVERY
                 voxel of a sweep: the net for rare guard-band events that samples cannot catch
  config 4   real 10 x 100 x 512 x 512 size: step-wise at sweeps 1, 5, 10; packed vs generic over every voxel
  config 5   real 20 x 128 x 256 x 256 size, all eight (patch, window) points: step-wise at sweeps 1, 3, 5
"""
import functools

import numpy as np
import pytest

from tnlm_inputs import CONFIGS, make_stack as _make_stack, dynamic_range

pytestmark = pytest.mark.gpu

MAX_TOL = 1e-4     # x dynamic range of the input
L2_TOL = 1e-5


@pytest.fixture(scope="module")
def T():
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    import paper_1201_2450_b200 as T
    T.lib()
    return T


@functools.lru_cache(maxsize=1)
def _stack_of(name):
    return _make_stack(CONFIGS[name])


def make_stack(cfg):
    """The seeded stack of a BASELINE.json config (the recipe does not depend on d, M: sweep points share it)."""
    return _stack_of(cfg.name)


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def assert_parity(got, want, rng_scale, what):
    got = np.asarray(got, dtype=np.float64)
    want = np.asarray(want, dtype=np.float64)
    assert np.isfinite(got).all(), f"{what}: non-finite output"
    max_err = np.abs(got - want).max()
    l2 = np.linalg.norm(got - want) / max(np.linalg.norm(want), 1e-300)
    assert max_err <= MAX_TOL * rng_scale, f"{what}: max|d|={max_err:.3e} > {MAX_TOL * rng_scale:.3e}"
    assert l2 <= L2_TOL, f"{what}: rel L2={l2:.3e} > {L2_TOL}"
    return max_err, l2


def params_of(T, cfg):
    return T.TnlmParams.make(cfg.shape, cfg.patch_radius, cfg.search_radius, cfg.h, cfg.mu)


def gpu_iterates(T, p, gd, n_iter, keep):
    """f^k for k in `keep` (host arrays) from manual Gauss-Jacobi steps on the device, and f^n_iter (device)."""
    import torch
    ws = torch.empty(T.workspace_bytes(p), dtype=torch.uint8, device="cuda")
    out = {}
    f = gd
    for k in range(n_iter + 1):
        if k in keep:
            out[k] = f.cpu().numpy()
        if k < n_iter:
            f = T.tnlm_jacobi_step(p, f, gd, ws=ws)
    return out, f


def sample_indices(shape, n, seed, plane_z=None):
    """n random flat indices, the corners, and (optionally) every voxel of plane z of every phase."""
    P, Z, Y, X = shape
    size = P * Z * Y * X
    rng = np.random.default_rng(seed)
    parts = [rng.integers(0, size, n),
             np.array([0, size - 1, X - 1, (Y - 1) * X, (Z - 1) * Y * X, Z * Y * X - 1, Z * Y * X, 2 * Z * Y * X - 1])]
    if plane_z is not None:
        yx = np.arange(Y * X, dtype=np.int64)
        parts += [ph * Z * Y * X + plane_z * Y * X + yx for ph in range(P)]
    return np.unique(np.concatenate(parts).astype(np.int64))


def stepwise_parity(T, oracle, cfg, sweeps, n_samples, planes, what):
    """For k in `sweeps`: the oracle's Eq. 8 sweep from the GPU's own f^{k-1}, at sampled voxels, against the GPU's f^k."""
    import torch
    g = make_stack(cfg)
    p = params_of(T, cfg)
    gd = dev(g)
    keep = sorted({k - 1 for k in sweeps} | set(sweeps))
    it, f_last = gpu_iterates(T, p, gd, max(sweeps), keep)
    # the call bench.py times produces the same bits as the manual steps
    assert torch.equal(T.tnlm_enhance(p, gd, max(sweeps)), f_last), f"{what}: tnlm_enhance differs from manual steps"
    h, mu = np.float32(cfg.h), np.float32(cfg.mu)
    rs = dynamic_range(g)
    for k, pz in zip(sweeps, planes):
        idx = sample_indices(cfg.shape, n_samples, 100 + k, pz)
        want = oracle.jacobi_step_at(it[k - 1], g, cfg.patch_radius, cfg.search_radius, h, mu, idx)
        assert_parity(it[k].reshape(-1)[idx], want, rs, f"{what} sweep {k} ({idx.size} voxels)")
    last = it[max(sweeps)]
    assert last.min() >= g.min() - 1e-6 and last.max() <= g.max() + 1e-6, f"{what}: convex-combination bounds violated"


# ------------------------------------------------------------------ config 2: the whole trajectory, every voxel
def test_config2_full_trajectory(T, oracle):
    cfg = CONFIGS["config2"]
    g = make_stack(cfg)
    p = params_of(T, cfg)
    want = oracle.enhance(g, cfg.patch_radius, cfg.search_radius, np.float32(cfg.h), np.float32(cfg.mu), cfg.n_iter)
    got = T.tnlm_enhance(p, dev(g), cfg.n_iter).cpu().numpy()
    assert_parity(got, want, dynamic_range(g), "config2 full trajectory (5 sweeps, every voxel)")


# ------------------------------------------------------------------ config 3
def test_config3_stepwise_sweeps_1_5_10(T, oracle):
    cfg = CONFIGS["config3"]
    stepwise_parity(T, oracle, cfg, sweeps=(1, 5, 10), n_samples=100_000, planes=(cfg.nz // 2, 0, cfg.nz - 1), what="config3")


def crop_trajectory_parity(T, oracle, cfg, got_full, g, lo, hi, what):
    """Oracle trajectory on the crop [lo, hi) of all phases; compare where the crop's cut faces cannot have reached."""
    reach = cfg.n_iter * (cfg.search_radius + cfg.patch_radius)
    (z0, y0, x0), (z1, y1, x1) = lo, hi
    crop = np.ascontiguousarray(g[:, z0:z1, y0:y1, x0:x1])
    want = oracle.enhance(crop, cfg.patch_radius, cfg.search_radius, np.float32(cfg.h), np.float32(cfg.mu), cfg.n_iter)
    sl = []
    for a, b, n in ((z0, z1, cfg.nz), (y0, y1, cfg.ny), (x0, x1, cfg.nx)):
        va = 0 if a == 0 else reach             # a face that is a face of the volume is not a cut
        vb = (b - a) if b == n else (b - a) - reach
        assert vb > va, "crop too small for the dependence reach"
        sl.append(slice(va, vb))
    sub_want = want[:, sl[0], sl[1], sl[2]]
    sub_got = got_full[:, z0 + sl[0].start:z0 + sl[0].stop, y0 + sl[1].start:y0 + sl[1].stop, x0 + sl[2].start:x0 + sl[2].stop]
    assert sub_want.size > 0
    return assert_parity(sub_got, sub_want, dynamic_range(g), f"{what} ({sub_want.size} voxels of the 10-sweep result)")


def test_config3_full_trajectory_on_crops(T, oracle):
    cfg = CONFIGS["config3"]
    g = make_stack(cfg)
    p = params_of(T, cfg)
    got = T.tnlm_enhance(p, dev(g), cfg.n_iter).cpu().numpy()          # the 10-sweep result bench.py times
    # a corner of the volume (three volume faces: clamp-to-edge, reading P4) ...
    crop_trajectory_parity(T, oracle, cfg, got, g, (0, 0, 0), (40, 72, 72), "config3 corner crop")
    # ... and the moving tumour in the right lung (centre x = c_x + 0.20 X, y = c_y - 0.03 Y, z = c_z), the part of
    # the stack that changes most from phase to phase
    cz, cy, cx = (cfg.nz - 1) // 2, int((cfg.ny - 1) / 2 - 0.03 * cfg.ny), int((cfg.nx - 1) / 2 + 0.20 * cfg.nx)
    e = 38
    crop_trajectory_parity(T, oracle, cfg, got, g, (cz - e, cy - e, cx - e), (cz + e, cy + e, cx + e), "config3 tumour crop")


def every_voxel_packed_vs_generic(T, cfg, what):
    """One sweep from f^0 = g and one from f^1: the packed kernel (AUTO) against the generic kernel at every voxel."""
    g = make_stack(cfg)
    p = params_of(T, cfg)
    gd = dev(g)
    rs = dynamic_range(g)
    f = gd
    for k in (1, 2):
        a = T.tnlm_jacobi_step(p, f, gd, variant=T.VARIANT_AUTO)
        b = T.tnlm_jacobi_step(p, f, gd, variant=T.VARIANT_GENERIC)
        diff = (a.double() - b.double())
        max_err = diff.abs().max().item()
        l2 = (diff.norm() / b.double().norm()).item()
        assert bool(a.isfinite().all()), f"{what} sweep {k}: non-finite output"
        assert max_err <= MAX_TOL * rs and l2 <= L2_TOL, f"{what} sweep {k}: max|d|={max_err:.3e} relL2={l2:.3e} over every voxel"
        f = a


def test_config3_packed_vs_generic_every_voxel(T):
    every_voxel_packed_vs_generic(T, CONFIGS["config3"], "config3 packed vs generic")


# ------------------------------------------------------------------ config 4 at its real size
def test_config4_real_size_stepwise_sweeps_1_5_10(T, oracle):
    cfg = CONFIGS["config4"]
    stepwise_parity(T, oracle, cfg, sweeps=(1, 5, 10), n_samples=100_000, planes=(None, cfg.nz - 1, None), what="config4 (10x100x512x512)")


def test_config4_packed_vs_generic_every_voxel(T):
    every_voxel_packed_vs_generic(T, CONFIGS["config4"], "config4 packed vs generic")


# ------------------------------------------------------------------ config 5 at its real size, every sweep point
@pytest.mark.parametrize("d,M,n", [(1, 1, 100_000), (1, 2, 100_000), (1, 3, 60_000), (1, 4, 30_000),
                                   (2, 1, 60_000), (2, 2, 30_000), (2, 3, 12_000), (2, 4, 6_000)])
def test_config5_real_size_stepwise_sweeps_1_3_5(T, oracle, d, M, n):
    cfg = CONFIGS["config5"].scaled(patch_radius=d, search_radius=M)
    stepwise_parity(T, oracle, cfg, sweeps=(1, 3, 5), n_samples=n, planes=(None, None, None), what=f"config5 d={d} M={M}")
