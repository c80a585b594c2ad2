"""Pins of the metrics oracle (oracle/tnlm_metrics.py) against what the definitions fix:
closed forms, hand-computed tiny cases, invariances, and the direction of PAPER.md Table 1."""
import numpy as np
import pytest

from oracle import tnlm_metrics as Q
from tnlm_inputs import CONFIGS, make_stack


def test_tv_of_a_linear_ramp_closed_form():
    Z, Y, X = 5, 6, 7
    al, be, ga = 0.3, -1.1, 0.7           # slopes along x, y, z
    z, y, x = np.meshgrid(np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    h = al * x + be * y + ga * z + 2.0
    # forward differences vanish on the last index of their axis: count voxels by which components survive
    want = 0.0
    for hz in (0, 1):
        for hy in (0, 1):
            for hx in (0, 1):
                n = ((Z - 1) if hz else 1) * ((Y - 1) if hy else 1) * ((X - 1) if hx else 1)
                want += n * np.sqrt(hx * al * al + hy * be * be + hz * ga * ga)
    assert Q.tv_phase(h) == pytest.approx(want, rel=1e-13)


def test_tv_hand_computed_2x2x2():
    h = np.zeros((2, 2, 2))
    h[1, 1, 1] = 1.0
    # only voxels (0,1,1), (1,0,1), (1,1,0) see one unit forward difference each
    assert Q.tv_phase(h) == pytest.approx(3.0, abs=1e-15)
    h[0, 0, 0] = 2.0     # voxel (0,0,0): differences (-2,-2,-2) -> 2 sqrt 3
    assert Q.tv_phase(h) == pytest.approx(3.0 + 2.0 * np.sqrt(3.0), rel=1e-14)


def test_tv_invariances():
    rng = np.random.default_rng(0)
    h = rng.standard_normal((4, 5, 6))
    t = Q.tv_phase(h)
    assert Q.tv_phase(np.full((3, 4, 5), 7.0)) == 0.0
    assert Q.tv_phase(h + 3.5) == pytest.approx(t, rel=1e-12)            # constants do not count
    assert Q.tv_phase(-2.0 * h) == pytest.approx(2.0 * t, rel=1e-12)     # absolutely homogeneous
    assert Q.tv_phase(h[::-1, ::-1, ::-1].transpose(2, 1, 0)) != 0.0
    a = rng.standard_normal((3, 4, 5, 6)); b = rng.standard_normal((3, 4, 5, 6))
    assert np.allclose(Q.tv_diff(a, b), [Q.tv_phase(a[p] - b[p]) for p in range(3)], rtol=1e-14)
    assert np.allclose(Q.tv_diff(a), [Q.tv_phase(a[p]) for p in range(3)], rtol=1e-14)


def test_srr_special_cases():
    rng = np.random.default_rng(1)
    star = rng.standard_normal((2, 4, 5, 6)); fdk = star + 0.3 * rng.standard_normal(star.shape)
    assert np.allclose(Q.srr(fdk, star, star), 1.0)                       # all streaks removed
    assert np.allclose(Q.srr(fdk, fdk, star), 0.0)                        # nothing removed
    half = star + 0.5 * (fdk - star)
    assert np.allclose(Q.srr(fdk, half, star), 0.5, rtol=1e-12)           # TV is homogeneous: half the residual


def test_cnr_hand_computed():
    s = np.zeros((2, 3, 4, 8))
    s[1, 0:2, 0:2, 0:2] = np.array([1.0, 3.0] * 4).reshape(2, 2, 2)      # ROI: mean 2, population std 1
    s[1, 0:2, 0:2, 4:8] = np.array([5.0, 5.0, 7.0, 7.0] * 4).reshape(2, 2, 4)   # background: mean 6, std 1
    out = Q.cnr(s, 1, (0, 2, 0, 2, 0, 2), (0, 2, 0, 2, 4, 8))
    assert np.allclose(out, [2.0, 1.0, 6.0, 1.0, 2.0 * 4.0 / 2.0], rtol=1e-15)
    m, sd = Q.roi_stats(s, 1, (0, 2, 0, 2, 0, 2))
    v = s[1, 0:2, 0:2, 0:2].ravel()
    assert m == pytest.approx(v.mean()) and sd == pytest.approx(v.std(ddof=0))


def test_metrics_move_the_way_the_paper_reports(oracle):
    """PAPER.md:316-327 (Table 1): TNLM-E removes most streak energy (SRR well above 0) and raises the
    CNR of the tumour.  Same direction on the small synthetic thorax stack."""
    cfg = CONFIGS["config2"].scaled(nz=24, ny=64, nx=64, tumour_radius=4, si_amplitude=3)
    g = make_stack(cfg)
    star = make_stack(cfg, clean=True)
    f = oracle.enhance(g, cfg.patch_radius, cfg.search_radius, np.float32(cfg.h), np.float32(cfg.mu), 3)
    s = Q.srr(g, f, star)
    assert (s > 0.2).all() and (s < 1.0).all()
    # tumour ROI vs lung background in phase 0 (same region the phantom recipe paints)
    P, Z, Y, X = cfg.shape
    cz, cy, cx = (Z - 1) / 2, (Y - 1) / 2, (X - 1) / 2
    tz = int(round(cz - cfg.si_amplitude / 2 + cfg.si_amplitude)); ty = int(round(cy - 0.03 * Y)); tx = int(round(cx + 0.20 * X))
    roi = (tz - 1, tz + 2, ty - 1, ty + 2, tx - 1, tx + 2)
    bg = (tz - 1, tz + 2, ty + 6, ty + 9, tx - 1, tx + 2)
    assert Q.cnr(f, 0, roi, bg)[4] > Q.cnr(g, 0, roi, bg)[4]
