"""Oracle for the paper's two image-quality metrics (test infrastructure; plain numpy, fp64).

  * CNR = 2 |S - S_b| / (sigma + sigma_b)
        S, S_b = mean voxel value in the ROI and in a nearby background region, sigma, sigma_b =
        standard deviation of the voxel values in the two regions.
  * SRR = [TV(f_FDK - f*) - TV(f_TNLME - f*)] / TV(f_FDK - f*),  TV(h) = int dx |grad h(x)|
                                                                            PAPER.md:269-272 Eq. 10
Readings where the paper is silent:
  M1  regions are axis-aligned half-open boxes [z0,z1) x [y0,y1) x [x0,x1) of one phase;
  M2  "standard deviation" is the population one (divide by N);
  M3  TV is discretised with forward differences at unit voxel spacing, a difference that would reach
      outside the volume is 0 (replicate boundary), |grad h| = sqrt(hx^2 + hy^2 + hz^2) (isotropic),
      the integral is the plain sum over the voxels of one phase.
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module; it shares
no code with paper_1201_2450_b200/.
"""
from __future__ import annotations

import numpy as np


def tv_phase(h: np.ndarray) -> float:
    """TV(h) of ONE volume [Z][Y][X] (Eq. 10, reading M3), written as the definition."""
    h = np.asarray(h, dtype=np.float64)
    gz = np.zeros_like(h)
    gy = np.zeros_like(h)
    gx = np.zeros_like(h)
    gz[:-1, :, :] = h[1:, :, :] - h[:-1, :, :]
    gy[:, :-1, :] = h[:, 1:, :] - h[:, :-1, :]
    gx[:, :, :-1] = h[:, :, 1:] - h[:, :, :-1]
    return float(np.sqrt(gx * gx + gy * gy + gz * gz).sum())


def tv_diff(a: np.ndarray, b: np.ndarray | None = None) -> np.ndarray:
    """TV(a_p - b_p) for every phase p of two [P][Z][Y][X] stacks (b = None: TV(a_p)) -> fp64 [P]."""
    a = np.asarray(a, dtype=np.float64)
    d = a if b is None else a - np.asarray(b, dtype=np.float64)
    return np.array([tv_phase(d[p]) for p in range(d.shape[0])])


def srr(f_fdk: np.ndarray, f_enh: np.ndarray, f_star: np.ndarray) -> np.ndarray:
    """Streak-reduction ratio of Eq. 10 for every phase -> fp64 [P]."""
    t0 = tv_diff(f_fdk, f_star)
    t1 = tv_diff(f_enh, f_star)
    return (t0 - t1) / t0


def roi_stats(stack: np.ndarray, phase: int, box) -> tuple[float, float]:
    """(mean, population standard deviation) of the voxels of `phase` inside the half-open box (M1, M2)."""
    z0, z1, y0, y1, x0, x1 = (int(v) for v in box)
    v = np.asarray(stack[phase, z0:z1, y0:y1, x0:x1], dtype=np.float64).reshape(-1)
    mean = v.sum() / v.size
    return float(mean), float(np.sqrt(((v - mean) ** 2).sum() / v.size))


def cnr(stack: np.ndarray, phase: int, roi, roi_bg) -> np.ndarray:
    """[S, sigma, S_b, sigma_b, CNR] with CNR = 2 |S - S_b| / (sigma + sigma_b)."""
    s, sd = roi_stats(stack, phase, roi)
    sb, sdb = roi_stats(stack, phase, roi_bg)
    return np.array([s, sd, sb, sdb, 2.0 * abs(s - sb) / (sd + sdb)])
