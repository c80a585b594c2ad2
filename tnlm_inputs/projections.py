"""Seeded synthetic cone-beam projection data for the TNLM-R workload: geometry, view angles per phase,
and ANALYTIC line integrals of an ellipsoid phantom.  Input generation only: no TNLM arithmetic and no discretised
projector lives here (the projection operator P_i of the method is in the oracle and in the CUDA library, separately).

The paper's phantom study: 128^3 voxels of 0.2 cm, 10 phases, 300 projections over 360 degrees (30 per phase, equally
spaced, the phases interleaved), source-to-isocentre 100 cm, source-to-detector 153.6 cm, 512 x 512 detector pixels of
0.08 cm.  `paper_geometry(scale)` shrinks volume and detector together for tests.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class ConeGeometry:
    vol_shape: tuple          # (nz, ny, nx)
    voxel: float
    n_view: int               # views per phase
    nu: int
    nv: int
    du: float
    dv: float
    sid: float
    sdd: float


def paper_geometry(n=128, n_view=30, det=512):
    """PAPER.md:245 at n = 128, det = 512; smaller n / det keep the field of view (voxel and pixel sizes grow)."""
    return ConeGeometry((n, n, n), 25.6 / n, n_view, det, det, 40.96 / det, 40.96 / det, 100.0, 153.6)


def phase_angles(n_phase, n_view):
    """Gantry angles [n_phase][n_view]: n_phase * n_view views equally spaced over 360 degrees, dealt to the phases in
    turn (view m belongs to phase m mod n_phase), so every phase gets n_view views equally spaced in a full rotation
     and the phases' angle sets are interleaved (the streak directions differ between phases)."""
    m = np.arange(n_phase * n_view)
    theta = 2.0 * np.pi * m / (n_phase * n_view)
    return np.stack([theta[m % n_phase == p] for p in range(n_phase)]).astype(np.float64)


def thorax_ellipsoids(phase, n_phase, fov=25.6):
    """(centre xyz, semi-axes xyz, density increment) of a small thorax: body, two lungs, spine, a tumour that moves
    along z with cos^4 breathing.  Lengths in the volume's units (cm), isocentre at the origin."""
    s = fov / 2.0
    zt = 0.25 * s * (np.cos(np.pi * phase / n_phase) ** 4 - 0.5)
    return [
        ((0.0, 0.0, 0.0), (0.90 * s, 0.70 * s, 0.95 * s), 0.20),
        ((-0.40 * s, 0.0, 0.0), (0.28 * s, 0.40 * s, 0.80 * s), -0.18),
        ((0.40 * s, 0.0, 0.0), (0.28 * s, 0.40 * s, 0.80 * s), -0.18),
        ((0.0, 0.45 * s, 0.0), (0.10 * s, 0.10 * s, 0.90 * s), 0.80),
        ((0.40 * s, -0.05 * s, zt), (0.09 * s, 0.09 * s, 0.09 * s), 0.23),
    ]


def voxelise(geom: ConeGeometry, ellipsoids):
    """The phantom sampled at voxel centres, [nz][ny][nx] float32."""
    nz, ny, nx = geom.vol_shape
    z = (np.arange(nz) - 0.5 * (nz - 1)) * geom.voxel
    y = (np.arange(ny) - 0.5 * (ny - 1)) * geom.voxel
    x = (np.arange(nx) - 0.5 * (nx - 1)) * geom.voxel
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    vol = np.zeros(geom.vol_shape, dtype=np.float64)
    for (cx, cy, cz), (ax, ay, az), rho in ellipsoids:
        vol += rho * ((((X - cx) / ax) ** 2 + ((Y - cy) / ay) ** 2 + ((Z - cz) / az) ** 2) <= 1.0)
    return vol.astype(np.float32)


def analytic_projections(geom: ConeGeometry, angles, ellipsoids):
    """Exact line integrals of the ellipsoid phantom along the rays source -> pixel centre, [n_view][nv][nu] float64.
    Chord of a ray with an ellipsoid: scale space by the semi-axes, intersect with the unit sphere."""
    u = (np.arange(geom.nu) - 0.5 * (geom.nu - 1)) * geom.du
    v = (np.arange(geom.nv) - 0.5 * (geom.nv - 1)) * geom.dv
    out = np.zeros((len(angles), geom.nv, geom.nu), dtype=np.float64)
    for k, th in enumerate(angles):
        c, s = np.cos(th), np.sin(th)
        S = np.array([geom.sid * c, geom.sid * s, 0.0])
        D = np.empty((geom.nv, geom.nu, 3))
        D[..., 0] = (geom.sid - geom.sdd) * c - u[None, :] * s
        D[..., 1] = (geom.sid - geom.sdd) * s + u[None, :] * c
        D[..., 2] = v[:, None]
        dirv = D - S
        dirv /= np.linalg.norm(dirv, axis=-1, keepdims=True)
        for (cx, cy, cz), (ax, ay, az), rho in ellipsoids:
            sc = np.array([ax, ay, az])
            o = (S - np.array([cx, cy, cz])) / sc
            w = dirv / sc
            A = (w * w).sum(-1)
            B = (w * o).sum(-1)
            Cq = (o * o).sum() - 1.0
            disc = B * B - A * Cq
            out[k] += rho * np.where(disc > 0.0, 2.0 * np.sqrt(np.maximum(disc, 0.0)) / A, 0.0)
    return out


def make_projection_stack(geom: ConeGeometry, n_phase, noise=0.0, seed=0):
    """(angles [P][n_view], y [P][n_view][nv][nu] float32, clean phantom [P][nz][ny][nx] float32)."""
    rng = np.random.default_rng(seed)
    ang = phase_angles(n_phase, geom.n_view)
    fov = geom.voxel * geom.vol_shape[2]
    ys, vols = [], []
    for p in range(n_phase):
        ell = thorax_ellipsoids(p, n_phase, fov)
        y = analytic_projections(geom, ang[p], ell)
        if noise > 0.0:
            y = y + noise * rng.standard_normal(y.shape)
        ys.append(y.astype(np.float32))
        vols.append(voxelise(geom, ell))
    return ang, np.stack(ys), np.stack(vols)
