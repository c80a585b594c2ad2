"""Seeded synthetic 4D-CBCT phantom stacks (the ONLY inputs of tests and bench).

This module holds no TNLM arithmetic: it only paints phantoms, streaks and noise.
Both the CPU oracle (``oracle/``) and the CUDA path (``paper_1201_2450_b200/``) are fed
from here; neither imports the other.

What the stacks stand in for: the paper's workloads are 10-phase 128^3 thorax 4D-CBCT
stacks reconstructed by FDK from 30-60 views per phase (section 2.5):
smooth anatomy, a tumour that moves with breathing, view-aliasing streaks whose
directions differ from phase to phase, and noise.  The NCAT phantom and
the patient scan are not available; the recipes below (SURVEY.md section 8(d),
BASELINE.json ``configs``) reproduce that structure.  Everything is generated in
float64 from ``numpy.random.default_rng(seed)`` and cast to float32 last.

Layout of every returned stack: ``[phase][z][y][x]`` float32, C-contiguous.
"""
from __future__ import annotations

from dataclasses import dataclass, replace
import math

import numpy as np


@dataclass(frozen=True)
class TnlmConfig:
    """One BASELINE.json config: stack shape, TNLM parameters and the phantom recipe."""

    name: str
    n_phase: int
    nz: int
    ny: int
    nx: int
    patch_radius: int      # d : patch edge 2d+1
    search_radius: int     # M : window edge 2M+1
    h: float               # Eq. 3
    mu: float              # Eq. 4
    n_iter: int            # TNLM-E iterations
    seed: int
    kind: str              # "ellipsoid" (config 1) | "thorax" (configs 2-5)
    # thorax-only recipe numbers
    tumour_radius: float = 0.0
    si_amplitude: float = 0.0
    n_angles: int = 0
    streak_amp: float = 0.0
    sigma: float = 0.0
    lung_texture: bool = False
    breath_phases: int = 10

    @property
    def shape(self):
        return (self.n_phase, self.nz, self.ny, self.nx)

    @property
    def voxels_per_phase(self):
        return self.nz * self.ny * self.nx

    @property
    def n_offsets(self):
        return (2 * self.search_radius + 1) ** 3

    @property
    def updates_per_sweep(self):
        """Voxel-offset updates U = 2 P V (2M+1)^3 of one Gauss-Jacobi sweep."""
        return 2 * self.n_phase * self.voxels_per_phase * self.n_offsets

    def scaled(self, **kw) -> "TnlmConfig":
        return replace(self, **kw)


# BASELINE.json configs[0..4] (1-based names as in SURVEY.md section 8).
CONFIGS = {
    "config1": TnlmConfig("config1", 10, 16, 32, 32, 1, 1, 0.1, 1.0, 3, 0, "ellipsoid",
                          sigma=0.05),
    "config2": TnlmConfig("config2", 10, 64, 128, 128, 1, 2, 0.05, 0.5, 5, 1, "thorax",
                          tumour_radius=6, si_amplitude=5, n_angles=30, streak_amp=0.05,
                          sigma=0.03),
    "config3": TnlmConfig("config3", 10, 128, 256, 256, 1, 2, 0.05, 0.5, 10, 2, "thorax",
                          tumour_radius=10, si_amplitude=8, n_angles=40, streak_amp=0.05,
                          sigma=0.03),
    "config4": TnlmConfig("config4", 10, 100, 512, 512, 1, 3, 0.06, 0.5, 10, 3, "thorax",
                          tumour_radius=15, si_amplitude=12, n_angles=35, streak_amp=0.08,
                          sigma=0.04, lung_texture=True),
    # config 5 is a sweep over (d, M); this entry carries the stack recipe, d/M are
    # overridden per sweep point with .scaled(patch_radius=..., search_radius=...).
    "config5": TnlmConfig("config5", 20, 128, 256, 256, 1, 2, 0.05, 0.5, 5, 4, "thorax",
                          tumour_radius=10, si_amplitude=8, n_angles=40, streak_amp=0.05,
                          sigma=0.03, breath_phases=20),
}


def _grid(nz, ny, nx):
    z = np.arange(nz, dtype=np.float64)[:, None, None]
    y = np.arange(ny, dtype=np.float64)[None, :, None]
    x = np.arange(nx, dtype=np.float64)[None, None, :]
    c = ((nx - 1) / 2.0, (ny - 1) / 2.0, (nz - 1) / 2.0)
    return z, y, x, c


def _ellipsoid(z, y, x, centre, semi):
    cx, cy, cz = centre
    ax, ay, az = semi
    return ((x - cx) / ax) ** 2 + ((y - cy) / ay) ** 2 + ((z - cz) / az) ** 2 <= 1.0


def _clean_ellipsoid(cfg: TnlmConfig) -> np.ndarray:
    """Config 1: ellipsoid 1.0 on background 0.2 holding a moving sphere of 1.5."""
    P, Z, Y, X = cfg.shape
    z, y, x, c = _grid(Z, Y, X)
    out = np.empty(cfg.shape, dtype=np.float64)
    body = _ellipsoid(z, y, x, c, (0.40 * X, 0.40 * Y, 0.45 * Z))
    for p in range(P):
        vol = np.full((Z, Y, X), 0.2)
        vol[body] = 1.0
        zc = c[2] + 3.0 * math.sin(2.0 * math.pi * p / 10.0)
        vol[_ellipsoid(z, y, x, (c[0], c[1], zc), (4.0, 4.0, 4.0))] = 1.5
        out[p] = vol
    return out


def _tumour_centre(cfg: TnlmConfig, p: int, c):
    _, Z, Y, X = cfg.shape
    A = cfg.si_amplitude
    zc = c[2] - A / 2.0 + A * math.cos(math.pi * p / cfg.breath_phases) ** 4
    return (c[0] + 0.20 * X, c[1] - 0.03 * Y, zc)


def _clean_thorax(cfg: TnlmConfig, rng) -> np.ndarray:
    """Thorax phantom (configs 2-5).  ``rng`` is consumed only for the lung texture."""
    P, Z, Y, X = cfg.shape
    z, y, x, c = _grid(Z, Y, X)
    body = _ellipsoid(z, y, x, c, (0.45 * X, 0.35 * Y, 0.90 * Z))
    lung_l = _ellipsoid(z, y, x, (c[0] - 0.20 * X, c[1] - 0.03 * Y, c[2]),
                        (0.14 * X, 0.20 * Y, 0.42 * Z))
    lung_r = _ellipsoid(z, y, x, (c[0] + 0.20 * X, c[1] - 0.03 * Y, c[2]),
                        (0.14 * X, 0.20 * Y, 0.42 * Z))
    lungs = lung_l | lung_r
    spine = (((x - c[0]) ** 2 + (y - (c[1] + 0.22 * Y)) ** 2) <= (0.05 * X) ** 2) & body
    static = np.zeros((Z, Y, X))
    static[body] = 0.2
    static[lungs] = 0.02
    static[spine] = 1.0
    texture = None
    if cfg.lung_texture:
        from scipy.ndimage import gaussian_filter
        field = gaussian_filter(rng.random((Z, Y, X)), sigma=2.0)
        field = (field - field.min()) / (field.max() - field.min()) * 0.05
        texture = np.where(lungs, field, 0.0)
    out = np.empty(cfg.shape, dtype=np.float64)
    for p in range(P):
        vol = static.copy()
        vol[_ellipsoid(z, y, x, _tumour_centre(cfg, p, c), (cfg.tumour_radius,) * 3)] = 0.25
        if texture is not None:
            vol += texture
        out[p] = vol
    return out


def _streaks(cfg: TnlmConfig, p: int, rng) -> np.ndarray:
    """In-plane streak pattern of phase ``p`` (constant along z), shape [ny][nx]."""
    _, Z, Y, X = cfg.shape
    _, yy, xx, c = _grid(Z, Y, X)
    yy = yy[0]
    xx = xx[0]
    n_a = cfg.n_angles
    jitter = rng.random(n_a)
    sign = rng.choice(np.array([-1.0, 1.0]), n_a)
    spine_xy = (c[0], c[1] + 0.22 * Y)
    tum = _tumour_centre(cfg, p, c)
    tum_xy = (tum[0], tum[1])
    r0 = 4.0 * X / 128.0
    acc = np.zeros((Y, X))
    for k in range(n_a):
        theta = math.pi * (k + jitter[k]) / n_a
        sx, sy = spine_xy if k % 2 == 0 else tum_xy
        # distance from (x, y) to the line through (sx, sy) with direction (cos, sin)
        dist = (xx - sx) * math.sin(theta) - (yy - sy) * math.cos(theta)
        r2 = (xx - sx) ** 2 + (yy - sy) ** 2
        acc += sign[k] * np.exp(-dist ** 2 / (2.0 * 0.7 ** 2)) * (1.0 - np.exp(-r2 / (2.0 * r0 ** 2)))
    return cfg.streak_amp * acc


def make_stack(cfg: TnlmConfig, *, clean: bool = False) -> np.ndarray:
    """Return the degraded stack ``g`` (or the clean phantom) as float32 [P][Z][Y][X].

    Draw order (fixed): [lung texture] -> per phase {random(n_a), choice(+-1, n_a)} ->
    Gaussian noise for the whole stack, drawn phase by phase (the generator's stream is
    sequential, so this equals one ``standard_normal(shape)`` call).
    """
    rng = np.random.default_rng(cfg.seed)
    if cfg.kind == "ellipsoid":
        vol = _clean_ellipsoid(cfg)
    elif cfg.kind == "thorax":
        vol = _clean_thorax(cfg, rng)
    else:
        raise ValueError(f"unknown phantom kind {cfg.kind!r}")
    if clean:
        return np.ascontiguousarray(vol.astype(np.float32))
    out = np.empty(cfg.shape, dtype=np.float32)
    if cfg.kind == "thorax":
        for p in range(cfg.n_phase):
            vol[p] += _streaks(cfg, p, rng)[None, :, :]
    for p in range(cfg.n_phase):
        noise = rng.standard_normal(cfg.shape[1:])
        out[p] = (vol[p] + cfg.sigma * noise).astype(np.float32)
    return np.ascontiguousarray(out)


def dynamic_range(g: np.ndarray) -> float:
    """``max g - min g``: the scale of the parity tolerance (BASELINE.json north_star)."""
    return float(g.max()) - float(g.min())


def random_stack(shape, seed: int, lo: float = 0.0, hi: float = 1.0) -> np.ndarray:
    """Plain uniform noise stack for edge-case tests (ragged extents, P=2, ...)."""
    rng = np.random.default_rng(seed)
    return np.ascontiguousarray((lo + (hi - lo) * rng.random(shape)).astype(np.float32))


def z_slab(n: int, rank: int, world: int):
    """Balanced contiguous split of ``n`` planes over ``world`` ranks -> (start, stop)."""
    base, rem = divmod(n, world)
    start = rank * base + min(rank, rem)
    return start, start + base + (1 if rank < rem else 0)
