"""Seeded synthetic inputs for the MBS hot path (shared by tests, bench and the oracle's callers).

This module holds NO arithmetic of the method (no k^2, no absorber, no operators): it only
produces refractive-index maps n(r), physical sources y(r) and seeded random vectors, as
complex64 numpy arrays, plus the geometry each BASELINE.json config fixes.  It imports neither
the CUDA binding nor the oracle.

The media stand in for the paper's PoreSpy sphere packings (section 4), which
are not available; the recipe is the one SURVEY.md section 8(d) states and DESIGN.md repeats:
numpy `default_rng(241002395 + cfg)`, C order, axis 0 slowest, objects drawn in sequence with
later ones overwriting earlier ones.
"""
from __future__ import annotations

import dataclasses
from typing import Callable, Tuple

import numpy as np

SEED_BASE = 241002395


@dataclasses.dataclass(frozen=True)
class Workload:
    """Geometry and stopping parameters of one configuration (no arrays)."""

    name: str
    shape: Tuple[int, ...]
    n_subdomains: Tuple[int, ...]
    boundary_width: Tuple[int, ...]
    tol: float
    max_iter: int
    pixel_size: float = 0.25      # lambda / 4 (4 points per wavelength)
    wavelength: float = 1.0
    n_correction: int = 8         # t = 8
    periodic: Tuple[int, ...] = ()
    seed: int = 0
    medium: Callable[["Workload"], np.ndarray] = None   # -> complex64 n(r)
    source: Callable[["Workload"], np.ndarray] = None   # -> complex64 y(r)

    @property
    def ndim(self) -> int:
        return len(self.shape)

    @property
    def voxels(self) -> int:
        return int(np.prod(self.shape))

    def periodic_flags(self) -> Tuple[int, ...]:
        return self.periodic if self.periodic else (0,) * self.ndim

    def make_medium(self) -> np.ndarray:
        return self.medium(self)

    def make_source(self) -> np.ndarray:
        return self.source(self)


# --------------------------------------------------------------------------------------
# object painters (pure geometry)
# --------------------------------------------------------------------------------------
def _paint_balls(n: np.ndarray, centres: np.ndarray, radii: np.ndarray, values: np.ndarray) -> None:
    """Paint D-dimensional balls (distance <= radius) into n, in sequence; later overwrites earlier."""
    shape = n.shape
    D = n.ndim
    for ctr, rad, val in zip(centres, radii, values):
        lo = [max(int(np.floor(ctr[d] - rad)), 0) for d in range(D)]
        hi = [min(int(np.ceil(ctr[d] + rad)) + 1, shape[d]) for d in range(D)]
        if any(h <= l for l, h in zip(lo, hi)):
            continue
        d2 = np.zeros((), dtype=np.float32)
        for d in range(D):
            ax = (np.arange(lo[d], hi[d], dtype=np.float32) - np.float32(ctr[d])) ** 2
            sh = [1] * D
            sh[d] = ax.size
            d2 = d2 + ax.reshape(sh)
        sl = tuple(slice(l, h) for l, h in zip(lo, hi))
        n[sl][d2 <= np.float32(rad) ** 2] = val


def _random_balls(w: Workload, background: complex, count: int, r_lo: float, r_hi: float,
                  n_lo: float, n_hi: float, n_imag: float) -> np.ndarray:
    rng = np.random.default_rng(w.seed)
    n = np.full(w.shape, background, dtype=np.complex64)
    centres = rng.uniform(0.0, 1.0, size=(count, w.ndim)) * np.asarray(w.shape, dtype=np.float64)
    radii = rng.uniform(r_lo, r_hi, size=count)
    n_real = rng.uniform(n_lo, n_hi, size=count)
    values = (n_real + 1j * n_imag).astype(np.complex64)
    _paint_balls(n, centres, radii, values)
    return n


def _smooth_periodic(a: np.ndarray, sigma: float) -> np.ndarray:
    """Separable Gaussian smoothing with periodic wrap (direct convolution, float32)."""
    half = int(np.ceil(4.0 * sigma))
    taps = np.exp(-0.5 * (np.arange(-half, half + 1) / sigma) ** 2)
    taps = (taps / taps.sum()).astype(np.float32)
    for ax in range(a.ndim):
        out = np.zeros_like(a)
        for k, wgt in zip(range(-half, half + 1), taps):
            out += wgt * np.roll(a, k, axis=ax)
        a = out
    return a


# --------------------------------------------------------------------------------------
# the five BASELINE.json configs
# --------------------------------------------------------------------------------------
def _medium_cfg1(w: Workload) -> np.ndarray:
    n = np.ones(w.shape, dtype=np.complex64)
    scale = w.shape[0] / 256.0
    n[int(round(100 * scale)):int(round(160 * scale)) + 1] = 1.5 + 0.01j
    return n


def _source_cfg1(w: Workload) -> np.ndarray:
    y = np.zeros(w.shape, dtype=np.complex64)
    y[w.shape[0] // 4] = 1.0
    return y


def _medium_cfg2(w: Workload) -> np.ndarray:
    count = max(1, int(round(200 * w.voxels / 1024 ** 2)))
    return _random_balls(w, 1.0, count, 2.0, 20.0, 1.0, 1.5, 0.005)


def _source_cfg2(w: Workload) -> np.ndarray:
    y = np.zeros(w.shape, dtype=np.complex64)
    N1 = w.shape[1]
    j = np.arange(N1, dtype=np.float64)
    row = 2 * w.boundary_width[0]
    y[row, :] = np.exp(-(((j - (N1 - 1) / 2.0) / (N1 / 8.0)) ** 2)).astype(np.complex64)
    return y


def _medium_cfg3(w: Workload) -> np.ndarray:
    count = max(1, int(round(500 * w.voxels / 256 ** 3)))
    return _random_balls(w, 1.33, count, 3.0, 15.0, 1.33, 1.6, 0.002)


def _source_centre(w: Workload) -> np.ndarray:
    y = np.zeros(w.shape, dtype=np.complex64)
    y[tuple(s // 2 for s in w.shape)] = 1.0
    return y


def _medium_cfg4(w: Workload) -> np.ndarray:
    rng = np.random.default_rng(w.seed)
    g = rng.standard_normal(size=w.shape, dtype=np.float32)
    g = _smooth_periodic(g, 4.0)
    g /= g.std()
    np.clip(g, -1.0, 1.0, out=g)
    return (np.float32(1.33) + np.float32(0.1) * g).astype(np.complex64)


def _source_cfg4(w: Workload) -> np.ndarray:
    y = np.zeros(w.shape, dtype=np.complex64)
    y[w.boundary_width[0] + 8] = 1.0          # plane at axis-0 index 32 for W = 24
    return y


def _medium_cfg5(w: Workload) -> np.ndarray:
    count = max(1, int(round(20000 * w.voxels / 1024 ** 3)))
    return _random_balls(w, 1.0, count, 4.0, 40.0, 1.0, 1.5, 0.001)


def _source_cfg5(w: Workload) -> np.ndarray:
    y = np.zeros(w.shape, dtype=np.complex64)
    idx = (w.boundary_width[0] + w.boundary_width[0] // 2,) + tuple(s // 2 for s in w.shape[1:])
    y[idx] = 1.0                               # (48, 512, 512) at full size
    return y


def _medium_paper_large(w: Workload) -> np.ndarray:
    """Stand-in for the structure of the paper's large run (section 4.3): spheres of radius 6 wavelengths
    (24 px), n = 1.33 with a small imaginary part, in n = 1, with a clearance of 6 wavelengths between them.  PoreSpy
    is not available: the centres sit on a cubic lattice of pitch 2r + clearance = 72 px, each jittered by up to
    +-10 px per axis and kept with probability 0.8 (seeded), which keeps a clearance of at least 4 px."""
    rng = np.random.default_rng(w.seed)
    pitch, rad = 72.0, 24.0
    axes = [np.arange(pitch / 2, s, pitch) for s in w.shape]
    grid = np.stack(np.meshgrid(*axes, indexing="ij"), axis=-1).reshape(-1, w.ndim)
    grid = grid + rng.uniform(-10.0, 10.0, size=grid.shape)
    keep = rng.uniform(size=len(grid)) < 0.8
    centres = grid[keep]
    n = np.ones(w.shape, dtype=np.complex64)
    _paint_balls(n, centres, np.full(len(centres), rad), np.full(len(centres), 1.33 + 0.001j, dtype=np.complex64))
    return n


def _source_plane_near_face(w: Workload) -> np.ndarray:
    """Planar source just inside the absorbing layer of the axis-0 face ("planar source located at x = 0", section 4)."""
    y = np.zeros(w.shape, dtype=np.complex64)
    y[w.boundary_width[0] + 4] = 1.0
    return y


def config(cfg: int, shape: Tuple[int, ...] = None, boundary_width: Tuple[int, ...] = None,
           tol: float = None, max_iter: int = None) -> Workload:
    """BASELINE.json config `cfg` (1..5).  `shape` overrides the grid for the reduced-size
    parity stand-ins (same generator, same subdomain counts, object count scaled by volume).
    cfg 6 is not a BASELINE.json config: it is the SHAPE of the paper's own large run (1260^3 voxels = 315^3
    wavelengths, two subdomains along x, 5-wavelength absorbing layers; section 4.3, Table 1), with a
    synthetic stand-in for its structure; bench.py quotes it as context beside the paper's numbers."""
    table = {
        1: dict(shape=(256,), S=(2,), W=(8,), tol=1e-6, max_iter=20000,
                medium=_medium_cfg1, source=_source_cfg1),
        2: dict(shape=(1024, 1024), S=(2, 2), W=(16, 16), tol=1e-4, max_iter=60000,
                medium=_medium_cfg2, source=_source_cfg2),
        3: dict(shape=(256, 256, 256), S=(2, 1, 1), W=(16, 16, 16), tol=1e-3, max_iter=60000,
                medium=_medium_cfg3, source=_source_centre),
        4: dict(shape=(640, 640, 640), S=(2, 2, 2), W=(24, 24, 24), tol=1e-3, max_iter=100000,
                medium=_medium_cfg4, source=_source_cfg4),
        5: dict(shape=(1024, 1024, 1024), S=(4, 2, 2), W=(32, 32, 32), tol=1e-3, max_iter=200000,
                medium=_medium_cfg5, source=_source_cfg5),
        6: dict(shape=(1260, 1260, 1260), S=(2, 1, 1), W=(20, 20, 20), tol=1e-3, max_iter=200000,
                medium=_medium_paper_large, source=_source_plane_near_face),
    }
    e = table[cfg]
    shp = tuple(shape) if shape is not None else e["shape"]
    W = tuple(boundary_width) if boundary_width is not None else e["W"]
    name = "cfg%d_%s" % (cfg, "x".join(str(s) for s in shp))
    return Workload(name=name, shape=shp, n_subdomains=e["S"], boundary_width=W,
                    tol=e["tol"] if tol is None else tol,
                    max_iter=e["max_iter"] if max_iter is None else max_iter,
                    seed=SEED_BASE + cfg, medium=e["medium"], source=e["source"])


def random_field(shape, seed: int) -> np.ndarray:
    """Seeded complex64 white-noise vector for per-operator parity."""
    rng = np.random.default_rng(seed)
    re = rng.standard_normal(size=shape, dtype=np.float32)
    im = rng.standard_normal(size=shape, dtype=np.float32)
    return (re + 1j * im).astype(np.complex64)


def random_medium(shape, seed: int, n_lo: float = 1.0, n_hi: float = 1.5, n_imag: float = 0.01) -> np.ndarray:
    """Seeded voxel-wise random refractive index (edge-case tests): Re n uniform, Im n uniform >= 0."""
    rng = np.random.default_rng(seed)
    re = rng.uniform(n_lo, n_hi, size=shape).astype(np.float32)
    im = rng.uniform(0.0, n_imag, size=shape).astype(np.float32)
    return (re + 1j * im).astype(np.complex64)
