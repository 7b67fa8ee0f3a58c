"""Seeded synthetic trajectory frames for the five BASELINE.json configs.

These frames stand in for the paper's SPC/E-water and n-alkane trajectories
(section 2.1), which are not available.  The recipe for every config
is the one in SURVEY.md section 8(d) / BASELINE.json `configs` and is restated in
DESIGN.md ("Input recipe").

This module is the ONLY code shared by the CPU oracle's tests and the CUDA
path's tests/bench.  It holds none of the method's arithmetic: no minimum
image, no distances, no thresholds, no binning.  It only draws particle
coordinates and snaps them to the box/2^20 grid, so that every fp64 position
handed to either side is exactly  m * (box / 1048576.0)  for an integer m in
[0, 2^20).

Generator: numpy `default_rng(seed)` (PCG64), seed = 1708086190 + config index.
Frames of configs 1-4 are a Gaussian random walk (frame f = frame f-1 + step,
re-wrapped into the box); the walk is carried in un-snapped fp64 and each
emitted frame is snapped on its own.  Frames of config 5 are independent.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Iterator, Optional, Tuple

import numpy as np

GRID_BITS = 20
GRID = 1 << GRID_BITS            # grid points per box edge
BASE_SEED = 1708086190


@dataclass(frozen=True)
class Workload:
    index: int          # 1..5, BASELINE.json configs[index-1]
    name: str
    n: int              # particles per frame
    box: float          # cubic box edge L
    r_max: float        # cut-off on r_ij and r_ik
    n_r: int            # bins on each of r_ij, r_ik over [0, r_max)
    n_t: int            # bins on r_jk over [0, 2 r_max)
    n_frames: int       # frames in the full workload
    kind: str           # "sc" | "diamond" | "chains" | "uniform"
    lattice_cells: int = 0      # cells per edge for "sc"/"diamond"
    jitter: float = 0.0         # sigma of the initial Gaussian jitter
    step: float = 0.0           # sigma of the per-frame Gaussian step
    chains: int = 0
    beads: int = 0
    bond: float = 0.0
    angle_deg: float = 0.0

    @property
    def seed(self) -> int:
        return BASE_SEED + self.index


WORKLOADS = {
    1: Workload(1, "tiny-lj", n=216, box=6.0, r_max=2.5, n_r=32, n_t=32, n_frames=10,
                kind="sc", lattice_cells=6, jitter=0.1, step=0.05),
    2: Workload(2, "water-4096", n=4096, box=4.96826, r_max=0.6, n_r=64, n_t=64, n_frames=100,
                kind="diamond", lattice_cells=8, jitter=0.03, step=0.01),
    3: Workload(3, "alkane-8192", n=8192, box=6.30451, r_max=1.0, n_r=64, n_t=64, n_frames=200,
                kind="chains", step=0.005, chains=512, beads=16, bond=0.154, angle_deg=114.0),
    4: Workload(4, "water-32768", n=32768, box=9.93652, r_max=0.7, n_r=64, n_t=64, n_frames=500,
                kind="diamond", lattice_cells=16, jitter=0.03, step=0.01),
    5: Workload(5, "ideal-262144", n=262144, box=19.87305, r_max=0.8, n_r=128, n_t=128,
                n_frames=100, kind="uniform"),
}


def grid_to_pos(m: np.ndarray, box: float) -> np.ndarray:
    """fp64 positions of integer grid coordinates: exactly m * (box / 2^20)."""
    return m.astype(np.float64) * (box / float(GRID))


def _snap(x: np.ndarray, box: float) -> np.ndarray:
    """Snap fp64 coordinates to the box/2^20 grid, wrapped into [0, 2^20)."""
    m = np.rint(x * (float(GRID) / box)).astype(np.int64)
    return np.mod(m, GRID).astype(np.int32)


def _diamond_sites(cells: int, box: float) -> np.ndarray:
    a = box / cells
    fcc = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]], dtype=np.float64)
    basis = np.concatenate([fcc, fcc + 0.25], axis=0)                  # 8 sites per cubic cell
    idx = np.arange(cells)
    cell = np.stack(np.meshgrid(idx, idx, idx, indexing="ij"), axis=-1).reshape(-1, 1, 3)
    return ((cell + basis[None, :, :]) * a).reshape(-1, 3)


def _sc_sites(cells: int, box: float) -> np.ndarray:
    a = box / cells
    idx = np.arange(cells)
    cell = np.stack(np.meshgrid(idx, idx, idx, indexing="ij"), axis=-1).reshape(-1, 3)
    return (cell + 0.5) * a


def _chain_sites(w: Workload, rng: np.random.Generator) -> np.ndarray:
    """Freely-rotating walks: fixed bond length and bond angle, uniform torsion,
    uniform random start, no excluded volume, wrapped into the box afterwards."""
    c, b = w.chains, w.beads
    gamma = np.deg2rad(180.0 - w.angle_deg)       # angle between successive bond vectors
    pos = np.empty((c, b, 3), dtype=np.float64)
    pos[:, 0, :] = rng.random((c, 3)) * w.box
    u = rng.normal(size=(c, 3))
    u /= np.linalg.norm(u, axis=1, keepdims=True)
    pos[:, 1, :] = pos[:, 0, :] + w.bond * u
    for s in range(2, b):
        helper = np.where(np.abs(u[:, :1]) < 0.9, np.array([[1.0, 0.0, 0.0]]), np.array([[0.0, 1.0, 0.0]]))
        e1 = np.cross(u, helper)
        e1 /= np.linalg.norm(e1, axis=1, keepdims=True)
        e2 = np.cross(u, e1)
        phi = rng.random((c, 1)) * (2.0 * np.pi)
        u = np.cos(gamma) * u + np.sin(gamma) * (np.cos(phi) * e1 + np.sin(phi) * e2)
        u /= np.linalg.norm(u, axis=1, keepdims=True)
        pos[:, s, :] = pos[:, s - 1, :] + w.bond * u
    return pos.reshape(-1, 3)


def frame_iter(w: Workload, n_frames: Optional[int] = None,
               seed: Optional[int] = None) -> Iterator[np.ndarray]:
    """Yield int32 [n, 3] grid coordinates, frame after frame, from the config's seed
    (or from `seed`: a different trajectory of the same recipe, e.g. one per rank).

    The first `k` frames are the same whatever `n_frames` is asked for."""
    total = w.n_frames if n_frames is None else int(n_frames)
    rng = np.random.default_rng(w.seed if seed is None else seed)
    if w.kind == "uniform":
        for _ in range(total):
            yield rng.integers(0, GRID, size=(w.n, 3), dtype=np.int64).astype(np.int32)
        return
    if w.kind == "sc":
        x = _sc_sites(w.lattice_cells, w.box)
        x = x + rng.normal(scale=w.jitter, size=x.shape)
    elif w.kind == "diamond":
        x = _diamond_sites(w.lattice_cells, w.box)
        x = x + rng.normal(scale=w.jitter, size=x.shape)
    elif w.kind == "chains":
        x = _chain_sites(w, rng)
    else:
        raise ValueError(w.kind)
    assert x.shape == (w.n, 3), (x.shape, w.n)
    for f in range(total):
        if f > 0:
            x = x + rng.normal(scale=w.step, size=x.shape)
        x = np.mod(x, w.box)
        yield _snap(x, w.box)


def frames(w: Workload, n_frames: Optional[int] = None) -> Tuple[np.ndarray, np.ndarray]:
    """(m int32 [F, n, 3], pos float64 [F, n, 3]) for the first F frames of workload `w`."""
    ms = list(frame_iter(w, n_frames))
    m = np.stack(ms, axis=0) if ms else np.zeros((0, w.n, 3), dtype=np.int32)
    return m, grid_to_pos(m, w.box)


def uniform_frame(n: int, seed: int) -> np.ndarray:
    """int32 [n, 3] uniform random grid coordinates (ideal gas) for ad-hoc test sizes."""
    rng = np.random.default_rng(seed)
    return rng.integers(0, GRID, size=(n, 3), dtype=np.int64).astype(np.int32)


def unwrapped_walk(n: int, n_frames: int, seed: int, step_sigma: float = 1000.0) -> np.ndarray:
    """int64 [F, n, 3] UNWRAPPED grid coordinates of a Gaussian random walk (for the MSD path,
    PAPER.md:642 "Starting from unwrapped"): uniform start in the box, then integer steps
    rint(N(0, step_sigma)) per coordinate and frame, never wrapped.  No method arithmetic."""
    rng = np.random.default_rng(seed)
    start = rng.integers(0, GRID, size=(1, n, 3), dtype=np.int64)
    steps = np.rint(rng.normal(scale=step_sigma, size=(n_frames - 1, n, 3))).astype(np.int64)
    return np.concatenate([start, start + np.cumsum(steps, axis=0)], axis=0)
