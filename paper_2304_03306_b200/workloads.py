"""Seeded synthetic inputs shaped like the paper's workloads (disks of growing radius, dumbbells
of two overlapping circles, small random initial field).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic: only binary geometry masks, random numbers and the config table of
BASELINE.json.  It imports neither ``oracle`` nor the CUDA binding.  Recipe: DESIGN.md §4.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional, Tuple

import numpy as np

SEED0 = 230403306   # seed = SEED0 + config index


def disk_mask(Nx: int, Ny: int, dx: float, R: float) -> np.ndarray:
    """K_naive = 1 for ||x|| >= R (inclusive), 0 inside; centre at grid index (Nx/2, Ny/2)
    (reading R11).  Returned as uint8 [Ny, Nx], 1 = masked."""
    i = np.arange(Nx, dtype=np.float64)[None, :] - Nx // 2
    j = np.arange(Ny, dtype=np.float64)[:, None] - Ny // 2
    return ((i * i + j * j) * (dx * dx) >= R * R).astype(np.uint8)


def dumbbell_mask(Nx: int, Ny: int, dx: float, R: float, d: float) -> np.ndarray:
    """Two overlapping circles of radius R whose centres are d apart along x ("left/right",
    PAPER.md:183, :199); masked iff outside BOTH circles (logical AND of the two circle masks,
    PAPER.md:371)."""
    j = np.arange(Ny, dtype=np.float64)[:, None] - Ny // 2
    out = np.ones((Ny, Nx), dtype=bool)
    for s in (-0.5, +0.5):
        i = np.arange(Nx, dtype=np.float64)[None, :] - Nx // 2 - s * d / dx
        out &= (i * i + j * j) * (dx * dx) >= R * R
    return out.astype(np.uint8)


def gaussian_velocity(Nx: int, Ny: int, seed: int, amplitude: float = 1e-2,
                      mask: Optional[np.ndarray] = None) -> Tuple[np.ndarray, np.ndarray]:
    """i.i.d. Gaussian, `amplitude` per component, zeroed where mask == 1 (BASELINE.json configs).
    Counter-based generator (Philox) keyed by (seed, component).  fp64 [Ny, Nx] each.  The
    divergence-free projection named by the configs is done by ttsh_set_velocity on both sides."""
    out = []
    for comp in (0, 1):
        g = np.random.Generator(np.random.Philox(key=[seed, comp]))
        f = amplitude * g.standard_normal((Ny, Nx))
        if mask is not None:
            f = np.where(np.asarray(mask) != 0, 0.0, f)
        out.append(np.ascontiguousarray(f))
    return out[0], out[1]


def planewave_velocity(Nx: int, Ny: int, dx: float, seed: int, amplitude: float = 1.0,
                       nmodes: int = 24, kmax: float = 1.5) -> Tuple[np.ndarray, np.ndarray]:
    """O(1) smooth start (reading R17): a sum of `nmodes` random plane waves with grid-periodic
    wavevectors |k| <= kmax and random phases, scaled so that rms |v| ~ amplitude.  Used so that
    advection, cubic and damping terms are all O(1) in the 1- and 100-step parity checks."""
    g = np.random.Generator(np.random.Philox(key=[seed, 7]))
    x = np.arange(Nx, dtype=np.float64)[None, :]
    y = np.arange(Ny, dtype=np.float64)[:, None]
    mxmax = max(1, int(kmax * Nx * dx / (2 * np.pi)))
    mymax = max(1, int(kmax * Ny * dx / (2 * np.pi)))
    vx = np.zeros((Ny, Nx))
    vy = np.zeros((Ny, Nx))
    for _ in range(nmodes):
        mx = int(g.integers(-mxmax, mxmax + 1))
        my = int(g.integers(-mymax, mymax + 1))
        phase = float(g.uniform(0.0, 2 * np.pi))
        ax, ay = g.standard_normal(2)
        c = np.cos(2 * np.pi * ((mx * x) / Nx + (my * y) / Ny) + phase)
        vx += ax * c
        vy += ay * c
    s = amplitude / np.sqrt(np.mean(vx * vx + vy * vy))
    return np.ascontiguousarray(vx * s), np.ascontiguousarray(vy * s)


@dataclass(frozen=True)
class Config:
    """One row of BASELINE.json:configs (grid as array shape [Ny][Nx], reading R11)."""
    name: str
    Nx: int
    Ny: int
    dx: float = 0.5
    dt: float = 1e-2
    geometry: str = "disk"           # "disk" | "dumbbell" | "none"
    R: float = 0.0
    d: float = 0.0
    steps: int = 100
    dtypes: Tuple[str, ...] = ("f64",)
    index: int = 0
    sweep: Tuple[float, ...] = field(default_factory=tuple)
    preset: str = "baseline"         # "baseline" (BASELINE.json's parameters) | "paper" (Table I)

    @property
    def seed(self) -> int:
        return SEED0 + self.index

    def mask(self, R: Optional[float] = None, d: Optional[float] = None) -> Optional[np.ndarray]:
        R = self.R if R is None else R
        d = self.d if d is None else d
        if self.geometry == "disk":
            return disk_mask(self.Nx, self.Ny, self.dx, R)
        if self.geometry == "dumbbell":
            return dumbbell_mask(self.Nx, self.Ny, self.dx, R, d)
        return None

    def initial_velocity(self, mask: Optional[np.ndarray] = None, amplitude: float = 1e-2):
        return gaussian_velocity(self.Nx, self.Ny, self.seed, amplitude, mask)


CONFIGS = {
    "C1": Config("C1", 64, 64, geometry="disk", R=12.0, steps=100, index=0),
    "C2": Config("C2", 256, 256, geometry="disk", R=30.0, steps=20000, index=1),
    "C3": Config("C3", 1024, 1024, geometry="disk", R=160.0, steps=10000, dtypes=("f64", "f32"),
                 index=2, sweep=(40.0, 80.0, 160.0, 240.0)),
    "C4": Config("C4", 2048, 1024, geometry="dumbbell", R=60.0, d=100.0, steps=10000, index=3,
                 sweep=(80.0, 100.0, 110.0, 118.0)),
    "C5": Config("C5", 4096, 4096, geometry="disk", R=900.0, steps=2000, dtypes=("f64", "f32"), index=4),
    "C5p": Config("C5p", 4096, 4096, geometry="none", steps=2000, dtypes=("f64", "f32"), index=4),
    # the paper's own production run (Table I :264-278): 8192 x 8192, dx = 0.005 (L = 40.96), dt = 0.01, the paper's
    # parameters, a disk of radius R = 5.2 (just above the onset of the single vortex): about 95 % of the box is masked
    "C6": Config("C6", 8192, 8192, dx=0.005, dt=0.01, geometry="disk", R=5.2, steps=2000, dtypes=("f64", "f32"), index=5, preset="paper"),
    # the grid of Fig. 6(f) (Table I footnote a): (N, dx) = (16384, 0.0025), the same box L = 40.96 and disk as C6 at
    # twice the resolution; 27 GB of workspace in fp64, 13.5 GB in fp32
    "C7": Config("C7", 16384, 16384, dx=0.0025, dt=0.01, geometry="disk", R=5.2, steps=2000, dtypes=("f64", "f32"), index=6, preset="paper"),
}
