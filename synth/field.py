"""Magnetic-field inputs: uniform Bz, or the float32 grid of configs[2].

The analytic map: Bx = a B0 x z, By = a B0 y z,
Bz = B0 (1 - a z^2), B0 = 2 T, a = 0.3e-6 mm^-2 (divergence-free).
The grid samples it at 20 mm spacing over [-1100, 1100]^3 mm, rounded to
float32, layout [ix][iy][iz][3].  Trilinear interpolation is NOT here: it is
part of the method and lives (twice, independently) in oracle/ and csrc/.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import numpy as np

B0 = 2.0
A_INHOM = 0.3e-6


@dataclass
class FieldSpec:
    kind: int                       # 0 uniform, 1 grid
    uniform_b: np.ndarray           # [3] f64 tesla
    n: np.ndarray                   # [3] i32
    origin: np.ndarray              # [3] f64 mm
    spacing: np.ndarray             # [3] f64 mm
    grid: Optional[np.ndarray]      # [n0,n1,n2,3] f32 or None


def analytic_b(pos: np.ndarray, inhomogeneous: bool) -> np.ndarray:
    """Truth field at positions [n,3] (used by the event simulator only)."""
    pos = np.asarray(pos, np.float64)
    b = np.zeros_like(pos)
    if inhomogeneous:
        x, y, z = pos[..., 0], pos[..., 1], pos[..., 2]
        b[..., 0] = A_INHOM * B0 * x * z
        b[..., 1] = A_INHOM * B0 * y * z
        b[..., 2] = B0 * (1.0 - A_INHOM * z * z)
    else:
        b[..., 2] = B0
    return b


def uniform_field(bz: float = B0) -> FieldSpec:
    return FieldSpec(0, np.array([0.0, 0.0, bz]), np.zeros(3, np.int32), np.zeros(3), np.ones(3), None)


def grid_field(half_extent: float = 1100.0, spacing: float = 20.0) -> FieldSpec:
    n = int(round(2 * half_extent / spacing)) + 1          # 111
    ax = -half_extent + spacing * np.arange(n)
    X, Y, Z = np.meshgrid(ax, ax, ax, indexing="ij")
    pos = np.stack([X, Y, Z], axis=-1)
    grid = analytic_b(pos, True).astype(np.float32)
    return FieldSpec(1, np.array([0.0, 0.0, B0]), np.array([n, n, n], np.int32),
                     np.full(3, -half_extent), np.full(3, spacing), np.ascontiguousarray(grid))
