"""Barrel detector of BASELINE.json configs[0].

10 cylindrical layers tiled by flat rectangular modules tangent to the
cylinder.  Pure array construction — no tracking arithmetic.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

LAYER_R = (32.0, 72.0, 116.0, 172.0, 260.0, 360.0, 500.0, 660.0, 820.0, 1020.0)
HALF_Z = 1000.0
X_OVER_X0 = 0.0016          # 0.15 mm silicon, configs[0]
# measurement resolution (sigma loc0, sigma loc1) per layer, configs[0]
SIGMA_PIXEL = (0.015, 0.05)  # layers 0-3
SIGMA_STRIP = (0.04, 1.0)    # layers 4-9


@dataclass
class Detector:
    """Flat arrays in exactly the layout of `ckf_geometry` (include/ckf.h)."""
    n_layers: int
    layer_r: np.ndarray        # [L] f64 mm
    layer_half_z: np.ndarray   # [L] f64 mm
    n_phi: np.ndarray          # [L] i32
    n_z: np.ndarray            # [L] i32
    module_offset: np.ndarray  # [L+1] i32 ; module id = module_offset[l] + i_phi*n_z[l] + i_z
    n_modules: int
    center: np.ndarray         # [M,3] f64
    axis_u: np.ndarray         # [M,3] f64  (loc0 direction, along phi)
    axis_v: np.ndarray         # [M,3] f64  (loc1 direction, along z)
    half_u: np.ndarray         # [M] f64
    half_v: np.ndarray         # [M] f64
    x_over_x0: np.ndarray      # [M] f64
    module_layer: np.ndarray   # [M] i32 (convenience; derivable from module_offset)
    sigma: np.ndarray          # [L,2] f64 measurement resolution per layer (data recipe only)

    def module_len_z(self, layer: int) -> float:
        return 2.0 * float(self.half_v[self.module_offset[layer]])


def build_detector(layer_r=LAYER_R, half_z: float = HALF_Z, x_over_x0: float = X_OVER_X0) -> Detector:
    L = len(layer_r)
    n_phi = np.zeros(L, np.int32)
    n_z = np.zeros(L, np.int32)
    off = np.zeros(L + 1, np.int32)
    widths, lens = [], []
    for l, r in enumerate(layer_r):
        w, ln = (20.0, 40.0) if l < 4 else (40.0, 100.0)
        n_phi[l] = math.ceil(1.05 * 2.0 * math.pi * r / w)
        n_z[l] = math.ceil(2.0 * half_z / ln)
        off[l + 1] = off[l] + n_phi[l] * n_z[l]
        widths.append(w)
        lens.append(ln)
    M = int(off[L])
    center = np.zeros((M, 3))
    au = np.zeros((M, 3))
    av = np.zeros((M, 3))
    hu = np.zeros(M)
    hv = np.zeros(M)
    lay = np.zeros(M, np.int32)
    for l, r in enumerate(layer_r):
        i = np.repeat(np.arange(n_phi[l]), n_z[l])
        j = np.tile(np.arange(n_z[l]), n_phi[l])
        phi = 2.0 * np.pi * i / n_phi[l]
        z = -half_z + (j + 0.5) * lens[l]
        sl = slice(off[l], off[l + 1])
        center[sl, 0] = r * np.cos(phi)
        center[sl, 1] = r * np.sin(phi)
        center[sl, 2] = z
        au[sl, 0] = -np.sin(phi)
        au[sl, 1] = np.cos(phi)
        av[sl, 2] = 1.0
        hu[sl] = widths[l] / 2.0
        hv[sl] = lens[l] / 2.0
        lay[sl] = l
    sigma = np.array([SIGMA_PIXEL if l < 4 else SIGMA_STRIP for l in range(L)], dtype=np.float64)
    return Detector(
        n_layers=L, layer_r=np.asarray(layer_r, np.float64), layer_half_z=np.full(L, half_z),
        n_phi=n_phi, n_z=n_z, module_offset=off, n_modules=M, center=center, axis_u=au, axis_v=av,
        half_u=hu, half_v=hv, x_over_x0=np.full(M, x_over_x0), module_layer=lay, sigma=sigma,
    )
