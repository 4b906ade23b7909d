"""Barrel detector of BASELINE.json configs[0], optionally closed by endcap discs (row f3).

10 cylindrical layers tiled by flat rectangular modules tangent to the
cylinder.  With `disc_z`, disc layers at z = +-disc_z[k] follow the barrel layers (all +z discs by increasing z, then all
-z discs by increasing |z|): rings in r x n_phi flat rectangular modules lying in the disc plane, loc0 along phi, loc1
along r, normal pointing away from the centre.  Pure array construction — no tracking arithmetic.
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
    # endcap discs (None / absent = barrel only).  For a disc layer l: layer_r[l] = outer radius, layer_r_min[l] = inner
    # radius, layer_half_z[l] = signed z of the disc plane, n_z[l] = number of rings, id = offset + i_phi * n_rings + i_ring
    layer_kind: np.ndarray = None    # [L] i32: 0 barrel cylinder, 1 disc
    layer_r_min: np.ndarray = None   # [L] f64 (0 for barrel layers)

    @property
    def n_barrel(self) -> int:
        return self.n_layers if self.layer_kind is None else int(np.sum(self.layer_kind == 0))

    def module_len_z(self, layer: int) -> float:
        return 2.0 * float(self.half_v[self.module_offset[layer]])


def build_detector(layer_r=LAYER_R, half_z: float = HALF_Z, x_over_x0: float = X_OVER_X0, disc_z=None,
                   disc_r=(30.0, 1010.0), disc_rings: int = 11, disc_n_phi: int = 160) -> Detector:
    # (the discs' outer radius deliberately differs from every barrel radius: a tip standing exactly on a cylinder would
    # otherwise compare its radius with the same number, a decision at rounding level)
    det = _build_barrel(layer_r, half_z, x_over_x0)
    if disc_z:
        det = _add_discs(det, [float(z) for z in disc_z], float(disc_r[0]), float(disc_r[1]), int(disc_rings),
                         int(disc_n_phi), x_over_x0)
    return det


def _add_discs(b: Detector, disc_z, r_min, r_max, n_rings, n_phi_d, x_over_x0) -> Detector:
    """Discs at +disc_z (ascending) then -disc_z: pixel resolution on the two innermost discs of a side, strips beyond."""
    zs = sorted(abs(z) for z in disc_z)
    planes = [z for z in zs] + [-z for z in zs]
    nd = len(planes)
    L = b.n_layers + nd
    per = n_phi_d * n_rings
    off = np.concatenate([b.module_offset, b.module_offset[-1] + per * np.arange(1, nd + 1)]).astype(np.int32)
    M = int(off[-1])
    pitch = (r_max - r_min) / n_rings
    center, au, av = np.zeros((M, 3)), np.zeros((M, 3)), np.zeros((M, 3))
    hu, hv, lay = np.zeros(M), np.zeros(M), np.zeros(M, np.int32)
    nb = b.n_modules
    center[:nb], au[:nb], av[:nb], hu[:nb], hv[:nb], lay[:nb] = b.center, b.axis_u, b.axis_v, b.half_u, b.half_v, b.module_layer
    for k, zd in enumerate(planes):
        l = b.n_layers + k
        i = np.repeat(np.arange(n_phi_d), n_rings)
        j = np.tile(np.arange(n_rings), n_phi_d)
        phi = 2.0 * np.pi * i / n_phi_d
        rc = r_min + (j + 0.5) * pitch
        sl = slice(off[l], off[l + 1])
        center[sl, 0], center[sl, 1], center[sl, 2] = rc * np.cos(phi), rc * np.sin(phi), zd
        sgn = 1.0 if zd > 0 else -1.0
        au[sl, 0], au[sl, 1] = sgn * np.sin(phi), -sgn * np.cos(phi)       # u x v = sign(z) e_z
        av[sl, 0], av[sl, 1] = np.cos(phi), np.sin(phi)
        hu[sl] = 1.05 * np.pi * (rc + 0.5 * pitch) / n_phi_d               # covers the ring's outer edge, 5 % overlap
        hv[sl] = 0.5 * pitch
        lay[sl] = l
    sig_d = np.array([SIGMA_PIXEL if (k % len(zs)) < 2 else SIGMA_STRIP for k in range(nd)], dtype=np.float64)
    return Detector(
        n_layers=L, layer_r=np.concatenate([b.layer_r, np.full(nd, r_max)]),
        layer_half_z=np.concatenate([b.layer_half_z, np.array(planes)]),
        n_phi=np.concatenate([b.n_phi, np.full(nd, n_phi_d, np.int32)]).astype(np.int32),
        n_z=np.concatenate([b.n_z, np.full(nd, n_rings, np.int32)]).astype(np.int32),
        module_offset=off, n_modules=M, center=center, axis_u=au, axis_v=av, half_u=hu, half_v=hv,
        x_over_x0=np.full(M, x_over_x0), module_layer=lay, sigma=np.concatenate([b.sigma, sig_d], axis=0),
        layer_kind=np.concatenate([np.zeros(b.n_layers, np.int32), np.ones(nd, np.int32)]).astype(np.int32),
        layer_r_min=np.concatenate([np.zeros(b.n_layers), np.full(nd, r_min)]),
    )


def _build_barrel(layer_r, half_z, x_over_x0) -> Detector:
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
