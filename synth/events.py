"""Seeded synthetic events for BASELINE.json configs[0..4].

What stands in for the paper's Geant4 ttbar samples in the Open Data Detector
(§3): a particle gun of muons through the 10-layer barrel of
`detector.py`, truth transport by a fixed-step classical RK4 of the Lorentz
equation in the *analytic* field, Highland multiple-scattering kicks after
every crossed module, Gaussian-smeared 2-D measurements, uniform noise hits,
truth-smeared seeds and (configs 3-4) fake seeds.  All random numbers come from
one counter-based generator, numpy's Philox, keyed by 1000*config + event.

This is a simulator of the *data*.  It contains no CKF arithmetic and is shared
by the oracle-side and the CUDA-side tests as the only common module.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field as dc_field
from typing import Dict, Optional

import numpy as np

from .detector import Detector, build_detector
from .field import FieldSpec, analytic_b, grid_field, uniform_field

KAPPA = 2.99792458e-4      # GeV / (T mm):  curvature = KAPPA * (q/p) * B
M_MUON = 0.1056583755      # GeV  ("assuming muon trajectories")
H_SIM = 25.0               # mm, fixed RK4 sub-step of the truth simulator
S_CLOSE = 1e-7             # mm, landing tolerance of the truth simulator


@dataclass
class CKFSettings:
    """Per-config CKF constants (BASELINE.json configs + SURVEY.md §8(c) readings)."""
    chi2_max: float = 10.0
    max_branches_per_surface: int = 1
    max_candidates_per_seed: int = 1
    max_holes: int = 3
    min_measurements: int = 3
    rk_tolerance_mm: float = 1e-4
    surface_tolerance_mm: float = 1e-5
    h_max_mm: float = 200.0
    particle_mass_gev: float = M_MUON
    max_rk_steps_per_surface: int = 64
    max_levels: int = 32
    energy_loss: int = 0          # rule E (mean energy loss per module); BASELINE configs: off
    field_gradient: int = 0       # transport Jacobian with field-gradient terms (rule J2'); BASELINE configs: off
    bidirectional: int = 0        # navigate radially inward-moving tips too (row f3); BASELINE configs: off (reading A7)


@dataclass
class SeedSettings:
    """Triplet seeding + parameter estimation constants (DESIGN.md rules S0-S6; readings: the paper gives no cut)."""
    layer_b: int = 0
    layer_m: int = 1
    layer_t: int = 2
    dphi_max: float = 0.05          # rad, doublet (pT >= 0.4 GeV bends 0.033 rad between the seeding layers)
    cot_max: float = 10.5           # |eta| <= 3
    z0_max: float = 200.0           # mm: 4 sigma of the vertex spread
    dcot_max: float = 0.01          # ~5 sigma of resolution + scattering between the two doublets
    pt_min: float = 0.4             # GeV, below the 0.5 GeV of the workloads
    d0_max: float = 2.0             # mm
    sigma_angle: float = 2e-3       # rad
    rel_sigma_qop: float = 0.1
    cov_scale: float = 10.0         # BASELINE seeds: covariance = 10 x the smearing variances


@dataclass
class EventConfig:
    config: int
    n_particles: int
    pt_min: float
    pt_max: float
    noise_fraction: float
    n_fake_seeds: int
    inhomogeneous: bool
    precision: int              # 32 or 64 : element type of measurement/seed arrays
    ckf: CKFSettings = dc_field(default_factory=CKFSettings)


CONFIGS: Dict[int, EventConfig] = {
    0: EventConfig(0, 100, 1.0, 10.0, 0.0, 0, False, 64,
                   CKFSettings(max_branches_per_surface=1, max_candidates_per_seed=1)),
    1: EventConfig(1, 2000, 0.5, 50.0, 0.2, 0, False, 64,
                   CKFSettings(max_branches_per_surface=5, max_candidates_per_seed=50)),
    2: EventConfig(2, 10000, 0.5, 50.0, 0.2, 0, True, 32,
                   CKFSettings(max_branches_per_surface=5, max_candidates_per_seed=50,
                               surface_tolerance_mm=1e-2)),
    3: EventConfig(3, 40000, 0.5, 50.0, 0.2, 4000, True, 32,
                   CKFSettings(max_branches_per_surface=10, max_candidates_per_seed=100,
                               surface_tolerance_mm=1e-2)),
    # config 4 = 64 events of config 3's recipe with event index 0..63 (streamed)
    4: EventConfig(4, 40000, 0.5, 50.0, 0.2, 4000, True, 32,
                   CKFSettings(max_branches_per_surface=10, max_candidates_per_seed=100,
                               surface_tolerance_mm=1e-2)),
}


@dataclass
class Event:
    """One event in the layout of `ckf_measurements` / `ckf_seeds` (include/ckf.h)."""
    config: int
    event_index: int
    precision: int
    # measurements, CSR by module id
    module_offsets: np.ndarray      # [M+1] i32
    loc: np.ndarray                 # [n,2] T
    var: np.ndarray                 # [n,2] T
    meas_particle: np.ndarray       # [n] i32 truth particle id, -1 = noise   (never given to the CKF)
    meas_module: np.ndarray         # [n] i32 (convenience)
    # seeds
    seed_module: np.ndarray         # [S] i32
    seed_params: np.ndarray         # [S,6] T   loc0 loc1 phi theta q/p t
    seed_cov: np.ndarray            # [S,36] T  row-major symmetric
    seed_particle: np.ndarray       # [S] i32 truth particle id, -1 = fake
    # truth
    particle_q: np.ndarray
    particle_pt: np.ndarray
    particle_eta: np.ndarray
    particle_phi: np.ndarray
    particle_z0: np.ndarray
    n_signal: int = 0
    n_noise: int = 0

    @property
    def n_measurements(self) -> int:
        return int(self.loc.shape[0])

    @property
    def n_seeds(self) -> int:
        return int(self.seed_module.shape[0])


# --------------------------------------------------------------------------- simulator helpers
def _cross(a: np.ndarray, b: np.ndarray) -> np.ndarray:
    out = np.empty_like(a)
    out[:, 0] = a[:, 1] * b[:, 2] - a[:, 2] * b[:, 1]
    out[:, 1] = a[:, 2] * b[:, 0] - a[:, 0] * b[:, 2]
    out[:, 2] = a[:, 0] * b[:, 1] - a[:, 1] * b[:, 0]
    return out


def _rk4(r, d, lam, h, inhom):
    """One classical RK4 step of r' = d, d' = lam d x B(r); h per particle (0 = stay)."""
    hh = h[:, None]
    lm = lam[:, None]

    def acc(rr, dd):
        return lm * _cross(dd, analytic_b(rr, inhom))

    k1d = acc(r, d)
    d2 = d + 0.5 * hh * k1d
    k2d = acc(r + 0.5 * hh * d, d2)
    d3 = d + 0.5 * hh * k2d
    k3d = acc(r + 0.5 * hh * d2, d3)
    d4 = d + hh * k3d
    k4d = acc(r + hh * d3, d4)
    rn = r + hh / 6.0 * (d + 2.0 * d2 + 2.0 * d3 + d4)
    dn = d + hh / 6.0 * (k1d + 2.0 * k2d + 2.0 * k3d + k4d)
    dn /= np.linalg.norm(dn, axis=1)[:, None]
    return rn, dn


def _to_cylinder(r, d, lam, R, inhom):
    """Transport every particle to the cylinder of radius R.  Returns (r, d, ok)."""
    n = r.shape[0]
    ok = np.ones(n, bool)
    for _ in range(400):
        a = d[:, 0] ** 2 + d[:, 1] ** 2
        b = r[:, 0] * d[:, 0] + r[:, 1] * d[:, 1]
        cc = r[:, 0] ** 2 + r[:, 1] ** 2 - R * R
        disc = b * b - a * cc
        den = b + np.sqrt(np.where(disc > 0.0, disc, 0.0))
        ok &= (disc >= 0.0) & (den > 0.0)
        s = np.where(ok, -cc / np.where(ok, den, 1.0), 0.0)
        todo = ok & (np.abs(s) > S_CLOSE)
        if not todo.any():
            r = r + s[:, None] * d
            break
        h = np.where(todo, np.clip(s, -H_SIM, H_SIM), 0.0)
        r, d = _rk4(r, d, lam, h, inhom)
    return r, d, ok


def _to_plane(r, d, lam, c, nrm, inhom):
    for _ in range(400):
        dn = np.einsum("ij,ij->i", d, nrm)
        s = np.einsum("ij,ij->i", c - r, nrm) / dn
        todo = np.abs(s) > S_CLOSE
        if not todo.any():
            r = r + s[:, None] * d
            break
        h = np.where(todo, np.clip(s, -H_SIM, H_SIM), 0.0)
        r, d = _rk4(r, d, lam, h, inhom)
    return r, d


def _pick_module(det: Detector, normal, layer, i0, j0, r, d, s_min, exclude):
    """Nearest in-bounds module among the 3x3 (phi wraps, z clamps) around (i0, j0).

    Straight-line test from the current point.  Returns module id or -1.
    """
    n = r.shape[0]
    nphi = int(det.n_phi[layer])
    nz = int(det.n_z[layer])
    off = int(det.module_offset[layer])
    best_s = np.full(n, np.inf)
    best_id = np.full(n, -1, np.int64)
    for di in (-1, 0, 1):
        ii = (i0 + di) % nphi
        for dj in (-1, 0, 1):
            jj = j0 + dj
            valid = (jj >= 0) & (jj < nz)
            mid = off + ii * nz + np.clip(jj, 0, nz - 1)
            c = det.center[mid]
            nk = normal[mid]
            dn = np.einsum("ij,ij->i", d, nk)
            good = valid & (dn > 1e-6) & (mid != exclude)
            s = np.einsum("ij,ij->i", c - r, nk) / np.where(good, dn, 1.0)
            q = r + s[:, None] * d - c
            lu = np.einsum("ij,ij->i", q, det.axis_u[mid])
            lv = np.einsum("ij,ij->i", q, det.axis_v[mid])
            good &= (np.abs(lu) <= det.half_u[mid]) & (np.abs(lv) <= det.half_v[mid]) & (s > s_min)
            better = good & ((s < best_s) | ((s == best_s) & (mid < best_id)))
            best_s = np.where(better, s, best_s)
            best_id = np.where(better, mid, best_id)
    return best_id


def _highland(p, x_eff):
    beta = p / np.sqrt(p * p + M_MUON * M_MUON)
    return 0.0136 / (beta * p) * np.sqrt(x_eff) * (1.0 + 0.038 * np.log(x_eff / (beta * beta)))


def _draw_particles(rng, n, pt_min, pt_max):
    q = np.where(rng.random(n) < 0.5, -1.0, 1.0)
    pt = np.exp(rng.uniform(math.log(pt_min), math.log(pt_max), n))
    eta = rng.uniform(-1.0, 1.0, n)
    phi = rng.uniform(0.0, 2.0 * math.pi, n)
    return q, pt, eta, phi


# --------------------------------------------------------------------------- the event generator
def make_event(config: int, event_index: int = 0, det: Optional[Detector] = None,
               n_particles: Optional[int] = None, n_fake_seeds: Optional[int] = None) -> Event:
    """Generate one event of BASELINE.json configs[config]; seed = 1000*config + event_index.

    `n_particles` / `n_fake_seeds` override the config's sizes (for small test cases).
    Config 4's events are config 3's recipe keyed 4000 + event_index.
    """
    cfg = CONFIGS[config]
    det = det or build_detector()
    normal = np.cross(det.axis_u, det.axis_v)
    rng = np.random.Generator(np.random.Philox(key=1000 * config + event_index))
    npart = cfg.n_particles if n_particles is None else int(n_particles)
    nfake = cfg.n_fake_seeds if n_fake_seeds is None else int(n_fake_seeds)
    inhom = cfg.inhomogeneous

    q, pt, eta, phi0 = _draw_particles(rng, npart, cfg.pt_min, cfg.pt_max)
    z0 = rng.normal(0.0, 50.0, npart)
    theta = 2.0 * np.arctan(np.exp(-eta))
    p = pt * np.cosh(eta)
    qop = q / p
    lam = KAPPA * qop

    r = np.stack([np.zeros(npart), np.zeros(npart), z0], axis=1)
    d = np.stack([np.sin(theta) * np.cos(phi0), np.sin(theta) * np.sin(phi0), np.cos(theta)], axis=1)
    alive = np.ones(npart, bool)

    hit_pid, hit_mod, hit_l0, hit_l1 = [], [], [], []
    seed_found = np.zeros(npart, bool)
    seed_mod = np.full(npart, -1, np.int64)
    seed_par = np.zeros((npart, 6))

    for layer in range(det.n_layers):
        idx = np.nonzero(alive)[0]
        if idx.size == 0:
            break
        rr, dd, ok = _to_cylinder(r[idx], d[idx], lam[idx], float(det.layer_r[layer]), inhom)
        r[idx[ok]] = rr[ok]
        d[idx[ok]] = dd[ok]
        alive[idx[~ok]] = False
        idx = idx[ok]
        # acceptance in z (a track outside simply has no hit on this layer)
        inz = np.abs(r[idx, 2]) <= det.layer_half_z[layer]
        idx = idx[inz]
        nphi = int(det.n_phi[layer])
        nz = int(det.n_z[layer])
        ln = 2.0 * float(det.half_v[det.module_offset[layer]])
        ph = np.arctan2(r[idx, 1], r[idx, 0])
        i0 = np.rint(ph * nphi / (2.0 * np.pi)).astype(np.int64) % nphi
        j0 = np.clip(np.floor((r[idx, 2] + det.layer_half_z[layer]) / ln).astype(np.int64), 0, nz - 1)
        exclude = np.full(idx.size, -1, np.int64)
        s_min = -1e-3
        for _cross_no in range(3):
            if idx.size == 0:
                break
            mid = _pick_module(det, normal, layer, i0, j0, r[idx], d[idx], s_min, exclude)
            has = mid >= 0
            idx, mid = idx[has], mid[has]
            if idx.size == 0:
                break
            rr, dd = _to_plane(r[idx], d[idx], lam[idx], det.center[mid], normal[mid], inhom)
            r[idx] = rr
            d[idx] = dd
            rel = rr - det.center[mid]
            l0 = np.einsum("ij,ij->i", rel, det.axis_u[mid])
            l1 = np.einsum("ij,ij->i", rel, det.axis_v[mid])
            hit_pid.append(idx.copy())
            hit_mod.append(mid.copy())
            hit_l0.append(l0)
            hit_l1.append(l1)
            if layer == 0:
                first = ~seed_found[idx]
                fi = idx[first]
                seed_found[fi] = True
                seed_mod[fi] = mid[first]
                seed_par[fi, 0] = l0[first]
                seed_par[fi, 1] = l1[first]
                seed_par[fi, 2] = np.arctan2(dd[first, 1], dd[first, 0])
                seed_par[fi, 3] = np.arctan2(np.hypot(dd[first, 0], dd[first, 1]), dd[first, 2])
                seed_par[fi, 4] = qop[fi]
            # multiple scattering: two independent projected kicks (Highland theta0)
            cosi = np.abs(np.einsum("ij,ij->i", dd, normal[mid]))
            th0 = _highland(p[idx], det.x_over_x0[mid] / cosi)
            k1 = rng.standard_normal(idx.size) * th0
            k2 = rng.standard_normal(idx.size) * th0
            e1 = _cross(dd, np.broadcast_to(np.array([0.0, 0.0, 1.0]), dd.shape).copy())
            e1 /= np.linalg.norm(e1, axis=1)[:, None]
            e2 = _cross(dd, e1)
            dk = dd + k1[:, None] * e1 + k2[:, None] * e2
            dk /= np.linalg.norm(dk, axis=1)[:, None]
            d[idx] = dk
            # next crossing on the same layer (phi overlap): neighbours of the module just hit
            loc_id = mid - int(det.module_offset[layer])
            i0 = loc_id // nz
            j0 = loc_id % nz
            exclude = mid
            s_min = 1e-3

    # ---- measurements
    if hit_pid:
        pid = np.concatenate(hit_pid)
        mod = np.concatenate(hit_mod)
        tl0 = np.concatenate(hit_l0)
        tl1 = np.concatenate(hit_l1)
    else:
        pid = np.zeros(0, np.int64); mod = np.zeros(0, np.int64); tl0 = np.zeros(0); tl1 = np.zeros(0)
    nsig = pid.size
    lay = det.module_layer[mod]
    sig = det.sigma[lay]
    m0 = tl0 + rng.standard_normal(nsig) * sig[:, 0]
    m1 = tl1 + rng.standard_normal(nsig) * sig[:, 1]
    nnoise = int(round(cfg.noise_fraction * nsig))
    nmod = rng.integers(0, det.n_modules, nnoise)
    n0 = rng.uniform(-1.0, 1.0, nnoise) * det.half_u[nmod]
    n1 = rng.uniform(-1.0, 1.0, nnoise) * det.half_v[nmod]
    nsg = det.sigma[det.module_layer[nmod]]
    all_mod = np.concatenate([mod, nmod])
    all_loc = np.stack([np.concatenate([m0, n0]), np.concatenate([m1, n1])], axis=1)
    all_var = np.concatenate([sig, nsg], axis=0) ** 2
    all_pid = np.concatenate([pid, np.full(nnoise, -1, np.int64)])
    order = np.argsort(all_mod, kind="stable")
    all_mod, all_loc, all_var, all_pid = all_mod[order], all_loc[order], all_var[order], all_pid[order]
    offsets = np.zeros(det.n_modules + 1, np.int64)
    np.add.at(offsets, all_mod + 1, 1)
    offsets = np.cumsum(offsets)

    # ---- seeds: truth bound state on the first layer-0 module, smeared
    sp = np.nonzero(seed_found)[0]
    par = seed_par[sp].copy()
    sig_s = np.stack([np.full(sp.size, 0.05), np.full(sp.size, 0.1), np.full(sp.size, 1e-3),
                      np.full(sp.size, 1e-3), 0.05 * np.abs(par[:, 4]), np.zeros(sp.size)], axis=1)
    par += rng.standard_normal((sp.size, 6)) * sig_s
    smod = seed_mod[sp]
    spid = sp.astype(np.int64)
    if nfake > 0:
        fq, fpt, feta, fphi = _draw_particles(rng, nfake, cfg.pt_min, cfg.pt_max)
        fmod = rng.integers(0, int(det.module_offset[1]), nfake)
        fpar = np.zeros((nfake, 6))
        fpar[:, 0] = rng.uniform(-1.0, 1.0, nfake) * det.half_u[fmod]
        fpar[:, 1] = rng.uniform(-1.0, 1.0, nfake) * det.half_v[fmod]
        fpar[:, 2] = np.where(fphi > np.pi, fphi - 2.0 * np.pi, fphi)
        fpar[:, 3] = 2.0 * np.arctan(np.exp(-feta))
        fpar[:, 4] = fq / (fpt * np.cosh(feta))
        fsig = np.stack([np.full(nfake, 0.05), np.full(nfake, 0.1), np.full(nfake, 1e-3),
                         np.full(nfake, 1e-3), 0.05 * np.abs(fpar[:, 4]), np.zeros(nfake)], axis=1)
        par = np.concatenate([par, fpar], axis=0)
        sig_s = np.concatenate([sig_s, fsig], axis=0)
        smod = np.concatenate([smod, fmod])
        spid = np.concatenate([spid, np.full(nfake, -1, np.int64)])
    S = par.shape[0]
    cov = np.zeros((S, 6, 6))
    diag = 10.0 * sig_s ** 2
    diag[:, 5] = 1.0
    cov[:, np.arange(6), np.arange(6)] = diag

    T = np.float64 if cfg.precision == 64 else np.float32
    return Event(
        config=config, event_index=event_index, precision=cfg.precision,
        module_offsets=offsets.astype(np.int32),
        loc=np.ascontiguousarray(all_loc.astype(T)), var=np.ascontiguousarray(all_var.astype(T)),
        meas_particle=all_pid.astype(np.int32), meas_module=all_mod.astype(np.int32),
        seed_module=smod.astype(np.int32), seed_params=np.ascontiguousarray(par.astype(T)),
        seed_cov=np.ascontiguousarray(cov.reshape(S, 36).astype(T)), seed_particle=spid.astype(np.int32),
        particle_q=q, particle_pt=pt, particle_eta=eta, particle_phi=phi0, particle_z0=z0,
        n_signal=int(nsig), n_noise=int(nnoise),
    )


def config_bundle(config: int):
    """(detector, field spec, event config) of BASELINE.json configs[config]."""
    cfg = CONFIGS[config]
    det = build_detector()
    fld = grid_field() if cfg.inhomogeneous else uniform_field()
    return det, fld, cfg
