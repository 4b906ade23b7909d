"""Seeded synthetic events for a barrel + endcap-disc detector (row f3: |eta| up to 3; "barrel + endcaps").

Same recipe as `events.make_event` (muon gun, fixed-step RK4 truth transport in the analytic field, Highland kicks after
every crossed module, Gaussian-smeared hits, uniform noise, truth-smeared seeds on the first layer-0 module), but the
particles are walked from surface to surface in whatever order THEY meet the barrel cylinders and the disc planes, so
that forward tracks leave the barrel through its end and continue over the discs.  A simulator of the data: no CKF
arithmetic, shared by the oracle-side and the CUDA-side tests.
"""
from __future__ import annotations

import math

import numpy as np

from .detector import Detector
from .events import (KAPPA, M_MUON, S_CLOSE, H_SIM, Event, _cross, _highland, _pick_module, _rk4, _to_plane)


def _to_cylinder_arr(r, d, lam, R, inhom):
    """Transport every particle to ITS cylinder of radius R[i] (outward).  Returns (r, d, ok)."""
    ok = np.ones(r.shape[0], bool)
    for _ in range(600):
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


def make_endcap_event(det: Detector, n_particles: int, seed: int, pt_min: float = 0.5, pt_max: float = 50.0,
                      eta_max: float = 3.0, noise_fraction: float = 0.2, n_fake_seeds: int = 0,
                      inhomogeneous: bool = False, precision: int = 64) -> Event:
    assert det.layer_kind is not None, "needs a detector with disc layers (build_detector(disc_z=...))"
    normal = np.cross(det.axis_u, det.axis_v)
    rng = np.random.Generator(np.random.Philox(key=seed))
    nb = det.n_barrel
    Rb, hzb = det.layer_r[:nb], det.layer_half_z[:nb]
    zd, rmin, rmax = det.layer_half_z, det.layer_r_min, det.layer_r
    # next disc of the same side (larger |z|), per layer; first disc of each side
    nxt = np.full(det.n_layers, -1, np.int64)
    for l in range(nb, det.n_layers):
        cand = [k for k in range(nb, det.n_layers) if (zd[k] > 0) == (zd[l] > 0) and abs(zd[k]) > abs(zd[l])]
        if cand:
            nxt[l] = min(cand, key=lambda k: abs(zd[k]))
    pos = [k for k in range(nb, det.n_layers) if zd[k] > 0]
    neg = [k for k in range(nb, det.n_layers) if zd[k] < 0]
    first_pos = min(pos, key=lambda k: zd[k]) if pos else -1
    first_neg = min(neg, key=lambda k: -zd[k]) if neg else -1

    n = int(n_particles)
    q = np.where(rng.random(n) < 0.5, -1.0, 1.0)
    pt = np.exp(rng.uniform(math.log(pt_min), math.log(pt_max), n))
    eta = rng.uniform(-eta_max, eta_max, n)
    phi0 = rng.uniform(0.0, 2.0 * math.pi, n)
    z0 = rng.normal(0.0, 50.0, n)
    theta = 2.0 * np.arctan(np.exp(-eta))
    p = pt * np.cosh(eta)
    qop = q / p
    lam = KAPPA * qop
    r = np.stack([np.zeros(n), np.zeros(n), z0], axis=1)
    d = np.stack([np.sin(theta) * np.cos(phi0), np.sin(theta) * np.sin(phi0), np.cos(theta)], axis=1)
    alive = np.ones(n, bool)
    lb = np.full(n, -1, np.int64)
    ld = np.where(d[:, 2] > 0, first_pos, first_neg).astype(np.int64)

    hit_pid, hit_mod, hit_l0, hit_l1 = [], [], [], []
    seed_found = np.zeros(n, bool)
    seed_mod = np.full(n, -1, np.int64)
    seed_par = np.zeros((n, 6))

    def cross_modules(layer, idx, i0, j0):
        """Module crossings of particles `idx` standing on the portal of `layer` near bin (i0, j0): the module hit and
        its overlap neighbours, hits recorded, Highland kicks applied."""
        nz = int(det.n_z[layer])
        exclude = np.full(idx.size, -1, np.int64)
        s_min = -1e-3
        for _ in range(3):
            if idx.size == 0:
                return
            mid = _pick_module(det, normal, layer, i0, j0, r[idx], d[idx], s_min, exclude)
            has = mid >= 0
            idx, mid = idx[has], mid[has]
            if idx.size == 0:
                return
            rr, dd = _to_plane(r[idx], d[idx], lam[idx], det.center[mid], normal[mid], inhomogeneous)
            r[idx], d[idx] = rr, dd
            rel = rr - det.center[mid]
            l0 = np.einsum("ij,ij->i", rel, det.axis_u[mid])
            l1 = np.einsum("ij,ij->i", rel, det.axis_v[mid])
            hit_pid.append(idx.copy()); hit_mod.append(mid.copy()); hit_l0.append(l0); hit_l1.append(l1)
            if layer == 0:
                first = ~seed_found[idx]
                fi = idx[first]
                seed_found[fi] = True
                seed_mod[fi] = mid[first]
                seed_par[fi, 0], seed_par[fi, 1] = l0[first], l1[first]
                seed_par[fi, 2] = np.arctan2(dd[first, 1], dd[first, 0])
                seed_par[fi, 3] = np.arctan2(np.hypot(dd[first, 0], dd[first, 1]), dd[first, 2])
                seed_par[fi, 4] = qop[fi]
            cosi = np.abs(np.einsum("ij,ij->i", dd, normal[mid]))
            th0 = _highland(p[idx], det.x_over_x0[mid] / cosi)
            k1 = rng.standard_normal(idx.size) * th0
            k2 = rng.standard_normal(idx.size) * th0
            # two directions orthogonal to d (d is never along z for both: fall back to x when it is)
            ref = np.where(np.abs(dd[:, 2:3]) < 0.9, np.array([[0.0, 0.0, 1.0]]), np.array([[1.0, 0.0, 0.0]]))
            e1 = _cross(dd, np.ascontiguousarray(np.broadcast_to(ref, dd.shape)))
            e1 /= np.linalg.norm(e1, axis=1)[:, None]
            e2 = _cross(dd, e1)
            dk = dd + k1[:, None] * e1 + k2[:, None] * e2
            dk /= np.linalg.norm(dk, axis=1)[:, None]
            d[idx] = dk
            loc_id = mid - int(det.module_offset[layer])
            i0, j0 = loc_id // nz, loc_id % nz
            exclude, s_min = mid, 1e-3

    for _it in range(4 * det.n_layers):
        if not alive.any():
            break
        z, dz = r[:, 2], d[:, 2]
        bxy = r[:, 0] * d[:, 0] + r[:, 1] * d[:, 1]
        rho2 = r[:, 0] ** 2 + r[:, 1] ** 2
        for _k in range(nb):                                    # barrel layers whose half length is already behind
            nx = np.minimum(lb + 1, nb - 1)
            skip = alive & (lb + 1 < nb) & (np.abs(z) > hzb[nx]) & (z * dz > 0.0)
            if not skip.any():
                break
            lb[skip] += 1
        for _k in range(det.n_layers):                          # discs not ahead, or radially behind
            lk = np.maximum(ld, 0)
            skip = alive & (ld >= 0) & (((zd[lk] - z) * dz <= 0.0) | ((rho2 > rmax[lk] ** 2) & (bxy > 0.0)))
            if not skip.any():
                break
            ld[skip] = nxt[lk[skip]]
        lc = np.where(lb + 1 < nb, lb + 1, -1)
        alive &= ~((lc < 0) & (ld < 0))
        a = d[:, 0] ** 2 + d[:, 1] ** 2
        cc = rho2 - Rb[np.maximum(lc, 0)] ** 2
        disc = bxy * bxy - a * cc
        den = bxy + np.sqrt(np.where(disc > 0, disc, 0.0))
        okc = (lc >= 0) & (disc >= 0.0) & (den > 0.0)           # (a particle on the beam line has bxy = 0 and still leaves)
        s_c = np.where(okc, -cc / np.where(okc, den, 1.0), np.inf)
        s_d = np.where(ld >= 0, (zd[np.maximum(ld, 0)] - z) / np.where(dz != 0.0, dz, 1.0), np.inf)
        to_disc = alive & (ld >= 0) & ((lc < 0) | (s_d < s_c))
        to_cyl = alive & ~to_disc
        alive &= ~(to_cyl & ~okc)                               # not radially outgoing and no disc ahead
        to_cyl &= alive
        # ---- cylinder portals
        idx = np.nonzero(to_cyl)[0]
        if idx.size:
            rr, dd, ok = _to_cylinder_arr(r[idx], d[idx], lam[idx], Rb[lc[idx]], inhomogeneous)
            r[idx[ok]], d[idx[ok]] = rr[ok], dd[ok]
            alive[idx[~ok]] = False
            idx = idx[ok]
            lay = lc[idx]
            lb[idx] = lay
            inacc = np.abs(r[idx, 2]) <= hzb[lay]
            idx, lay = idx[inacc], lay[inacc]
            for layer in np.unique(lay):
                sel = idx[lay == layer]
                nphi, nz = int(det.n_phi[layer]), int(det.n_z[layer])
                ln = 2.0 * float(det.half_v[det.module_offset[layer]])
                ph = np.arctan2(r[sel, 1], r[sel, 0])
                i0 = np.rint(ph * nphi / (2.0 * np.pi)).astype(np.int64) % nphi
                j0 = np.clip(np.floor((r[sel, 2] + hzb[layer]) / ln).astype(np.int64), 0, nz - 1)
                cross_modules(int(layer), sel, i0, j0)
        # ---- disc portals
        idx = np.nonzero(to_disc)[0]
        if idx.size:
            lay = ld[idx]
            c = np.stack([np.zeros(idx.size), np.zeros(idx.size), zd[lay]], axis=1)
            nrm = np.stack([np.zeros(idx.size), np.zeros(idx.size), np.sign(zd[lay])], axis=1)
            rr, dd = _to_plane(r[idx], d[idx], lam[idx], c, nrm, inhomogeneous)
            r[idx], d[idx] = rr, dd
            ld[idx] = nxt[lay]
            rho = np.hypot(rr[:, 0], rr[:, 1])
            lb[idx] = np.searchsorted(Rb, rho, side="right") - 1
            inacc = (rho >= rmin[lay]) & (rho <= rmax[lay])
            idx, lay, rho = idx[inacc], lay[inacc], rho[inacc]
            for layer in np.unique(lay):
                m = lay == layer
                sel = idx[m]
                nphi, nz = int(det.n_phi[layer]), int(det.n_z[layer])
                ln = 2.0 * float(det.half_v[det.module_offset[layer]])
                ph = np.arctan2(r[sel, 1], r[sel, 0])
                i0 = np.rint(ph * nphi / (2.0 * np.pi)).astype(np.int64) % nphi
                j0 = np.clip(np.floor((rho[m] - rmin[layer]) / ln).astype(np.int64), 0, nz - 1)
                cross_modules(int(layer), sel, i0, j0)

    # ---- measurements, noise, seeds: as in events.make_event
    pid = np.concatenate(hit_pid) if hit_pid else np.zeros(0, np.int64)
    mod = np.concatenate(hit_mod) if hit_mod else np.zeros(0, np.int64)
    tl0 = np.concatenate(hit_l0) if hit_l0 else np.zeros(0)
    tl1 = np.concatenate(hit_l1) if hit_l1 else np.zeros(0)
    nsig = pid.size
    sig = det.sigma[det.module_layer[mod]]
    m0 = tl0 + rng.standard_normal(nsig) * sig[:, 0]
    m1 = tl1 + rng.standard_normal(nsig) * sig[:, 1]
    nnoise = int(round(noise_fraction * nsig))
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

    sp = np.nonzero(seed_found)[0]
    par = seed_par[sp].copy()
    sig_s = np.stack([np.full(sp.size, 0.05), np.full(sp.size, 0.1), np.full(sp.size, 1e-3), np.full(sp.size, 1e-3),
                      0.05 * np.abs(par[:, 4]), np.zeros(sp.size)], axis=1)
    par += rng.standard_normal((sp.size, 6)) * sig_s
    smod, spid = seed_mod[sp], sp.astype(np.int64)
    if n_fake_seeds > 0:
        nf = int(n_fake_seeds)
        fq = np.where(rng.random(nf) < 0.5, -1.0, 1.0)
        fpt = np.exp(rng.uniform(math.log(pt_min), math.log(pt_max), nf))
        feta = rng.uniform(-eta_max, eta_max, nf)
        fphi = rng.uniform(-math.pi, math.pi, nf)
        fmod = rng.integers(0, int(det.module_offset[1]), nf)
        fpar = np.zeros((nf, 6))
        fpar[:, 0] = rng.uniform(-1.0, 1.0, nf) * det.half_u[fmod]
        fpar[:, 1] = rng.uniform(-1.0, 1.0, nf) * det.half_v[fmod]
        fpar[:, 2], fpar[:, 3] = fphi, 2.0 * np.arctan(np.exp(-feta))
        fpar[:, 4] = fq / (fpt * np.cosh(feta))
        fsig = np.stack([np.full(nf, 0.05), np.full(nf, 0.1), np.full(nf, 1e-3), np.full(nf, 1e-3),
                         0.05 * np.abs(fpar[:, 4]), np.zeros(nf)], axis=1)
        par, sig_s = np.concatenate([par, fpar]), np.concatenate([sig_s, fsig])
        smod, spid = np.concatenate([smod, fmod]), np.concatenate([spid, np.full(nf, -1, np.int64)])
    S = par.shape[0]
    cov = np.zeros((S, 6, 6))
    diag = 10.0 * sig_s ** 2
    diag[:, 5] = 1.0
    cov[:, np.arange(6), np.arange(6)] = diag
    T = np.float64 if precision == 64 else np.float32
    return Event(config=-1, event_index=seed, precision=precision, module_offsets=offsets.astype(np.int32),
                 loc=np.ascontiguousarray(all_loc.astype(T)), var=np.ascontiguousarray(all_var.astype(T)),
                 meas_particle=all_pid.astype(np.int32), meas_module=all_mod.astype(np.int32),
                 seed_module=smod.astype(np.int32), seed_params=np.ascontiguousarray(par.astype(T)),
                 seed_cov=np.ascontiguousarray(cov.reshape(S, 36).astype(T)), seed_particle=spid.astype(np.int32),
                 particle_q=q, particle_pt=pt, particle_eta=eta, particle_phi=phi0, particle_z0=z0,
                 n_signal=int(nsig), n_noise=int(nnoise))
