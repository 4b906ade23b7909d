"""Pins of the oracle's triplet seeding and helix parameter estimation (rules S0-S6)."""
import math

import numpy as np
import pytest

import oracle
import synth
from synth.events import CKFSettings, KAPPA
from tests.test_oracle_pins import _helix


def _cross_module_on_helix(det, layer, r0, d0, qop, bz):
    """Analytic helix -> the module of `layer` it crosses: bisection on every module plane of the layer near the
    helix's azimuth; returns (module, local l0, l1, arc length)."""
    n_all = np.cross(det.axis_u, det.axis_v)
    best = None
    for k in range(det.module_offset[layer], det.module_offset[layer + 1]):
        c, n = det.center[k], n_all[k]
        if np.dot(n[:2], d0[:2]) < 0.5 * np.hypot(*d0[:2]):
            continue
        f = lambda s: float(np.dot(_helix(r0, d0, qop, bz, s)[0] - c, n))
        lo, hi = 0.0, 400.0
        if not (f(lo) < 0.0 < f(hi)):
            continue
        for _ in range(100):
            mid = 0.5 * (lo + hi)
            if f(mid) < 0.0:
                lo = mid
            else:
                hi = mid
        s = 0.5 * (lo + hi)
        q = _helix(r0, d0, qop, bz, s)[0] - c
        l0, l1 = float(np.dot(q, det.axis_u[k])), float(np.dot(q, det.axis_v[k]))
        if abs(l0) <= det.half_u[k] and abs(l1) <= det.half_v[k] and (best is None or s < best[3]):
            best = (k, l0, l1, s)
    return best


@pytest.mark.parametrize("pt,q,eta,phi", [(0.6, 1.0, 0.3, 0.4), (2.0, -1.0, -0.8, 2.9), (20.0, 1.0, 0.9, -1.7),
                                         (1.0, -1.0, 0.0, 5.0)])
def test_parameter_estimation_is_exact_on_a_helix(detector, pt, q, eta, phi):
    """Three exact points of a helix in a uniform field determine it: S5 must return the tangent direction and q/p at
    the bottom point (closed form written here) to rounding."""
    det = detector
    theta = 2.0 * math.atan(math.exp(-eta))
    qop = q / (pt * math.cosh(eta))
    d0 = np.array([math.sin(theta) * math.cos(phi), math.sin(theta) * math.sin(phi), math.cos(theta)])
    r0 = np.array([0.3, -0.2, 12.0])
    hits = [_cross_module_on_helix(det, l, r0, d0, qop, 2.0) for l in (0, 1, 2)]
    assert all(h is not None for h in hits)
    order = np.argsort([h[0] for h in hits])
    mods = np.array([hits[i][0] for i in order])
    loc = np.array([[hits[i][1], hits[i][2]] for i in order])
    off = np.zeros(det.n_modules + 1, np.int32)
    np.add.at(off, mods + 1, 1)
    off = np.cumsum(off).astype(np.int32)
    var = np.tile([0.015 ** 2, 0.05 ** 2], (3, 1))
    st = oracle.Setup(det, synth.uniform_field(), CKFSettings())
    sd = oracle.seed_find(st, synth.SeedSettings(), off, loc, var)
    assert len(sd["module"]) == 1 and sd["module"][0] == hits[0][0]
    _, dB = _helix(r0, d0, qop, 2.0, hits[0][3])                      # truth direction at the bottom point
    x = sd["params"][0]
    assert abs(x[0] - hits[0][1]) < 1e-12 and abs(x[1] - hits[0][2]) < 1e-12
    dphi = (x[2] - math.atan2(dB[1], dB[0]) + math.pi) % (2 * math.pi) - math.pi
    assert abs(dphi) < 1e-9
    assert abs(x[3] - math.atan2(math.hypot(dB[0], dB[1]), dB[2])) < 1e-9
    assert abs(x[4] / qop - 1.0) < 1e-8
    C = sd["cov"][0].reshape(6, 6)
    assert np.count_nonzero(C - np.diag(np.diag(C))) == 0 and np.all(np.diag(C) > 0) and C[5, 5] == 1.0


@pytest.mark.parametrize("tight", [False, True])
def test_triplets_equal_brute_force_with_textbook_formulas(detector, tight):
    """S1-S4 on a small event against a vectorised enumeration of ALL (bottom, middle, top) combinations, the cuts
    evaluated with other textbook formulas than the oracle's: circumradius from the side lengths and the triangle area
    (R = abc / 4A), distance of the circle from the axis through the power of the origin."""
    det, fld, cfg = synth.config_bundle(1)
    ev = synth.make_event(1, det=det, n_particles=70)
    # tight: every cut binds on this small event (a wrong z0, d0 or dphi expression then changes the set)
    s = synth.SeedSettings(dphi_max=0.02, z0_max=25.0, dcot_max=0.004, pt_min=0.8, d0_max=0.3, cot_max=0.7) if tight \
        else synth.SeedSettings()
    st = oracle.Setup(det, fld, cfg.ckf)
    sd = oracle.seed_find(st, s, ev.module_offsets, ev.loc, ev.var)
    got = {tuple(int(v) for v in t) for t in sd["triplets"]}
    mod = ev.meas_module
    g = det.center[mod] + ev.loc[:, :1] * det.axis_u[mod] + ev.loc[:, 1:] * det.axis_v[mod]
    lay = det.module_layer[mod]
    idx = [np.flatnonzero(lay == l) for l in (s.layer_b, s.layer_m, s.layer_t)]
    B, M, T = (g[i] for i in idx)
    rho = lambda P: np.hypot(P[:, 0], P[:, 1])
    phi = lambda P: np.arctan2(P[:, 1], P[:, 0])

    def doublet(I, O):
        dphi = (phi(O)[None, :] - phi(I)[:, None] + np.pi) % (2 * np.pi) - np.pi
        drho = rho(O)[None, :] - rho(I)[:, None]
        cot = (O[None, :, 2] - I[:, None, 2]) / drho
        z0 = I[:, None, 2] - rho(I)[:, None] * cot
        return (np.abs(dphi) <= s.dphi_max) & (drho > 0) & (np.abs(cot) <= s.cot_max) & (np.abs(z0) <= s.z0_max), cot

    ok_bm, cot_bm = doublet(B, M)
    ok_mt, cot_mt = doublet(M, T)
    want = set()
    for ib, im in zip(*np.nonzero(ok_bm)):
        for it in np.flatnonzero(ok_mt[im] & (np.abs(cot_bm[ib, im] - cot_mt[im]) <= s.dcot_max)):
            P, Q, R3 = B[ib, :2], M[im, :2], T[it, :2]
            a, b, c = np.linalg.norm(Q - R3), np.linalg.norm(P - R3), np.linalg.norm(P - Q)
            area = 0.5 * abs((Q[0] - P[0]) * (R3[1] - P[1]) - (Q[1] - P[1]) * (R3[0] - P[0]))
            if area == 0.0:
                continue
            R = a * b * c / (4.0 * area)
            if KAPPA * 2.0 * R < s.pt_min:
                continue
            # power of the origin w.r.t. the circle = |OC|^2 - R^2 = (|OC| - R)(|OC| + R); |OC| from the perpendicular
            # bisectors solved as a 2x2 linear system
            A2 = 2.0 * np.array([Q - P, R3 - P])
            rhs = np.array([Q @ Q - P @ P, R3 @ R3 - P @ P])
            C = np.linalg.solve(A2, rhs)
            if abs(np.linalg.norm(C) - R) > s.d0_max:
                continue
            want.add((int(idx[0][ib]), int(idx[1][im]), int(idx[2][it])))
    assert len(want) >= (10 if tight else 70)
    assert got == want


def test_seeding_efficiency_pulls_and_the_chain_to_candidates():
    """Physics sanity (not a parity pin): every particle has a true triplet among the seeds, q/p pulls of the true
    triplets are unit-ish with the S6 variance, and the CKF started from the ESTIMATED seeds finds the particles."""
    det, fld, cfg = synth.config_bundle(1)
    ev = synth.make_event(1, det=det, n_particles=600)
    st = oracle.Setup(det, fld, cfg.ckf)
    s = synth.SeedSettings()
    sd = oracle.seed_find(st, s, ev.module_offsets, ev.loc, ev.var, n_threads=8)
    tp = ev.meas_particle[sd["triplets"]]
    true = (tp[:, 0] >= 0) & (tp[:, 0] == tp[:, 1]) & (tp[:, 1] == tp[:, 2])
    assert np.unique(tp[true, 0]).size >= 0.99 * 600
    qop = ev.particle_q / (ev.particle_pt * np.cosh(ev.particle_eta))
    pull = (sd["params"][true, 4] - qop[tp[true, 0]]) / np.sqrt(sd["cov"][true, 28] / s.cov_scale)
    assert abs(pull.mean()) < 0.15 and 0.5 < pull.std() < 1.3
    tr = oracle.ckf_find(st, ev.module_offsets, ev.loc, ev.var, sd["module"], sd["params"], sd["cov"], n_threads=8)
    found = set()
    n_p = np.bincount(ev.meas_particle[ev.meas_particle >= 0], minlength=600)
    for k in range(tr.n_tracks):
        p = ev.meas_particle[tr.meas_list(k)]
        p = p[p >= 0]
        if p.size:
            v, c = np.unique(p, return_counts=True)
            j = int(np.argmax(c))
            if 2 * c[j] > len(tr.meas_list(k)) and 2 * c[j] > n_p[v[j]]:      # PAPER.md:76 double matching
                found.add(int(v[j]))
    assert len(found) >= 0.98 * 600
