"""Pins of the oracle's CKF control flow (R9-R11, V2, V4) by brute force, plus physics sanity on config 0."""
import numpy as np
import pytest

import oracle
import synth
from synth.events import CKFSettings


def _toy(n_particles=5, n_layers=4, dup_sigma=1.0, seed_cfg=1):
    det = synth.build_detector(layer_r=synth.detector.LAYER_R[:n_layers])
    ev = synth.make_event(seed_cfg, det=det, n_particles=n_particles)
    # add, next to every true hit, a displaced copy so that branching really happens
    rng = np.random.default_rng(11)
    sig = np.sqrt(ev.var)
    keep = ev.meas_particle >= 0
    loc2 = ev.loc[keep] + dup_sigma * sig[keep] * rng.choice([-1.0, 1.0], size=(keep.sum(), 2))
    mod = np.concatenate([ev.meas_module, ev.meas_module[keep]])
    loc = np.concatenate([ev.loc, loc2])
    var = np.concatenate([ev.var, ev.var[keep]])
    order = np.argsort(mod, kind="stable")
    mod, loc, var = mod[order], loc[order], var[order]
    off = np.zeros(det.n_modules + 1, np.int64)
    np.add.at(off, mod + 1, 1)
    off = np.cumsum(off).astype(np.int32)
    return det, ev, off, loc, var


def _brute_force(st, ckf, off, loc, var, seed_module, seed_params, seed_cov):
    """Depth-first enumeration of every chi2-gated measurement combination (no caps)."""
    out = []

    def finish(seed, meas, chi2s, x, Cm):
        if len(meas) >= ckf.min_measurements:
            out.append((seed, tuple(meas), sum(chi2s), x, Cm))

    def rec(seed, module, x, Cm, first, meas, chi2s, n_holes, xs, Cs, level):
        if level >= ckf.max_levels:
            finish(seed, meas, chi2s, xs, Cs)
            return
        if first:
            tg, xp, Cp = module, x, Cm
        else:
            code, tg, xp, Cp, _ = oracle.move(st, module, x, Cm)
            if code != 0:
                finish(seed, meas, chi2s, xs, Cs)
                return
        passers = []
        for i in range(off[tg], off[tg + 1]):
            c2 = oracle.predicted_chi2(xp, Cp, loc[i], var[i])
            if c2 < ckf.chi2_max:
                passers.append((c2, i))
        if not passers:
            if n_holes + 1 > ckf.max_holes:
                finish(seed, meas, chi2s, xs, Cs)
            else:
                rec(seed, tg, xp, Cp, False, meas, chi2s, n_holes + 1, xs, Cs, level + 1)
            return
        for c2, i in passers:
            xu, Cu = oracle.kalman_update(xp, Cp, loc[i], var[i])
            rec(seed, tg, xu, Cu, False, meas + [i], chi2s + [c2], n_holes, xu, Cu, level + 1)

    for s in range(len(seed_module)):
        rec(s, int(seed_module[s]), seed_params[s].astype(np.float64), seed_cov[s].reshape(6, 6).astype(np.float64),
            True, [], [], 0, None, None, 0)
    return out


def test_toy_ckf_equals_brute_force_enumeration():
    det, ev, off, loc, var = _toy()
    ckf = CKFSettings(max_branches_per_surface=1000, max_candidates_per_seed=1000000, max_holes=3,
                      min_measurements=1, chi2_max=10.0)
    st = oracle.Setup(det, synth.uniform_field(), ckf)
    tr = oracle.ckf_find(st, off, loc, var, ev.seed_module, ev.seed_params, ev.seed_cov)
    bf = _brute_force(st, ckf, off, loc, var, ev.seed_module, ev.seed_params, ev.seed_cov)
    got = {(int(tr.seed_id[t]), tuple(int(i) for i in tr.meas_list(t))): t for t in range(tr.n_tracks)}
    want = {(s, m): (c2, x, Cm) for s, m, c2, x, Cm in bf}
    assert len(got) == tr.n_tracks            # two branches of one seed never share a list (R11)
    assert set(got) == set(want)
    assert tr.n_tracks > 3 * ev.n_seeds       # the toy really branches
    for key, t in got.items():
        c2, x, Cm = want[key]
        assert abs(tr.chi2_sum[t] - c2) < 1e-9 * max(1.0, c2)
        assert np.allclose(tr.params[t], x, rtol=1e-12, atol=1e-12)
        assert np.allclose(tr.cov[t].reshape(6, 6), Cm, rtol=1e-10, atol=1e-18)
        assert np.allclose(tr.entry_chi2[tr.track_offsets[t]:tr.track_offsets[t + 1]].sum(), c2)


def test_more_branches_only_add_candidates_when_cap_is_lifted():
    det, ev, off, loc, var = _toy(n_particles=8)
    prev = None
    for k in (1, 2, 3, 1000):
        ckf = CKFSettings(max_branches_per_surface=k, max_candidates_per_seed=1000000, min_measurements=1)
        st = oracle.Setup(det, synth.uniform_field(), ckf)
        tr = oracle.ckf_find(st, off, loc, var, ev.seed_module, ev.seed_params, ev.seed_cov)
        cur = {(int(tr.seed_id[t]), tuple(int(i) for i in tr.meas_list(t))) for t in range(tr.n_tracks)}
        if prev is not None:
            assert prev <= cur
        prev = cur


def test_branch_ranking_and_cap_order():
    """V2 ranks by (chi2, index); R10 keeps each tip's best-ranked children and cuts in tip order."""
    det, ev, off, loc, var = _toy(n_particles=6)
    big = CKFSettings(max_branches_per_surface=1000, max_candidates_per_seed=1000000, min_measurements=1)
    st = oracle.Setup(det, synth.uniform_field(), big)
    full = oracle.ckf_find(st, off, loc, var, ev.seed_module, ev.seed_params, ev.seed_cov)
    one = CKFSettings(max_branches_per_surface=1, max_candidates_per_seed=1, min_measurements=1)
    st1 = oracle.Setup(det, synth.uniform_field(), one)
    best = oracle.ckf_find(st1, off, loc, var, ev.seed_module, ev.seed_params, ev.seed_cov)
    # k = 1: the single candidate per seed follows, at every surface, the smallest chi2 among the full set's
    # continuations of the same prefix
    for t in range(best.n_tracks):
        s = int(best.seed_id[t])
        ml = [int(i) for i in best.meas_list(t)]
        c2 = best.entry_chi2[best.track_offsets[t]:best.track_offsets[t + 1]]
        for depth in range(len(ml)):
            alts = []
            for u in range(full.n_tracks):
                if int(full.seed_id[u]) != s:
                    continue
                mu = [int(i) for i in full.meas_list(u)]
                if mu[:depth] == ml[:depth] and len(mu) > depth:
                    alts.append((full.entry_chi2[full.track_offsets[u] + depth], mu[depth]))
            assert min(alts) == (c2[depth], ml[depth])
    # cap: never more candidates per seed than allowed, and the number of leaves is exactly min(cap, uncapped)
    for cap in (1, 2, 3, 7):
        c = CKFSettings(max_branches_per_surface=1000, max_candidates_per_seed=cap, min_measurements=0)
        trc = oracle.ckf_find(oracle.Setup(det, synth.uniform_field(), c), off, loc, var, ev.seed_module,
                              ev.seed_params, ev.seed_cov)
        cnt = np.bincount(trc.seed_id, minlength=ev.n_seeds)
        assert cnt.max() <= cap and cnt.min() >= 1


def test_k1_without_noise_is_the_plain_kalman_filter_along_truth(detector):
    det, fld, cfg = synth.config_bundle(0)
    ev = synth.make_event(0, det=det)
    st = oracle.Setup(det, fld, cfg.ckf)
    tr = oracle.find_event(st, ev)
    n_checked = 0
    for t in range(tr.n_tracks):
        s = int(tr.seed_id[t])
        ml = [int(i) for i in tr.meas_list(t)]
        truth = [int(i) for i in np.nonzero(ev.meas_particle == ev.seed_particle[s])[0]]
        if sorted(ml) != sorted(truth) or tr.n_holes[t] != 0:
            continue
        # sequential KF over the found list with the primitives
        x = ev.seed_params[s].astype(np.float64)
        Cm = ev.seed_cov[s].reshape(6, 6).astype(np.float64)
        m = int(ev.seed_module[s])
        c2sum = 0.0
        for n, i in enumerate(ml):
            if n > 0:
                code, m, x, Cm, _ = oracle.move(st, m, x, Cm)
                assert code == 0 and m == ev.meas_module[i]
            c2sum += oracle.predicted_chi2(x, Cm, ev.loc[i], ev.var[i])
            x, Cm = oracle.kalman_update(x, Cm, ev.loc[i], ev.var[i])
        assert np.allclose(tr.params[t], x, rtol=1e-12, atol=1e-12)
        assert abs(tr.chi2_sum[t] - c2sum) < 1e-9
        n_checked += 1
    assert n_checked >= 80


def test_config0_physics_sanity():
    """Statistical sanity (not a parity pin): chi2 per 2-dof hit ~ 2, q/p pull ~ N(0,1), own hits recovered."""
    det, fld, cfg = synth.config_bundle(0)
    pulls, chi2_per_hit, own = [], [], 0
    n_seeds = 0
    for e in range(4):
        ev = synth.make_event(0, event_index=e, det=det)
        st = oracle.Setup(det, fld, cfg.ckf)
        tr = oracle.find_event(st, ev)
        n_seeds += ev.n_seeds
        for t in range(tr.n_tracks):
            s = int(tr.seed_id[t])
            pid = int(ev.seed_particle[s])
            ml = tr.meas_list(t)
            truth = np.nonzero(ev.meas_particle == pid)[0]
            if set(ml.tolist()) == set(truth.tolist()):
                own += 1
            qop_true = ev.particle_q[pid] / (ev.particle_pt[pid] * np.cosh(ev.particle_eta[pid]))
            pulls.append((tr.params[t, 4] - qop_true) / np.sqrt(tr.cov[t, 4 * 6 + 4]))
            chi2_per_hit.append(tr.chi2_sum[t] / len(ml))
    pulls = np.array(pulls)
    assert own >= 0.85 * n_seeds
    assert abs(np.mean(pulls)) < 0.25 and 0.7 < np.std(pulls) < 1.4
    assert 1.0 < np.mean(chi2_per_hit) < 2.4
