"""GPU-less check of the CUDA path's per-tip arithmetic (csrc/ckf_math.cuh, ckf_nav.cuh compiled for the host by
tests/hostcheck) against the oracle: every surface-to-surface move and every update along config 0 / config 2
tracks.  The kernels inline exactly these functions; the -m gpu tests then check the orchestration."""
import numpy as np
import pytest

import oracle
import synth
from tests.hostcheck import HostMath


def _rel(a, b, floor):
    return np.abs(a - b) / np.maximum(np.maximum(np.abs(a), np.abs(b)), floor)


@pytest.mark.parametrize("config,precision,tol_x,tol_c,eloss", [(0, 64, 1e-10, 1e-9, 0), (2, 64, 1e-10, 1e-9, 0),
                                                                (2, 32, 1e-9, 2e-6, 0), (1, 64, 1e-10, 1e-9, 1),
                                                                (2, 32, 1e-9, 2e-6, 1)])
def test_moves_and_updates_match_oracle(config, precision, tol_x, tol_c, eloss):
    import copy
    det, fld, cfg = synth.config_bundle(config)
    cfg = copy.deepcopy(cfg)
    cfg.ckf.energy_loss = eloss        # rule E (mean energy loss per module), off in the BASELINE configs
    ev = synth.make_event(config, det=det, n_particles=60, n_fake_seeds=0)
    st = oracle.Setup(det, fld, cfg.ckf)
    hm = HostMath(det, fld, cfg.ckf)
    floor_x = np.array([1.0, 1.0, 1.0, 1.0, 0.0, 1.0])
    n_moves = n_upd = 0
    for s in range(ev.n_seeds):
        x = ev.seed_params[s].astype(np.float64)
        Cm = ev.seed_cov[s].reshape(6, 6).astype(np.float64)
        m = int(ev.seed_module[s])
        truth = np.nonzero(ev.meas_particle == ev.seed_particle[s])[0]
        for level in range(20):
            if level > 0:
                co, tgo, xo, Co, _ = oracle.move(st, m, x, Cm)
                ch, tgh, xh, Ch, _ = hm.move(precision, m, x, Cm)
                assert co == ch
                if co != 0:
                    break
                assert tgo == tgh
                fl = floor_x.copy()
                fl[4] = abs(xo[4])
                assert np.max(_rel(xo, xh, fl)) < tol_x
                scale = np.sqrt(np.outer(np.diag(Co), np.diag(Co)))
                assert np.max(np.abs(Co - Ch) / scale) < tol_c
                n_moves += 1
                x, Cm, m = xo, Co, tgo
            # update with this particle's hit on the module, if any
            hits = [i for i in truth if ev.meas_module[i] == m]
            if hits:
                i = hits[0]
                loc, var = ev.loc[i].astype(np.float64), ev.var[i].astype(np.float64)
                xu, Cu = oracle.kalman_update(x, Cm, loc, var)
                c2 = oracle.predicted_chi2(x, Cm, loc, var)
                xh, Ch, c2h = hm.update(precision, x, Cm, loc, var)
                assert abs(c2 - c2h) < 1e-9 * max(1.0, c2)       # chi2 is a float64 function of its inputs in both modes
                fl = floor_x.copy()
                fl[4] = abs(xu[4])
                assert np.max(_rel(xu, xh, fl)) < 1e-12
                scale = np.sqrt(np.outer(np.diag(Cu), np.diag(Cu)))
                assert np.max(np.abs(Cu - Ch) / scale) < 1e-9
                n_upd += 1
                x, Cm = xu, Cu
    assert n_moves > 400 and n_upd > 400


def test_field_read_matches_oracle():
    det, fld, cfg = synth.config_bundle(2)
    st = oracle.Setup(det, fld, cfg.ckf)
    hm = HostMath(det, fld, cfg.ckf)
    rng = np.random.default_rng(2)
    for _ in range(300):
        r = rng.uniform(-1090, 1090, 3)
        assert np.max(np.abs(oracle.field_at(st, r) - hm.field(r))) < 1e-12


@pytest.mark.parametrize("precision", [64, 32])
def test_moves_with_endcap_discs_match_oracle(precision):
    """Row f3: barrel -> disc -> disc navigation (N3' portals) of the CUDA path's per-tip code against the oracle, move by
    move along the truth of forward and central particles (|eta| up to 3)."""
    from synth.events import CKFSettings
    det = synth.build_detector(half_z=500.0, disc_z=(560.0, 640.0, 740.0, 860.0, 1000.0))
    fld = synth.uniform_field()
    ev = synth.make_endcap_event(det, 150, seed=11, noise_fraction=0.0)
    ckf = CKFSettings(surface_tolerance_mm=1e-5 if precision == 64 else 1e-2)
    st = oracle.Setup(det, fld, ckf)
    hm = HostMath(det, fld, ckf)
    floor_x = np.array([1.0, 1.0, 1.0, 1.0, 0.0, 1.0])
    n_moves = n_disc = n_exit = 0
    for s in range(ev.n_seeds):
        x = ev.seed_params[s].astype(np.float64)
        Cm = ev.seed_cov[s].reshape(6, 6).astype(np.float64)
        m = int(ev.seed_module[s])
        for level in range(30):
            co, tgo, xo, Co, _ = oracle.move(st, m, x, Cm)
            ch, tgh, xh, Ch, trials = hm.move(precision, m, x, Cm)
            assert co == ch, (s, level, co, ch)
            assert trials == oracle.last_move_trials(), (s, level)     # same sequence of RKN4 trials, stops included
            if co != 0:
                n_exit += oracle.STOP_NAMES[co] == "EXIT"
                break
            assert tgo == tgh, (s, level, tgo, tgh)
            fl = floor_x.copy()
            fl[4] = abs(xo[4])
            assert np.max(_rel(xo, xh, fl)) < (1e-10 if precision == 64 else 1e-9)
            scale = np.sqrt(np.outer(np.diag(Co), np.diag(Co)))
            assert np.max(np.abs(Co - Ch) / scale) < (1e-9 if precision == 64 else 2e-6)
            n_moves += 1
            n_disc += int(det.layer_kind[det.module_layer[tgo]])
            x, Cm, m = xo, Co, tgo
    assert n_moves > 900 and n_disc > 300 and n_exit > 100


@pytest.mark.parametrize("endcap", [False, True])
def test_bidirectional_moves_match_oracle(endcap):
    """config.bidirectional = 1 (rules N3''): inward-pointing fake seeds are walked through the inner layers, past the
    beam line and out of the far side; every move of the CUDA path's per-tip code against the oracle (stop codes,
    targets, RKN4 trial counts, parameters)."""
    from synth.events import CKFSettings
    if endcap:
        det = synth.build_detector(half_z=500.0, disc_z=(560.0, 640.0, 740.0, 860.0, 1000.0))
        ev = synth.make_endcap_event(det, 40, seed=5, n_fake_seeds=260, noise_fraction=0.0)
    else:
        det = synth.build_detector()
        ev = synth.make_event(1, det=det, n_particles=40, n_fake_seeds=260)
    fld = synth.uniform_field()
    ckf = CKFSettings(bidirectional=1)
    st = oracle.Setup(det, fld, ckf)
    hm = HostMath(det, fld, ckf)
    n_moves = n_inward = n_exit = 0
    for s in range(ev.n_seeds):
        x = ev.seed_params[s].astype(np.float64)
        Cm = ev.seed_cov[s].reshape(6, 6).astype(np.float64)
        m = int(ev.seed_module[s])
        for level in range(40):
            nrm = np.cross(det.axis_u[m], det.axis_v[m])
            d = np.array([np.sin(x[3]) * np.cos(x[2]), np.sin(x[3]) * np.sin(x[2]), np.cos(x[3])])
            co, tgo, xo, Co, _ = oracle.move(st, m, x, Cm)
            ch, tgh, xh, Ch, trials = hm.move(64, m, x, Cm)
            assert co == ch and trials == oracle.last_move_trials(), (s, level, co, ch)
            if co != 0:
                n_exit += oracle.STOP_NAMES[co] == "EXIT"
                break
            assert tgo == tgh, (s, level)
            assert np.max(np.abs(xo - xh) / np.maximum(np.abs(xo), 1.0)) < 1e-10
            scale = np.sqrt(np.outer(np.diag(Co), np.diag(Co)))
            assert np.max(np.abs(Co - Ch) / scale) < 1e-9
            n_moves += 1
            n_inward += int(np.dot(d, nrm) < 0.0)
            x, Cm, m = xo, Co, tgo
    assert n_moves > 2000 and n_inward > 80 and n_exit > 250, (n_moves, n_inward, n_exit)


def test_field_gradient_read_is_the_derivative_of_the_field_read():
    """J2' on the CUDA side: field_gradient_at against central differences of ITS OWN field_at inside a cell (the
    interpolant is trilinear: the difference quotient along one axis is exact up to rounding), at random points."""
    det, fld, cfg = synth.config_bundle(2)
    hm = HostMath(det, fld, cfg.ckf)
    rng = np.random.default_rng(5)
    sp = float(fld.spacing[0])
    worst = 0.0
    for _ in range(200):
        cell = rng.integers(2, int(fld.n[0]) - 3, 3)
        r = fld.origin + sp * (cell + rng.uniform(0.2, 0.8, 3))
        G = hm.field_gradient(r)
        for j in range(3):
            e = np.zeros(3)
            e[j] = 0.1 * sp
            fd = (hm.field(r + e) - hm.field(r - e)) / (2 * e[j])
            worst = max(worst, float(np.max(np.abs(G[:, j] - fd))))
    scale = float(np.max(np.abs(hm.field_gradient(fld.origin + sp * 20.3))))
    assert scale > 1e-7 and worst < 1e-9 * max(1.0, scale / 1e-6), (worst, scale)


@pytest.mark.parametrize("precision,tol_x,tol_c", [(64, 1e-10, 1e-9), (32, 1e-9, 2e-6)])
def test_moves_with_field_gradient_match_oracle(precision, tol_x, tol_c):
    """Row f3, J2' (config.field_gradient = 1, reading A13): the CUDA path's transport with the field-gradient terms
    (MoveG: the d-, q- and the two position columns pushed through the four stages, csrc/ckf_math.cuh) against the
    oracle's 8 x 8 tangent form, move by move through the inhomogeneous grid field of config 2 -- and the terms must
    matter: against the oracle WITHOUT them the same covariances differ by far more than the tolerance."""
    import copy
    det, fld, cfg = synth.config_bundle(2)
    cfg = copy.deepcopy(cfg)
    cfg.ckf.field_gradient = 1
    off = copy.deepcopy(cfg)
    off.ckf.field_gradient = 0
    ev = synth.make_event(2, det=det, n_particles=60, n_fake_seeds=0)
    st, st_off = oracle.Setup(det, fld, cfg.ckf), oracle.Setup(det, fld, off.ckf)
    hm = HostMath(det, fld, cfg.ckf)
    floor_x = np.array([1.0, 1.0, 1.0, 1.0, 0.0, 1.0])
    n_moves, worst_c, effect = 0, 0.0, 0.0
    for s in range(ev.n_seeds):
        x = ev.seed_params[s].astype(np.float64)
        Cm = ev.seed_cov[s].reshape(6, 6).astype(np.float64)
        m = int(ev.seed_module[s])
        for level in range(1, 14):
            co, tgo, xo, Co, _ = oracle.move(st, m, x, Cm)
            tro = oracle.last_move_trials()
            ch, tgh, xh, Ch, trh = hm.move(precision, m, x, Cm)
            assert co == ch
            if co != 0:
                break
            assert tgo == tgh and tro == trh
            fl = floor_x.copy()
            fl[4] = abs(xo[4])
            assert np.max(_rel(xo, xh, fl)) < tol_x
            scale = np.sqrt(np.outer(np.diag(Co), np.diag(Co)))
            worst_c = max(worst_c, float(np.max(np.abs(Co - Ch) / scale)))
            _, _, x0, C0, _ = oracle.move(st_off, m, x, Cm)
            assert np.array_equal(x0, xo)                        # the flag never touches the state
            effect = max(effect, float(np.max(np.abs(Co - C0) / scale)))
            n_moves += 1
            x, Cm, m = xo, Co, tgo
    assert n_moves > 400 and worst_c < tol_c, (n_moves, worst_c)
    assert effect > 100 * tol_c, effect
