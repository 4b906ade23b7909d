"""Pins of the oracle's KF fit + RTS smoother (rules K1-K5, refs [8], [19]).

Nothing here calls the CUDA path.  What fixes the smoother from outside:
  * a scalar random walk, whose posterior has an information-form closed form (2 states) and a dense Gaussian
    conditioning (3 states) written here independently of the recursion;
  * on real tracks, the RTS output must be the exact posterior of the linear-Gaussian model defined by the
    stored Jacobians, predictions and noise: a dense joint covariance + one conditioning (40-digit mpmath);
  * the forward pass must reproduce the state the CKF reports for that candidate (it walks the same path);
  * pulls of the smoothed theta and q/p at the first measurement against the generator's truth.
"""
import numpy as np

import oracle
import synth


def _embed(vals, base=0.0):
    """[n] scalars -> [n, 6] vectors with the scalar in component 0."""
    out = np.full((len(vals), 6), base)
    out[:, 0] = vals
    return out


def _embed_cov(vals):
    out = np.tile(np.eye(6), (len(vals), 1, 1))
    out[:, 0, 0] = vals
    return out


def _scalar_forward(x0, p0, q, r, meas):
    xp, pp, xf, pf = [], [], [], []
    x, p = x0, p0
    for k, m in enumerate(meas):
        if k > 0:
            p = p + q
        xp.append(x); pp.append(p)
        g = p / (p + r)
        x = x + g * (m - x)
        p = (1.0 - g) * p
        xf.append(x); pf.append(p)
    return np.array(xp), np.array(pp), np.array(xf), np.array(pf)


def test_rts_scalar_random_walk_two_states_closed_form():
    x0, p0, q, r = 0.3, 2.0, 0.7, 0.25
    m = [1.1, -0.4]
    xp, pp, xf, pf = _scalar_forward(x0, p0, q, r, m)
    J = np.tile(np.eye(6), (2, 1, 1))
    rc, xs, Cs = oracle.rts_smooth(_embed(xp), _embed_cov(pp), _embed(xf), _embed_cov(pf), J)
    assert rc == 0
    # information form: z0 is seen by the prior, by m0 (variance r) and by m1 = z0 + w + v (variance q + r)
    prec = 1.0 / p0 + 1.0 / r + 1.0 / (q + r)
    want = (x0 / p0 + m[0] / r + m[1] / (q + r)) / prec
    assert abs(xs[0, 0] - want) < 1e-14
    assert abs(Cs[0, 0, 0] - 1.0 / prec) < 1e-14
    assert abs(xs[1, 0] - xf[1]) < 1e-15 and abs(Cs[1, 0, 0] - pf[1]) < 1e-15
    # the spectator components (identity model, nothing measured) stay put
    assert np.allclose(xs[:, 1:], 0.0) and np.allclose(Cs[:, 1:, 1:], np.eye(5))


def test_rts_scalar_three_states_dense_conditioning_with_drift():
    # z_{k+1} = a z_k + w: a != 1 catches a transposed / misplaced Jacobian, three states catch an index slip
    x0, p0, q, r, a = -0.2, 1.5, 0.4, 0.1, 0.8
    m = np.array([0.5, 0.9, -0.3])
    xp, pp, xf, pf = [], [], [], []
    x, p = x0, p0
    for k in range(3):
        if k > 0:
            x, p = a * x, a * a * p + q
        xp.append(x); pp.append(p)
        g = p / (p + r)
        x, p = x + g * (m[k] - x), (1 - g) * p
        xf.append(x); pf.append(p)
    J = np.tile(np.eye(6), (3, 1, 1))
    J[:, 0, 0] = a
    rc, xs, Cs = oracle.rts_smooth(_embed(xp), _embed_cov(pp), _embed(xf), _embed_cov(pf), J)
    assert rc == 0
    # dense: joint prior of (z0, z1, z2), then one conditioning on the three measurements
    mu = np.array([x0, a * x0, a * a * x0])
    S = np.zeros((3, 3))
    S[0, 0] = p0
    S[1, 1] = a * a * p0 + q
    S[2, 2] = a * a * S[1, 1] + q
    S[0, 1] = S[1, 0] = a * p0
    S[0, 2] = S[2, 0] = a * a * p0
    S[1, 2] = S[2, 1] = a * S[1, 1]
    G = S + r * np.eye(3)
    post = mu + S @ np.linalg.solve(G, m - mu)
    Spost = S - S @ np.linalg.solve(G, S)
    assert np.allclose(xs[:, 0], post, rtol=0, atol=1e-13)
    assert np.allclose(Cs[:, 0, 0], np.diag(Spost), rtol=0, atol=1e-13)


def _event_and_candidates(config, n_particles):
    det, fld, cfg = synth.config_bundle(config)
    ev = synth.make_event(config, det=det, n_particles=n_particles)
    st = oracle.Setup(det, fld, cfg.ckf)
    tr = oracle.find_event(st, ev, n_threads=4)
    return det, fld, cfg, ev, st, tr


def test_forward_pass_reproduces_the_ckf_candidate():
    _, _, _, ev, st, tr = _event_and_candidates(1, 60)
    assert tr.n_tracks > 40
    fit = oracle.kf_fit(st, ev, tr.track_offsets, tr.meas_idx, tr.seed_id, n_threads=4)
    assert np.all(fit.status == 0)
    # same path, same arithmetic: the filtered state at the last measurement IS the candidate's state (K2)
    assert np.array_equal(fit.last_params, tr.params)
    assert np.array_equal(fit.last_cov, tr.cov)
    assert np.allclose(fit.chi2_sum, tr.chi2_sum, rtol=1e-13, atol=0)
    n_meas = np.diff(tr.track_offsets)
    assert np.all(fit.n_states >= n_meas) and np.all(fit.n_states <= n_meas + tr.n_holes)
    # the last state is not smoothed: its smoothed parameters are the filtered ones
    last_entry = tr.track_offsets[1:] - 1
    assert np.array_equal(fit.entry_params[last_entry], tr.params)


def _dense_posterior(s, ev):
    """Exact posterior of the linear-Gaussian model the fit's stored quantities define (numpy, dense)."""
    n = len(s["module"])
    mu = np.zeros((n, 6))
    S = np.zeros((n, 6, n, 6))
    mu[0] = s["xp"][0]
    S[0, :, 0, :] = s["Cp"][0]
    for k in range(n - 1):
        Jk = s["J"][k + 1]
        mu[k + 1] = s["xp"][k + 1] + Jk @ (mu[k] - s["xf"][k])
        W = s["Cp"][k + 1] - Jk @ s["Cf"][k] @ Jk.T   # process noise of the step, in the arrival frame
        for j in range(k + 1):
            S[k + 1, :, j, :] = Jk @ S[k, :, j, :]
            S[j, :, k + 1, :] = S[k + 1, :, j, :].T
        S[k + 1, :, k + 1, :] = Jk @ S[k, :, k, :] @ Jk.T + W
    S = S.reshape(6 * n, 6 * n)
    # one conditioning on all measurements.  H only selects (l0, l1) of the measured states, so it is index work;
    # the prior variances of late states are 1e4 x the posterior ones, so the subtraction is done in 40 digits
    import mpmath as mp
    mp.mp.dps = 40
    idx, y, v = [], [], []
    for k in range(n):
        i = s["meas"][k]
        if i < 0:
            continue
        for a in range(2):
            idx.append(6 * k + a); y.append(float(ev.loc[i, a])); v.append(float(ev.var[i, a]))
    m = len(idx)
    Sm = mp.matrix(S.tolist())
    SH = mp.matrix(6 * n, m)
    G = mp.matrix(m, m)
    for c, j in enumerate(idx):
        for r in range(6 * n):
            SH[r, c] = Sm[r, j]
        for c2, j2 in enumerate(idx):
            G[c, c2] = Sm[j, j2] + (mp.mpf(v[c]) if c == c2 else 0)
    mu_f = mp.matrix(mu.reshape(-1).tolist())
    resid = mp.matrix([mp.mpf(y[c]) - mu_f[idx[c]] for c in range(m)])
    Gi = G ** -1
    K = SH * Gi
    post = mu_f + K * resid
    Spost = Sm - K * SH.T
    post = np.array([float(post[r]) for r in range(6 * n)]).reshape(n, 6)
    Spost = np.array([[float(Spost[r, c]) for c in range(6 * n)] for r in range(6 * n)]).reshape(n, 6, n, 6)
    return post, Spost


def test_rts_is_the_dense_posterior_of_the_linearised_track_model():
    _, _, _, ev, st, tr = _event_and_candidates(1, 40)
    checked = with_hole = 0
    for t in range(tr.n_tracks):
        meas = tr.meas_list(t)
        s = oracle.kf_fit_states(st, ev, int(tr.seed_id[t]), meas)
        assert s["status"] == 0
        if np.any(np.abs(s["xs"][:, 2]) > 3.0):
            continue                      # keep the dense model away from the phi wrap
        post, Spost = _dense_posterior(s, ev)
        n = len(s["module"])
        for k in range(n):
            sig = np.sqrt(np.diag(s["Cs"][k]))
            # the recursion and the dense solve agree to a small fraction of the smoothed sigma
            assert np.all(np.abs(s["xs"][k] - post[k]) < 1e-6 * sig), (t, k)
            Ck = Spost[k, :, k, :]
            assert np.all(np.abs(s["Cs"][k] - Ck) < 1e-5 * np.outer(sig, sig) + 1e-300), (t, k)
        with_hole += int(np.any(s["meas"] < 0))
        checked += 1
        if checked >= 12 and with_hole >= 1:
            break
    assert checked >= 10


def test_smoothing_tightens_the_first_state_and_pulls_are_unit():
    det, fld, cfg, ev, st, tr = _event_and_candidates(0, 100)
    fit = oracle.kf_fit(st, ev, tr.track_offsets, tr.meas_idx, tr.seed_id, n_threads=4)
    ok = fit.status == 0
    assert ok.sum() >= 90
    first = tr.track_offsets[:-1][ok]
    xs0 = fit.entry_params[first]
    C0 = fit.first_cov[ok].reshape(-1, 6, 6)
    pid = ev.seed_particle[tr.seed_id[ok]]
    p = ev.particle_pt[pid] * np.cosh(ev.particle_eta[pid])
    qop_true = ev.particle_q[pid] / p
    theta_true = 2.0 * np.arctan(np.exp(-ev.particle_eta[pid]))
    pull_q = (xs0[:, 4] - qop_true) / np.sqrt(C0[:, 4, 4])
    pull_t = (xs0[:, 3] - theta_true) / np.sqrt(C0[:, 3, 3])
    for pull in (pull_q, pull_t):
        assert abs(np.mean(pull)) < 0.4 and 0.6 < np.std(pull) < 1.5, (np.mean(pull), np.std(pull))
    # the seed knows q/p to 5 % (x sqrt(10) in its covariance); ten measurements in 2 T know it far better
    seed_var = ev.seed_cov.reshape(-1, 6, 6)[tr.seed_id[ok], 4, 4]
    assert np.median(C0[:, 4, 4] / seed_var) < 0.05
    # smoothed covariances are symmetric positive definite
    assert np.allclose(C0, np.swapaxes(C0, 1, 2))
    assert np.all(np.linalg.eigvalsh(C0 / np.sqrt(np.einsum("nii,njj->nij", C0, C0))) > 0)


# ---------------------------------------------------------------------------------- K4': two-filter smoother
def test_two_filter_smoother_is_the_dense_posterior_too():
    """The two-filter ('optimal') smoother of PAPER.md:100 shares nothing with the RTS recursion but the forward
    pass; on the same linearised model it must give the same exact posterior (40-digit dense conditioning) at EVERY
    state, and therefore the RTS result."""
    _, _, _, ev, st, tr = _event_and_candidates(1, 40)
    checked = with_hole = 0
    for t in range(tr.n_tracks):
        meas = tr.meas_list(t)
        s = oracle.kf_fit_states(st, ev, int(tr.seed_id[t]), meas, smoother=1)
        r = oracle.kf_fit_states(st, ev, int(tr.seed_id[t]), meas, smoother=0)
        assert s["status"] == 0 and r["status"] == 0
        sig = np.sqrt(np.einsum("kii->ki", r["Cs"]))
        assert np.all(np.abs(s["xs"] - r["xs"]) < 1e-9 * sig), t           # equals RTS
        assert np.all(np.abs(s["Cs"] - r["Cs"]) < 1e-7 * sig[:, :, None] * sig[:, None, :]), t
        if np.any(np.abs(s["xs"][:, 2]) > 3.0) or checked >= 8:
            continue
        post, Spost = _dense_posterior(s, ev)                              # and the dense posterior, on its own
        for k in range(len(s["module"])):
            assert np.all(np.abs(s["xs"][k] - post[k]) < 1e-6 * sig[k]), (t, k)
            assert np.all(np.abs(s["Cs"][k] - Spost[k, :, k, :]) < 1e-5 * np.outer(sig[k], sig[k])), (t, k)
        with_hole += int(np.any(s["meas"] < 0))
        checked += 1
    assert checked >= 8


def test_two_filter_smoother_scalar_closed_form():
    # the same two-state random walk as above, through the full fit interface is not possible (no detector), so the
    # closed form is checked on a real single-measurement-per-state track instead: with ONE state the smoothed state is
    # the filtered one, whatever the smoother
    det, fld, cfg, ev, st, tr = _event_and_candidates(0, 20)
    t = 0
    one = tr.meas_list(t)[:1]
    for kind in (0, 1):
        s = oracle.kf_fit_states(st, ev, int(tr.seed_id[t]), one, smoother=kind)
        assert s["status"] == 0 and len(s["module"]) == 1
        assert np.allclose(s["xs"][0], s["xf"][0], rtol=0, atol=1e-13 * np.maximum(1.0, np.abs(s["xf"][0])))
        sig = np.sqrt(np.diag(s["Cf"][0]))
        assert np.all(np.abs(s["Cs"][0] - s["Cf"][0]) < 1e-9 * np.outer(sig, sig))
