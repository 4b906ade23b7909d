"""More pins of the CPU oracle (round 2): the parts the round-1 pins left open.

* P2/P3 stage points in a NON-uniform field: the oracle's adaptive RKN4 against an independent ODE integrator
  (scipy DOP853, rtol 1e-13) of dr/ds = d, dd/ds = lambda d x B(r) -- in the analytic map of configs[2] (a pin hook of
  the oracle, field kind 2) and through the float32 grid read by scipy's own multilinear interpolator.
* V5 path factor x/X0 / |d.n| for an inclined track, the incidence computed here from the module normal.
* R10 against a literal greedy written here: one extra child at a time, in tip order, until the seed holds `cap` leaves.
* D11 against the literal SURVEY N3 walk: same candidates, only stop reasons may differ.
None of these re-types an oracle formula.
"""
import math

import numpy as np
import pytest

import oracle
import synth
from synth.events import CKFSettings, KAPPA, M_MUON
from synth.field import A_INHOM, B0, FieldSpec

pytestmark = pytest.mark.filterwarnings("ignore")


def _analytic_field_spec():
    """Oracle pin hook (field kind 2): B0 in uniform_b[2], a in origin[0]."""
    return FieldSpec(2, np.array([0.0, 0.0, B0]), np.zeros(3, np.int32), np.array([A_INHOM, 0.0, 0.0]), np.ones(3), None)


def _dop853(bfun, r0, d0, qop, s_end):
    from scipy.integrate import solve_ivp
    lam = KAPPA * qop

    def rhs(_s, y):
        return np.concatenate([y[3:], lam * np.cross(y[3:], bfun(y[:3]))])

    sol = solve_ivp(rhs, [0.0, s_end], np.concatenate([r0, d0]), method="DOP853", rtol=1e-13, atol=1e-13)
    assert sol.success
    return sol.y[:3, -1], sol.y[3:, -1]


def _start(pt, q, theta, phi, r0):
    p = pt / math.sin(theta)
    d0 = np.array([math.sin(theta) * math.cos(phi), math.sin(theta) * math.sin(phi), math.cos(theta)])
    beta = p / math.sqrt(p * p + M_MUON ** 2)
    return np.concatenate([r0, [0.0], d0, [q / p]]), d0, q / p, beta


# ------------------------------------------------------------------ P2-P5 in a non-uniform field
@pytest.mark.parametrize("pt,q,theta", [(0.5, 1.0, 0.75), (0.8, -1.0, 2.2), (3.0, 1.0, 1.0)])
def test_stepping_in_analytic_nonuniform_field_vs_dop853(detector, pt, q, theta):
    """Far from z = 0 the map changes by ~1.5 % over one 100 mm step, so B1 != B2 != B4: a stage evaluated at the wrong
    point (or the wrong B in a stage) costs orders of magnitude here and nothing in a uniform field."""
    r0 = np.array([20.0, -10.0, 300.0 if theta < 1.5 else -300.0])
    y0, d0, qop, beta = _start(pt, q, theta, 0.4, r0)
    bfun = lambda r: synth.analytic_b(r[None, :], True)[0]
    errs, nsteps = [], []
    for tol in (1e-4, 1e-6, 1e-8):
        st = oracle.Setup(detector, _analytic_field_spec(),
                          CKFSettings(rk_tolerance_mm=tol, surface_tolerance_mm=1e-10, max_rk_steps_per_surface=100000))
        code, y1, _, ns = oracle.propagate_free(st, y0, cylinder_r=700.0)
        assert code == 0
        pos, dirn = _dop853(bfun, r0, d0, qop, y1[3] * beta)     # arc length from the time coordinate
        errs.append(max(np.max(np.abs(pos - y1[:3])), 1e3 * np.max(np.abs(dirn - y1[4:7]))))
        nsteps.append(ns)
    # the error follows the tolerance (~ linearly: global error ~ sum of local errors ~ tol) ...
    assert errs[0] > 5.0 * errs[1] > 25.0 * errs[2], errs
    assert errs[2] < 2e-7 and errs[1] < 2e-5, errs
    # ... and the estimator sees a 4th-order scheme: step counts grow like tol^(-1/4), not like tol^(-1/2) or worse
    assert nsteps[0] <= 60 and nsteps[2] <= 16 * nsteps[0], nsteps      # measured: 46 / 137 / 423 = x 3.0 per 100


def test_stepping_through_the_float32_grid_vs_dop853(detector):
    """Same check through the grid: the reference integrates the field scipy's multilinear interpolator reads from
    the same float32 nodes, so the two solve the same (piecewise smooth) ODE."""
    from scipy.interpolate import RegularGridInterpolator
    fs = synth.grid_field()
    axes = [fs.origin[a] + fs.spacing[a] * np.arange(fs.n[a]) for a in range(3)]
    interp = RegularGridInterpolator(axes, fs.grid.astype(np.float64), method="linear")
    bfun = lambda r: interp(r[None, :])[0]
    r0 = np.array([15.0, 5.0, 250.0])
    y0, d0, qop, beta = _start(0.6, -1.0, 0.8, -1.1, r0)
    errs = []
    for tol in (1e-5, 1e-7):
        st = oracle.Setup(detector, fs, CKFSettings(rk_tolerance_mm=tol, surface_tolerance_mm=1e-10,
                                                    max_rk_steps_per_surface=100000))
        code, y1, _, _ = oracle.propagate_free(st, y0, cylinder_r=600.0)
        assert code == 0
        pos, dirn = _dop853(bfun, r0, d0, qop, y1[3] * beta)
        errs.append(max(np.max(np.abs(pos - y1[:3])), 1e3 * np.max(np.abs(dirn - y1[4:7]))))
    # the interpolant is only C0, so the order drops at every cell face: measured 2.5e-4 / 1.5e-5 mm
    assert 5.0 * errs[1] < errs[0] < 1e-3 and errs[1] < 5e-5, errs


# ------------------------------------------------------------------ V5: path-length factor
@pytest.mark.parametrize("phi_off,theta", [(0.0, math.pi / 2), (0.5, 1.0), (-0.9, 2.3)])
def test_material_path_factor(detector, phi_off, theta):
    det = detector
    st = oracle.Setup(det, synth.uniform_field(), CKFSettings())
    m = int(det.module_offset[5] + 7 * det.n_z[5] + 3)
    n = np.cross(det.axis_u[m], det.axis_v[m])
    phi = math.atan2(n[1], n[0]) + phi_off
    x = np.array([1.0, -2.0, phi, theta, 1.0 / 1.7, 0.0])
    d = np.array([math.sin(theta) * math.cos(phi), math.sin(theta) * math.sin(phi), math.cos(theta)])
    cosi = abs(float(np.dot(d, n)))
    assert abs(cosi - math.sin(theta) * math.cos(phi_off)) < 1e-12      # the geometry of this test, by hand
    Q = oracle.add_material(st, m, x, np.zeros((6, 6)))
    th0 = oracle.highland_theta0(1.7, det.x_over_x0[m] / cosi, M_MUON)   # effective thickness x/X0 / |d.n|
    assert abs(Q[3, 3] - th0 ** 2) < 1e-15 * max(1.0, th0 ** 2) + 1e-22
    assert abs(Q[2, 2] - th0 ** 2 / math.sin(theta) ** 2) < 1e-12 * Q[2, 2]
    if phi_off != 0.0 or theta != math.pi / 2:
        # an inclined track sees MORE material than at normal incidence: 1/cosi, not cosi and not 1
        th_normal = oracle.highland_theta0(1.7, det.x_over_x0[m], M_MUON)
        assert Q[3, 3] > th_normal ** 2 * 1.05


# ------------------------------------------------------------------ R10: literal greedy
def _toy(n_particles=6, n_layers=4):
    from tests.test_oracle_ckf import _toy as toy
    return toy(n_particles=n_particles, n_layers=n_layers)


def _greedy_ckf(st, ckf, off, loc, var, seed_module, seed_params, seed_cov):
    """Level-synchronous CKF from the oracle's primitives with R10 as a LITERAL greedy: every tip that wants children
    gets one; further children are then handed out one at a time, walking the tips in order and each tip's ranked
    passers in order, for as long as the seed holds fewer than `cap` leaves (finished + live branches)."""
    out = []
    for s in range(len(seed_module)):
        tips = [dict(x=seed_params[s].astype(np.float64), C=seed_cov[s].reshape(6, 6).astype(np.float64),
                     module=int(seed_module[s]), meas=[], holes=0)]
        finished, level = 0, 0
        while tips:
            if level >= ckf.max_levels:
                break
            stage = []
            for t in tips:
                if level == 0:
                    code, tg, xp, Cp = 0, t["module"], t["x"], t["C"]
                else:
                    code, tg, xp, Cp, _ = oracle.move(st, t["module"], t["x"], t["C"])
                if code != 0:
                    stage.append(("stop", t))
                    continue
                passers = sorted((oracle.predicted_chi2(xp, Cp, loc[i], var[i]), i) for i in range(off[tg], off[tg + 1]))
                passers = [pi for pi in passers if pi[0] < ckf.chi2_max][:ckf.max_branches_per_surface]
                if not passers and t["holes"] + 1 > ckf.max_holes:
                    stage.append(("stop", t))
                else:
                    stage.append(("go", t, tg, xp, Cp, passers))
            leaves = finished + len(tips)
            grant = [1 if e[0] == "go" else 0 for e in stage]
            for k, e in enumerate(stage):                      # one extra child at a time, tip order
                if e[0] != "go":
                    continue
                for _ in range(max(len(e[5]), 1) - 1):
                    if leaves >= ckf.max_candidates_per_seed:
                        break
                    grant[k] += 1
                    leaves += 1
            nxt = []
            for k, e in enumerate(stage):
                if e[0] == "stop":
                    finished += 1
                    if len(e[1]["meas"]) >= ckf.min_measurements:
                        out.append((s, tuple(e[1]["meas"])))
                    continue
                _, t, tg, xp, Cp, passers = e
                if not passers:
                    nxt.append(dict(x=xp, C=Cp, module=tg, meas=t["meas"], holes=t["holes"] + 1))
                for c2, i in passers[:grant[k]]:
                    xu, Cu = oracle.kalman_update(xp, Cp, loc[i], var[i])
                    nxt.append(dict(x=xu, C=Cu, module=tg, meas=t["meas"] + [i], holes=t["holes"]))
            tips = nxt
            level += 1
    return out


@pytest.mark.parametrize("max_holes", [3, 0])
@pytest.mark.parametrize("cap", [1, 2, 3, 7, 50])
def test_r10_equals_literal_greedy(cap, max_holes):
    """max_holes = 0 makes branches finish at different levels (a branch without a passer stops at once), so the
    leaves of a seed are finished + live ones while the cap binds."""
    det, ev, off, loc, var = _toy(n_particles=8, n_layers=6)
    ckf = CKFSettings(max_branches_per_surface=1000, max_candidates_per_seed=cap, min_measurements=1, max_holes=max_holes)
    st = oracle.Setup(det, synth.uniform_field(), ckf)
    tr = oracle.ckf_find(st, off, loc, var, ev.seed_module, ev.seed_params, ev.seed_cov)
    got = sorted((int(tr.seed_id[t]), tuple(int(i) for i in tr.meas_list(t))) for t in range(tr.n_tracks))
    want = sorted(_greedy_ckf(st, ckf, off, loc, var, ev.seed_module, ev.seed_params, ev.seed_cov))
    assert got == want                                           # which children survive, not only how many
    big = CKFSettings(max_branches_per_surface=1000, max_candidates_per_seed=1000000, min_measurements=1, max_holes=max_holes)
    full = oracle.ckf_find(oracle.Setup(det, synth.uniform_field(), big), off, loc, var, ev.seed_module,
                           ev.seed_params, ev.seed_cov)
    # leaves per seed = min(cap, uncapped) whenever every leaf emits (min_measurements = 1 and a hit at level 0)
    unc = np.bincount(full.seed_id, minlength=ev.n_seeds)
    cnt = np.bincount(tr.seed_id, minlength=ev.n_seeds)
    assert unc.max() > 7                                         # the toy really exceeds the small caps
    assert np.array_equal(cnt, np.minimum(unc, cap))


# ------------------------------------------------------------------ D11 against the literal SURVEY N3 walk
def test_d11_early_exit_changes_no_candidate():
    """Reading D11 (a tip beyond every further half-length, moving away in z, stops EXIT at once) against the literal
    N3 walk over the remaining portal cylinders: identical candidates, parameters and chi2; only the stop reason of
    walks that would have ended NOT_OUTGOING (or STEP_LIMIT) may differ, and trial counters shrink."""
    det, fld, cfg = synth.config_bundle(1)
    ev = synth.make_event(1, det=det, n_particles=600)
    st = oracle.Setup(det, fld, cfg.ckf)
    try:
        oracle.set_n3_literal_walk(True)
        lit = oracle.find_event(st, ev, n_threads=4)
    finally:
        oracle.set_n3_literal_walk(False)
    d11 = oracle.find_event(st, ev, n_threads=4)
    assert lit.n_tracks == d11.n_tracks > 600
    for name in ("track_offsets", "meas_idx", "seed_id", "n_holes", "last_module"):
        assert np.array_equal(getattr(lit, name), getattr(d11, name)), name
    for name in ("params", "cov", "chi2_sum", "entry_chi2"):
        assert np.array_equal(getattr(lit, name), getattr(d11, name)), name
    diff = lit.stop_reason != d11.stop_reason
    # where they differ, D11 says EXIT and the literal walk ran out of barrel some other way
    assert np.all(d11.stop_reason[diff] == 1)
    assert set(np.unique(lit.stop_reason[diff]).tolist()) <= {3, 4}
    assert d11.counters["rk_trials"] <= lit.counters["rk_trials"]
    assert d11.counters["visits"] == lit.counters["visits"] and d11.counters["updates"] == lit.counters["updates"]


# ------------------------------------------------------------------ J2': field-gradient terms of the transport Jacobian
def _fd_jacobian(st, m_from, m_to, x0):
    steps = np.array([1e-3, 1e-3, 1e-6, 1e-6, 1e-6 * abs(x0[4]), 1e-3])
    Jfd = np.zeros((6, 6))
    for k in range(6):
        xa, xb = x0.copy(), x0.copy()
        xa[k] += steps[k]
        xb[k] -= steps[k]
        ca, pa, _ = oracle.bound_to_bound(st, m_from, m_to, xa)
        cb, pb, _ = oracle.bound_to_bound(st, m_from, m_to, xb)
        assert ca == 0 and cb == 0
        Jfd[:, k] = (pa - pb) / (2 * steps[k])
    return Jfd


@pytest.mark.parametrize("qop,layers", [(1.0 / 0.7, (4, 5)), (-1.0 / 1.5, (6, 7)), (1.0 / 0.6, (7, 8))])
def test_jacobian_with_field_gradient_vs_finite_differences(detector, qop, layers):
    """In the analytic NON-uniform field the Jacobian with the gradient terms (config.field_gradient = 1, reading A13)
    equals central finite differences of the bound->bound map to 1e-5; without them it is off at the 1e-3..1e-2 level
    (SURVEY.md pin table J1-J5).  This also pins which field value each stage of J2 uses: B1 = B2 = B4 only in a uniform
    field."""
    det = detector
    l0, l1 = layers
    m_from = int(det.module_offset[l0] + 0 * det.n_z[l0] + int(det.n_z[l0] * 0.8))     # z ~ +600 mm: dB/dz is large there
    m_to = int(det.module_offset[l1] + 0 * det.n_z[l1] + int(det.n_z[l1] * 0.8))
    x0 = np.array([2.0, 10.0, 0.03, 1.45, qop, 3.0])
    kw = dict(rk_tolerance_mm=1e-9, surface_tolerance_mm=1e-11, max_rk_steps_per_surface=100000)
    on = oracle.Setup(det, _analytic_field_spec(), CKFSettings(field_gradient=1, **kw))
    off = oracle.Setup(det, _analytic_field_spec(), CKFSettings(field_gradient=0, **kw))
    code, xp, J_on = oracle.bound_to_bound(on, m_from, m_to, x0)
    code2, xp2, J_off = oracle.bound_to_bound(off, m_from, m_to, x0)
    assert code == 0 and code2 == 0 and np.array_equal(xp, xp2)        # the flag never touches the state
    Jfd = _fd_jacobian(on, m_from, m_to, x0)
    scale = np.maximum(np.abs(Jfd), np.max(np.abs(Jfd), axis=1, keepdims=True) * 1e-3 + 1e-12)
    err_on = np.max(np.abs(J_on - Jfd) / scale)
    err_off = np.max(np.abs(J_off - Jfd) / scale)
    assert err_on < 1e-5, err_on
    assert err_off > 30 * err_on and err_off > 2e-4, (err_on, err_off)


def test_field_gradient_flag_is_neutral_in_a_uniform_field(detector):
    """G = 0: the tangent form of J2' must reproduce the matrix form of J2 (rounding apart), on every element."""
    det = detector
    m_from = int(det.module_offset[4] + det.n_z[4] // 2)
    m_to = int(det.module_offset[5] + det.n_z[5] // 2)
    x0 = np.array([2.0, 10.0, 0.05, 1.35, -1.0 / 0.8, 3.0])
    Js = []
    for flag in (0, 1):
        st = oracle.Setup(det, synth.uniform_field(), CKFSettings(field_gradient=flag))
        code, xp, J = oracle.bound_to_bound(st, m_from, m_to, x0)
        assert code == 0
        Js.append(J)
    assert np.allclose(Js[0], Js[1], rtol=1e-12, atol=1e-13)


def test_grid_field_gradient_is_the_derivative_of_the_interpolant(detector):
    """With the flag on in the float32 GRID field the Jacobian matches finite differences of the map through the same
    trilinear interpolant, as long as no stage point changes its cell under the perturbation (one short move)."""
    det = detector
    m_from = int(det.module_offset[2] + 0 * det.n_z[2] + int(det.n_z[2] * 0.7))
    m_to = int(det.module_offset[3] + 0 * det.n_z[3] + int(det.n_z[3] * 0.7))
    x0 = np.array([1.0, 3.0, 0.02, 1.5, 1.0 / 0.9, 0.0])
    kw = dict(rk_tolerance_mm=1e-9, surface_tolerance_mm=1e-11, max_rk_steps_per_surface=100000)
    on = oracle.Setup(det, synth.grid_field(), CKFSettings(field_gradient=1, **kw))
    code, xp, J = oracle.bound_to_bound(on, m_from, m_to, x0)
    assert code == 0
    Jfd = _fd_jacobian(on, m_from, m_to, x0)
    scale = np.maximum(np.abs(Jfd), np.max(np.abs(Jfd), axis=1, keepdims=True) * 1e-3 + 1e-12)
    assert np.max(np.abs(J - Jfd) / scale) < 5e-5


def test_matrix_form_of_j2_equals_tangent_form_without_gradient_in_a_nonuniform_field(detector):
    """The default Jacobian (J2, matrix form, gradient neglected) against the tangent form with G forced to zero (pin
    hook field_gradient = 2) where B1 != B2 != B4: pins which field value each stage of the DEFAULT path uses through
    the tangent form, which finite differences pin with the gradient on."""
    det = detector
    kw = dict(rk_tolerance_mm=1e-6, surface_tolerance_mm=1e-8)
    for l0, qop in ((4, 1.0 / 0.7), (7, -1.0 / 0.6)):
        m_from = int(det.module_offset[l0] + int(det.n_z[l0] * 0.8))
        m_to = int(det.module_offset[l0 + 1] + int(det.n_z[l0 + 1] * 0.8))
        x0 = np.array([2.0, 10.0, 0.03, 1.45, qop, 3.0])
        Js = []
        for flag in (0, 2):
            st = oracle.Setup(det, _analytic_field_spec(), CKFSettings(field_gradient=flag, **kw))
            code, _, J = oracle.bound_to_bound(st, m_from, m_to, x0)
            assert code == 0
            Js.append(J)
        scale = np.maximum(np.abs(Js[1]), np.max(np.abs(Js[1]), axis=1, keepdims=True) * 1e-6 + 1e-14)
        assert np.max(np.abs(Js[0] - Js[1]) / scale) < 1e-9
