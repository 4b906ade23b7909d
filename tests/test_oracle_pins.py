"""Pins of the CPU oracle against what the paper's cited mathematics fixes (SURVEY.md §8(c) pin table).

None of these re-types an oracle formula: each compares the oracle with a closed form, an invariant,
a finite difference, a textbook special case or a brute-force search.
"""
import math

import numpy as np
import pytest

import oracle
import synth
from synth.events import CKFSettings, KAPPA, M_MUON

pytestmark = pytest.mark.filterwarnings("ignore")


def _setup(det, inhom=False, **kw):
    fld = synth.grid_field() if inhom else synth.uniform_field()
    kw.setdefault("max_rk_steps_per_surface", 100000)
    return oracle.Setup(det, fld, CKFSettings(**kw))


def _helix(r0, d0, qop, bz, s):
    """Closed-form helix in uniform (0,0,bz): position and direction after arc length s."""
    lam = KAPPA * qop * bz            # d' = lam_b * d x z
    dx, dy, dz = d0
    # d x z = (dy, -dx, 0)  =>  (dx + i dy)' = -i lam (dx + i dy)
    w = complex(dx, dy)
    ws = w * np.exp(-1j * lam * s)
    pos_xy = complex(r0[0], r0[1]) + w * (np.exp(-1j * lam * s) - 1.0) / (-1j * lam)
    return np.array([pos_xy.real, pos_xy.imag, r0[2] + dz * s]), np.array([ws.real, ws.imag, dz])


# ------------------------------------------------------------------ P2-P5: stepping vs the analytic helix
@pytest.mark.parametrize("pt,q", [(0.5, 1.0), (1.0, -1.0), (10.0, 1.0)])
def test_helix_closed_form(detector, pt, q):
    st = _setup(detector, rk_tolerance_mm=1e-6, surface_tolerance_mm=1e-9)
    theta = 1.1
    p = pt / math.sin(theta)
    d0 = np.array([math.sin(theta) * math.cos(0.3), math.sin(theta) * math.sin(0.3), math.cos(theta)])
    r0 = np.array([5.0, -3.0, 12.0])
    y = np.concatenate([r0, [0.0], d0, [q / p]])
    R = 1020.0
    code, y1, D, nsteps = oracle.propagate_free(st, y, cylinder_r=R)
    assert code == 0
    assert abs(math.hypot(y1[0], y1[1]) - R) < 1e-9           # landed on the cylinder (P5)
    assert abs(np.linalg.norm(y1[4:7]) - 1.0) < 1e-14         # |d| = 1 (P2 invariant)
    # arc length from the time coordinate: t = s / beta
    beta = p / math.sqrt(p * p + M_MUON ** 2)
    s = y1[3] * beta
    pos, dirn = _helix(r0, d0, q / p, 2.0, s)
    assert np.max(np.abs(pos - y1[:3])) / 1500.0 < 1e-9       # north_star: 1e-9 relative
    assert np.max(np.abs(dirn - y1[4:7])) < 1e-9


def test_helix_error_scales_with_tolerance(detector):
    errs = []
    for tol in (1e-3, 1e-5, 1e-7):
        st = _setup(detector, rk_tolerance_mm=tol, surface_tolerance_mm=1e-9)
        th = 1.3
        p = 0.5 / math.sin(th)
        d0 = np.array([math.sin(th), 0.0, math.cos(th)])
        r0 = np.array([1.0, 0.5, 0.0])
        y = np.concatenate([r0, [0.0], d0, [1.0 / p]])
        code, y1, _, _ = oracle.propagate_free(st, y, cylinder_r=1000.0)
        assert code == 0
        beta = p / math.sqrt(p * p + M_MUON ** 2)
        pos, _ = _helix(r0, d0, 1.0 / p, 2.0, y1[3] * beta)
        errs.append(np.max(np.abs(pos - y1[:3])))
    assert errs[0] > errs[1] > errs[2]
    assert errs[2] < 1e-7


def test_forward_backward_returns(detector):
    st = _setup(detector, rk_tolerance_mm=1e-7, surface_tolerance_mm=1e-10)
    th = 0.9
    d0 = np.array([math.sin(th) * math.cos(1.0), math.sin(th) * math.sin(1.0), math.cos(th)])
    y0 = np.concatenate([[30.0, 10.0, -4.0, 0.0], d0, [-0.7]])
    n = np.array([math.cos(1.0), math.sin(1.0), 0.0])
    _, y1, _, _ = oracle.propagate_free(st, y0, plane=(400.0 * n, n))
    c0 = y0[:3]
    _, y2, _, _ = oracle.propagate_free(st, y1, plane=(c0, d0))   # back to the plane through r0 normal to d0
    assert np.max(np.abs(y2[:3] - y0[:3])) < 1e-7
    assert np.max(np.abs(y2[4:7] - y0[4:7])) < 1e-9
    assert abs(y2[3]) < 1e-7


def test_plane_landing_matches_bisection_on_helix(detector):
    st = _setup(detector, rk_tolerance_mm=1e-7, surface_tolerance_mm=1e-10)
    th = 1.2
    p = 0.8
    d0 = np.array([math.sin(th) * math.cos(0.2), math.sin(th) * math.sin(0.2), math.cos(th)])
    r0 = np.array([20.0, 5.0, 1.0])
    n = np.array([math.cos(0.35), math.sin(0.35), 0.0])
    c = 500.0 * n
    y = np.concatenate([r0, [0.0], d0, [1.0 / p]])
    code, y1, _, _ = oracle.propagate_free(st, y, plane=(c, n))
    assert code == 0
    f = lambda s: float(np.dot(_helix(r0, d0, 1.0 / p, 2.0, s)[0] - c, n))
    lo, hi = 0.0, 1000.0
    assert f(lo) < 0 < f(hi)
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if f(mid) < 0:
            lo = mid
        else:
            hi = mid
    pos, _ = _helix(r0, d0, 1.0 / p, 2.0, 0.5 * (lo + hi))
    assert np.max(np.abs(pos - y1[:3])) < 1e-6


def test_cylinder_not_outgoing(detector):
    st = _setup(detector)
    y = np.array([100.0, 0.0, 0.0, 0.0, -1.0, 0.0, 0.0, 0.5])   # moving radially inward
    code, *_ = oracle.propagate_free(st, y, cylinder_r=200.0)
    assert oracle.STOP_NAMES[code] == "NOT_OUTGOING"


# ------------------------------------------------------------------ F: trilinear field
def test_field_multilinear_components_exact(detector):
    st = _setup(detector, inhom=True)
    rng = np.random.default_rng(1)
    for _ in range(200):
        r = rng.uniform(-1050, 1050, 3)
        b = oracle.field_at(st, r)
        ana = synth.analytic_b(r[None, :], True)[0]
        # Bx = a B0 x z and By are multilinear: interpolant == analytic up to float32 rounding of the nodes
        assert abs(b[0] - ana[0]) < 1e-6 and abs(b[1] - ana[1]) < 1e-6
        # Bz quadratic in z: linear-interpolation bound |f''| h^2 / 8 with f'' = 2 a B0  ->  6e-5 T
        # (SURVEY.md quotes a B0 h^2 / 8 = 3e-5, dropping the factor 2 of the second derivative)
        assert abs(b[2] - ana[2]) <= 2.0 * 0.3e-6 * 2.0 * 20.0 ** 2 / 8.0 + 1e-6


def test_field_at_nodes_and_uniform(detector):
    st = _setup(detector, inhom=True)
    g = st.field  # noqa
    fs = synth.grid_field()
    for idx in [(0, 0, 0), (55, 55, 55), (110, 110, 110), (3, 77, 100)]:
        r = fs.origin + fs.spacing * np.array(idx)
        assert np.allclose(oracle.field_at(st, r), fs.grid[idx].astype(np.float64), atol=1e-7)
    su = _setup(detector)
    assert np.array_equal(oracle.field_at(su, [12.0, -7.0, 300.0]), [0.0, 0.0, 2.0])


# ------------------------------------------------------------------ J1-J5: Jacobian vs central finite differences
def _module_pair(det, l_from, l_to, iphi_frac=0.1):
    nphi_f, nz_f = det.n_phi[l_from], det.n_z[l_from]
    m_from = det.module_offset[l_from] + 0 * nz_f + nz_f // 2
    m_to = det.module_offset[l_to] + 0 * det.n_z[l_to] + det.n_z[l_to] // 2
    return int(m_from), int(m_to)


@pytest.mark.parametrize("qop", [1.0 / 0.8, -1.0 / 3.0])
def test_jacobian_finite_differences_uniform_field(detector, qop):
    st = _setup(detector, rk_tolerance_mm=1e-8, surface_tolerance_mm=1e-10)
    m_from, m_to = _module_pair(detector, 4, 5)
    x0 = np.array([2.0, 10.0, 0.05, 1.35, qop, 3.0])
    code, xp, J = oracle.bound_to_bound(st, m_from, m_to, x0)
    assert code == 0
    steps = np.array([1e-3, 1e-3, 1e-6, 1e-6, 1e-6 * abs(qop), 1e-3])
    Jfd = np.zeros((6, 6))
    for k in range(6):
        xa, xb = x0.copy(), x0.copy()
        xa[k] += steps[k]
        xb[k] -= steps[k]
        _, pa, _ = oracle.bound_to_bound(st, m_from, m_to, xa)
        _, pb, _ = oracle.bound_to_bound(st, m_from, m_to, xb)
        Jfd[:, k] = (pa - pb) / (2 * steps[k])
    scale = np.maximum(np.abs(Jfd), np.max(np.abs(Jfd), axis=1, keepdims=True) * 1e-3 + 1e-12)
    assert np.max(np.abs(J - Jfd) / scale) < 1e-6              # north_star: 1e-6


def test_jacobian_straight_line_limit(detector):
    """B = 0: the bound->bound map is elementary geometry; check against its closed form."""
    fld = synth.uniform_field(0.0)
    st = oracle.Setup(detector, fld, CKFSettings())
    m_from, m_to = _module_pair(detector, 2, 3)
    x0 = np.array([1.0, -4.0, 0.02, 1.2, 0.5, 0.0])
    code, xp, J = oracle.bound_to_bound(st, m_from, m_to, x0)
    assert code == 0
    det = detector
    # closed form: r = c0 + l0 u0 + l1 v0 + s d, with s fixed by the target plane
    def f(x):
        c0, u0, v0 = det.center[m_from], det.axis_u[m_from], det.axis_v[m_from]
        c1, u1, v1 = det.center[m_to], det.axis_u[m_to], det.axis_v[m_to]
        n1 = np.cross(u1, v1)
        d = np.array([math.sin(x[3]) * math.cos(x[2]), math.sin(x[3]) * math.sin(x[2]), math.cos(x[3])])
        r = c0 + x[0] * u0 + x[1] * v0
        s = np.dot(c1 - r, n1) / np.dot(d, n1)
        q = r + s * d - c1
        ib = math.sqrt(1 + (M_MUON * x[4]) ** 2)
        return np.array([np.dot(q, u1), np.dot(q, v1), x[2], x[3], x[4], x[5] + s * ib])
    assert np.allclose(xp, f(x0), atol=1e-10)
    Jfd = np.zeros((6, 6))
    for k in range(6):
        h = 1e-5
        xa, xb = x0.copy(), x0.copy()
        xa[k] += h
        xb[k] -= h
        Jfd[:, k] = (f(xa) - f(xb)) / (2 * h)
    assert np.max(np.abs(J - Jfd)) < 1e-6 * max(1.0, np.max(np.abs(Jfd)))


def test_covariance_transport_is_congruence(detector):
    rng = np.random.default_rng(3)
    J = rng.normal(size=(6, 6))
    A = rng.normal(size=(6, 6))
    Cm = A @ A.T
    out = oracle.transport_cov(J, Cm)
    assert np.allclose(out, J @ Cm @ J.T, rtol=1e-13, atol=1e-13)
    assert np.array_equal(out, out.T)


# ------------------------------------------------------------------ V1-V3: Kalman gate and update
def test_scalar_gain_closed_form():
    """One measured coordinate decoupled from the rest: gain = sp^2 / (sp^2 + sm^2) (north_star)."""
    sp2, sm2 = 0.04, 0.01
    Cm = np.diag([sp2, 1e-12, 1e-6, 1e-6, 1e-4, 1.0])
    x = np.array([1.0, 2.0, 0.1, 1.0, 0.3, 0.0])
    loc = np.array([1.3, 2.0])
    var = np.array([sm2, 1e12])                  # second coordinate carries no information
    xo, Co = oracle.kalman_update(x, Cm, loc, var)
    k = sp2 / (sp2 + sm2)
    assert abs(xo[0] - (1.0 + k * 0.3)) < 1e-12
    assert abs(Co[0, 0] - (1 - k) * sp2) < 1e-14
    chi2 = oracle.predicted_chi2(x, Cm, loc, var)
    assert abs(chi2 - 0.3 ** 2 / (sp2 + sm2)) < 1e-10


def _rand_cov(rng):
    A = rng.normal(size=(6, 6)) * np.array([0.1, 0.2, 1e-3, 1e-3, 1e-2, 1.0])[:, None]
    return A @ A.T + np.diag([1e-4, 1e-4, 1e-8, 1e-8, 1e-6, 1e-2])


def test_update_information_form_identity():
    rng = np.random.default_rng(5)
    H = np.zeros((2, 6))
    H[0, 0] = H[1, 1] = 1.0
    for _ in range(20):
        Cm = _rand_cov(rng)
        x = rng.normal(size=6)
        loc = x[:2] + rng.normal(size=2) * 0.1
        var = np.array([0.015 ** 2, 0.05 ** 2])
        xo, Co = oracle.kalman_update(x, Cm, loc, var)
        info = np.linalg.inv(Cm) + H.T @ np.diag(1 / var) @ H
        assert np.allclose(np.linalg.inv(Co), info, rtol=1e-7)
        # weighted-mean form of the state
        xw = np.linalg.solve(info, np.linalg.inv(Cm) @ x + H.T @ (loc / var))
        xw[2] = (xw[2] + np.pi) % (2 * np.pi) - np.pi
        assert np.allclose(xo, xw, rtol=1e-7, atol=1e-9)
        # predicted-residual chi2 == filtered-residual chi2 + state-pull chi2
        chi2 = oracle.predicted_chi2(x, Cm, loc, var)
        rf = loc - xo[:2]
        dx = xo - x
        chi2_f = rf @ np.diag(1 / var) @ rf + dx @ np.linalg.inv(Cm) @ dx
        assert abs(chi2 - chi2_f) < 1e-8 * max(1.0, chi2)


def test_two_sequential_updates_equal_one_batch():
    rng = np.random.default_rng(6)
    Cm = _rand_cov(rng)
    x = rng.normal(size=6) * 0.1
    la, va = np.array([0.1, -0.2]), np.array([0.01, 0.04])
    lb, vb = np.array([0.12, -0.25]), np.array([0.02, 0.03])
    x1, C1 = oracle.kalman_update(x, Cm, la, va)
    x2, C2 = oracle.kalman_update(x1, C1, lb, vb)
    # batch = one update with the precision-weighted mean of the two measurements
    vc = 1 / (1 / va + 1 / vb)
    lc = vc * (la / va + lb / vb)
    x3, C3 = oracle.kalman_update(x, Cm, lc, vc)
    assert np.allclose(x2, x3, rtol=1e-9, atol=1e-12)
    assert np.allclose(C2, C3, rtol=1e-8, atol=1e-15)


def test_phi_wrap():
    Cm = np.diag([1.0, 1.0, 1e-2, 1e-6, 1e-4, 1.0])
    Cm[0, 2] = Cm[2, 0] = 0.09
    x = np.array([0.0, 0.0, math.pi - 0.01, 1.0, 0.3, 0.0])
    xo, _ = oracle.kalman_update(x, Cm, np.array([1.0, 0.0]), np.array([1e-6, 1e-6]))
    assert -math.pi < xo[2] <= math.pi
    assert abs(xo[2] - (math.pi - 0.01 + 0.09 - 2 * math.pi)) < 1e-6


# ------------------------------------------------------------------ V5: Highland
def test_highland_values_and_order_independence(detector):
    golden = np.loadtxt("tests/golden/highland_theta0.txt", comments="#")
    for p, mrad in golden:
        assert abs(oracle.highland_theta0(p, 0.0016, M_MUON) * 1e3 - mrad) < 5e-4 * mrad
    # H Q = 0: material noise only touches (phi, theta) => adding it before or after the update is the same
    st = _setup(detector)
    rng = np.random.default_rng(7)
    Cm = _rand_cov(rng)
    x = np.array([0.3, 1.0, 0.2, 1.1, 0.5, 0.0])
    loc, var = np.array([0.31, 1.1]), np.array([2.25e-4, 2.5e-3])
    m = 100
    xa, Ca = oracle.kalman_update(x, Cm, loc, var)
    after = oracle.add_material(st, m, x, Ca)
    Q = oracle.add_material(st, m, x, np.zeros((6, 6)))
    assert np.count_nonzero(Q) == 2 and Q[2, 2] > 0 and Q[3, 3] > 0
    assert np.allclose(Q[2, 2] * math.sin(1.1) ** 2, Q[3, 3])
    assert np.allclose(after, Ca + Q)


# ------------------------------------------------------------------ N2-N5: navigation vs brute force over all modules
def test_visited_modules_equal_brute_force(detector):
    det = detector
    st = _setup(det, rk_tolerance_mm=1e-6, surface_tolerance_mm=1e-8)
    stt = _setup(det, rk_tolerance_mm=1e-8, surface_tolerance_mm=1e-10)
    ev = synth.make_event(0, det=det, n_particles=30)
    normal = np.cross(det.axis_u, det.axis_v)
    n_cmp = 0
    for s in range(ev.n_seeds):
        x = ev.seed_params[s].astype(np.float64)
        x[5] = 0.0
        m = int(ev.seed_module[s])
        Cm = np.eye(6) * 1e-6
        visited = [m]
        xm, mm = x, m
        while True:
            code, tg, xp, Cp, _ = oracle.move(st, mm, xm, Cm)
            if code != 0:
                break
            visited.append(tg)
            xm, mm = xp, tg
        # brute force: tight-tolerance trajectory to every module plane with a crude pre-filter, test rectangle
        c0 = det.center[m] + x[0] * det.axis_u[m] + x[1] * det.axis_v[m]
        d0 = np.array([math.sin(x[3]) * math.cos(x[2]), math.sin(x[3]) * math.sin(x[2]), math.cos(x[3])])
        y0 = np.concatenate([c0, [0.0], d0, [x[4]]])
        crossed = []
        near_edge = False
        # candidate modules: those whose centre is within 60 mm of the straight-ish path in phi/z (cheap prefilter)
        for k in range(det.n_modules):
            ck = det.center[k]
            # quick reject by azimuth of centre vs azimuth of track (tracks are stiff: pT >= 1 GeV)
            dphi = (math.atan2(ck[1], ck[0]) - x[2] + math.pi) % (2 * math.pi) - math.pi
            if abs(dphi) > 0.9:
                continue
            rk = math.hypot(ck[0], ck[1])
            zexp = c0[2] + (rk - 32.0) / math.tan(x[3])
            if abs(ck[2] - zexp) > 120.0:
                continue
            code, y1, _, _ = oracle.propagate_free(stt, y0, plane=(ck, normal[k]))
            if code != 0 or y1[3] < -1e-9:
                continue
            q = y1[:3] - ck
            lu, lv = np.dot(q, det.axis_u[k]), np.dot(q, det.axis_v[k])
            mu, mv = det.half_u[k] - abs(lu), det.half_v[k] - abs(lv)
            if mu >= 0 and mv >= 0:
                crossed.append((y1[3], k))
            if min(abs(mu), abs(mv)) < 0.02 and max(-mu, -mv) < 0.02:
                near_edge = True
        crossed = [k for _, k in sorted(crossed)]
        if near_edge:
            continue          # in-bounds is decided on the straight line from the portal (N2/N4): edge cases excepted
        n_cmp += 1
        assert visited == crossed, (s, visited, crossed)
    assert n_cmp >= 20
