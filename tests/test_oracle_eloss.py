"""Pins of the oracle's mean energy loss (rule E, PAPER.md:55 muon hypothesis)."""
import copy
import math

import numpy as np
import pytest

import oracle
import synth
from synth.events import CKFSettings, M_MUON

ME = 0.51099895e-3


def test_bethe_minimum_against_the_pdg_table():
    dedx_min, z_over_a, i_ev, x0 = np.loadtxt("tests/golden/bethe_silicon.txt", comments="#")
    ps = np.exp(np.linspace(math.log(0.05), math.log(50.0), 400))
    v = np.array([oracle.bethe_dedx(p, M_MUON) for p in ps]) * 1e3          # MeV cm^2 / g
    k = int(np.argmin(v))
    assert 3.0 < ps[k] / M_MUON < 4.0                                       # minimum ionisation at beta gamma ~ 3.5
    assert dedx_min <= v[k] <= 1.04 * dedx_min                              # no density correction: a little above


def test_bethe_nonrelativistic_limit():
    """beta << 1: gamma ~ 1, Wmax ~ 2 me beta^2, the bracket reduces to ln(2 me beta^2 / I) (textbook Bethe-Bloch)."""
    K, z_over_a, I = 0.307075e-3, 0.49848, 173.0e-9
    for beta in (0.02, 0.05):
        p = M_MUON * beta / math.sqrt(1 - beta * beta)
        nr = K * z_over_a / beta ** 2 * math.log(2 * ME * beta ** 2 / I)
        assert abs(oracle.bethe_dedx(p, M_MUON) / nr - 1.0) < 3.0 * beta ** 2 + 2 * ME / M_MUON


def test_energy_is_conserved_and_loss_scales_with_the_path(detector):
    det = detector
    st = oracle.Setup(det, synth.uniform_field(), CKFSettings(energy_loss=1))
    m = int(det.module_offset[4] + 3 * det.n_z[4] + 5)
    n = np.cross(det.axis_u[m], det.axis_v[m])
    phin = math.atan2(n[1], n[0])
    p = 0.8
    E = math.hypot(p, M_MUON)
    losses = []
    for dphi, theta in ((0.0, math.pi / 2), (0.6, 1.1)):
        x = np.array([0.0, 0.0, phin + dphi, theta, -1.0 / p, 0.0])
        dE, xo, g = oracle.energy_loss(st, m, x)
        cosi = math.sin(theta) * math.cos(dphi)
        losses.append(dE * cosi)
        p2 = 1.0 / abs(xo[4])
        assert xo[4] < 0 and np.array_equal(xo[[0, 1, 2, 3, 5]], x[[0, 1, 2, 3, 5]])
        assert abs(math.hypot(p2, M_MUON) - (E - dE)) < 1e-15 * E         # E' = E - dE
        # 0.15 mm of silicon costs a minimum-ionising muon ~ 0.06 MeV at normal incidence
        assert 0.04e-3 < dE * cosi < 0.09e-3
        # g = d(q/p)'/d(q/p) with dE frozen: finite differences of the plain kinematics, written here
        def qop_after(qop):
            pp = 1.0 / abs(qop)
            e2 = math.hypot(pp, M_MUON) - dE
            return math.copysign(1.0 / math.sqrt(e2 * e2 - M_MUON ** 2), qop)
        h = 1e-6 * abs(x[4])
        fd = (qop_after(x[4] + h) - qop_after(x[4] - h)) / (2 * h)
        assert abs(g / fd - 1.0) < 1e-7
    assert abs(losses[0] / losses[1] - 1.0) < 1e-12                        # dE * |d.n| does not depend on the incidence
    # switched off (BASELINE configs) nothing changes
    st0 = oracle.Setup(det, synth.uniform_field(), CKFSettings())
    dE, xo, g = oracle.energy_loss(st0, m, x)
    assert dE == 0.0 and g == 1.0 and np.array_equal(xo, x)
    # a particle that would stop in the module: q/p not finite -> the move ends NUMERIC
    slow = np.array([0.0, 0.0, phin, math.pi / 2, 1.0 / 0.002, 0.0])
    dE, xo, g = oracle.energy_loss(st, m, slow)
    assert not np.isfinite(xo[4])
    code, *_ = oracle.move(st, m, slow, np.eye(6) * 1e-6)
    assert oracle.STOP_NAMES[code] == "NUMERIC"


def test_move_with_energy_loss_jacobian_and_covariance(detector):
    """Where rule E sits in the chain: the arrival q/p is the q/p after the loss; d(arrival)/d(start) = J J_E by finite
    differences of the whole move; the transported covariance is J_total (C + Q) J_total^T."""
    det = detector
    ckf = CKFSettings(energy_loss=1, rk_tolerance_mm=1e-8, surface_tolerance_mm=1e-10)
    st = oracle.Setup(det, synth.uniform_field(), ckf)
    m = int(det.module_offset[4] + 0 * det.n_z[4] + det.n_z[4] // 2)
    x0 = np.array([2.0, 10.0, 0.05, 1.35, 1.0 / 0.6, 3.0])
    Cm = np.diag([1e-2, 1e-2, 1e-6, 1e-6, 1e-4, 1.0])
    code, tg, xp, Cp, J = oracle.move(st, m, x0, Cm)
    assert code == 0
    dE, xo, g = oracle.energy_loss(st, m, x0)
    assert xp[4] == xo[4] and abs(xo[4]) > abs(x0[4])                      # slower after the module
    steps = np.array([1e-3, 1e-3, 1e-6, 1e-6, 1e-6 * abs(x0[4]), 1e-3])
    Jfd = np.zeros((6, 6))
    for k in range(6):
        xa, xb = x0.copy(), x0.copy()
        xa[k] += steps[k]
        xb[k] -= steps[k]
        ca, tga, pa, _, _ = oracle.move(st, m, xa, Cm)
        cb, tgb, pb, _, _ = oracle.move(st, m, xb, Cm)
        assert ca == 0 and cb == 0 and tga == tg and tgb == tg
        Jfd[:, k] = (pa - pb) / (2 * steps[k])
    scale = np.maximum(np.abs(Jfd), np.max(np.abs(Jfd), axis=1, keepdims=True) * 1e-3 + 1e-12)
    rel = np.abs(J - Jfd) / scale
    # J_E treats dE as a constant (reading): its neglected dependence on the incidence angle shows in the phi / theta
    # columns at 1e-4, its dependence on p in the q/p column at 1e-5; g - 1 itself is 2e-4 here, so the q/p column
    # still pins that J_E is applied (and where)
    rows = [0, 1, 2, 3, 5]
    assert rel[:, [0, 1, 5]].max() < 1e-6 and rel[:, 4].max() < 3e-5 and rel[np.ix_(rows, [2, 3])].max() < 3e-4, rel
    assert np.all(J[4, [2, 3]] == 0.0) and np.abs(Jfd[4, [2, 3]]).max() < 1e-4   # d(q/p)'/d(angles) through dE: neglected
    assert abs(J[4, 4] - g) < 1e-12 and g - 1.0 > 1.5e-4
    assert np.max(np.abs(J[:, 4] / g - Jfd[:, 4]) / scale[:, 4]) > 1e-4    # without J_E the q/p column would be off
    Q = oracle.add_material(st, m, x0, np.zeros((6, 6)))
    want = J @ (Cm + Q) @ J.T
    assert np.allclose(Cp, want, rtol=1e-10, atol=1e-16)
    # and with the switch off the same move has J[4][4] = 1
    st0 = oracle.Setup(det, synth.uniform_field(), CKFSettings(rk_tolerance_mm=1e-8, surface_tolerance_mm=1e-10))
    _, _, xp0, _, J0 = oracle.move(st0, m, x0, Cm)
    assert xp0[4] == x0[4] and J0[4, 4] == 1.0
