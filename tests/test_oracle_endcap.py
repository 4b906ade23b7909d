"""Pins of the oracle's navigation with endcap discs (row f3; PAPER.md:55 "barrel + endcaps", :76 the transition region):
the visited-module sequence against a brute-force search over ALL modules, barrel and discs, for |eta| up to 3."""
import math

import numpy as np
import pytest

import oracle
import synth
from synth.events import CKFSettings

DISC_Z = (560.0, 640.0, 740.0, 860.0, 1000.0)


@pytest.fixture(scope="module")
def endcap_detector():
    return synth.build_detector(half_z=500.0, disc_z=DISC_Z)


def _crossings(det, stt, y0, x_phi, theta, z0, skip_near_edge=0.02):
    """Brute force: tight-tolerance trajectory to every module plane (crude pre-filter), keep those hit inside the
    rectangle, order by path length.  Returns (list of module ids, near_edge flag)."""
    normal = np.cross(det.axis_u, det.axis_v)
    layer = det.module_layer
    crossed, near_edge = [], False
    tan_t = math.tan(theta)
    for k in range(det.n_modules):
        ck = det.center[k]
        dphi = (math.atan2(ck[1], ck[0]) - x_phi + math.pi) % (2 * math.pi) - math.pi
        if abs(dphi) > 0.9:
            continue
        rk = math.hypot(ck[0], ck[1])
        if det.layer_kind[layer[k]] == 0:
            if abs(ck[2] - (z0 + rk / tan_t)) > 120.0:
                continue
        else:
            if (ck[2] > 0) != (math.cos(theta) > 0) or abs(rk - (ck[2] - z0) * tan_t) > 130.0:
                continue
        code, y1, _, _ = oracle.propagate_free(stt, y0, plane=(ck, normal[k]))
        if code != 0 or y1[3] < -1e-9:
            continue
        q = y1[:3] - ck
        mu = det.half_u[k] - abs(np.dot(q, det.axis_u[k]))
        mv = det.half_v[k] - abs(np.dot(q, det.axis_v[k]))
        if mu >= 0 and mv >= 0:
            crossed.append((y1[3], k))
        if min(abs(mu), abs(mv)) < skip_near_edge and max(-mu, -mv) < skip_near_edge:
            near_edge = True
    crossed.sort()
    # modules of one disc are coplanar and overlap in phi: the same crossing point lies on two of them; the navigator
    # visits one (nearest first, tie -> lower id), so the brute-force list keeps the lower id of such a pair
    out = []
    for t, k in crossed:
        if out and det.layer_kind[layer[k]] == 1 and layer[out[-1][1]] == layer[k] and abs(out[-1][0] - t) < 1e-6:
            if k < out[-1][1]:
                out[-1] = (t, k)
            continue
        out.append((t, k))
    return [k for _, k in out], near_edge


def test_visited_modules_equal_brute_force_with_discs(endcap_detector):
    det = endcap_detector
    st = oracle.Setup(det, synth.uniform_field(), CKFSettings(rk_tolerance_mm=1e-6, surface_tolerance_mm=1e-8,
                                                              max_rk_steps_per_surface=100000))
    stt = oracle.Setup(det, synth.uniform_field(), CKFSettings(rk_tolerance_mm=1e-8, surface_tolerance_mm=1e-10,
                                                               max_rk_steps_per_surface=100000))
    rng = np.random.default_rng(42)
    n_cmp = n_disc_visits = n_transition = 0
    for trial in range(46):
        eta = rng.uniform(-3.0, 3.0)
        theta = 2.0 * math.atan(math.exp(-eta))
        phi = rng.uniform(-math.pi, math.pi)
        pt = math.exp(rng.uniform(math.log(1.0), math.log(20.0)))
        q = 1.0 if rng.random() < 0.5 else -1.0
        z0 = rng.normal(0.0, 30.0)
        d0 = np.array([math.sin(theta) * math.cos(phi), math.sin(theta) * math.sin(phi), math.cos(theta)])
        y0 = np.concatenate([[0.0, 0.0, z0, 0.0], d0, [q / (pt * math.cosh(eta))]])
        want, near_edge = _crossings(det, stt, y0, phi, theta, z0)
        if near_edge or not want:
            continue
        # start the oracle on the first crossed module with the exact bound state there
        m = want[0]
        nrm = np.cross(det.axis_u[m], det.axis_v[m])
        code, y1, _, _ = oracle.propagate_free(stt, y0, plane=(det.center[m], nrm))
        assert code == 0
        rel = y1[:3] - det.center[m]
        x = np.array([np.dot(rel, det.axis_u[m]), np.dot(rel, det.axis_v[m]), math.atan2(y1[5], y1[4]),
                      math.atan2(math.hypot(y1[4], y1[5]), y1[6]), y1[7], 0.0])
        visited, mm, xm = [m], m, x
        while True:
            code, tg, xp, Cp, _ = oracle.move(st, mm, xm, np.eye(6) * 1e-6)
            if code != 0:
                assert oracle.STOP_NAMES[code] == "EXIT"
                break
            visited.append(tg)
            xm, mm = xp, tg
        assert visited == want, (trial, eta, visited, want)
        n_cmp += 1
        kinds = det.layer_kind[det.module_layer[np.array(want)]]
        n_disc_visits += int(kinds.sum())
        n_transition += int(kinds.min() == 0 and kinds.max() == 1)
    assert n_cmp >= 30 and n_disc_visits >= 40 and n_transition >= 8      # barrel-only, disc-rich and transition tracks


def test_barrel_only_detector_is_unchanged_by_the_portal_rule(detector):
    """With no disc layer the portal rule is SURVEY's N3 + D11: the sequence of a config-0 seed is what the brute force
    over the barrel gives (the round-1 pin), and an endcap detector whose discs no track reaches gives the same moves."""
    det = detector
    far = synth.build_detector(disc_z=(5000.0,))          # discs far beyond every track's exit point
    ev = synth.make_event(0, det=det, n_particles=20)
    sa = oracle.Setup(det, synth.uniform_field(), CKFSettings())
    sb = oracle.Setup(far, synth.uniform_field(), CKFSettings())
    for s in range(ev.n_seeds):
        xm, mm = ev.seed_params[s].astype(np.float64), int(ev.seed_module[s])
        xb, mb = xm.copy(), mm
        for _ in range(14):
            ca, ta, xa, Ca, _ = oracle.move(sa, mm, xm, np.eye(6) * 1e-6)
            cb, tb, xb2, Cb, _ = oracle.move(sb, mb, xb, np.eye(6) * 1e-6)
            if ca != 0:
                assert oracle.STOP_NAMES[ca] == "EXIT"
                # with a disc still ahead the tip walks on to it and leaves through its acceptance or past the last disc
                assert cb != 0 or far.layer_kind[far.module_layer[tb]] == 1
                break
            assert cb == 0 and ta == tb and np.array_equal(xa, xb2) and np.array_equal(Ca, Cb)
            xm, mm, xb, mb = xa, ta, xb2, tb


def _crossings_any_direction(det, stt, y0, start_module, margin=150.0):
    """Brute force for tips that may cross modules against their normal: every module whose centre lies within `margin`
    of the straight line ahead is tried with the tight-tolerance trajectory."""
    normal = np.cross(det.axis_u, det.axis_v)
    r0, d0 = y0[:3], y0[4:7]
    rel = det.center - r0
    along = rel @ d0
    perp = np.linalg.norm(rel - along[:, None] * d0, axis=1)
    crossed, near_edge = [], False
    for k in np.flatnonzero((along > -50.0) & (perp < margin)):
        if k == start_module:
            continue
        code, y1, _, _ = oracle.propagate_free(stt, y0, plane=(det.center[k], normal[k]))
        if code != 0 or y1[3] < 1e-6:
            continue
        q = y1[:3] - det.center[k]
        mu = det.half_u[k] - abs(np.dot(q, det.axis_u[k]))
        mv = det.half_v[k] - abs(np.dot(q, det.axis_v[k]))
        if mu >= 0 and mv >= 0:
            crossed.append((y1[3], int(k)))
        if min(abs(mu), abs(mv)) < 0.02 and max(-mu, -mv) < 0.02:
            near_edge = True
    crossed.sort()
    return [k for _, k in crossed], near_edge


def test_bidirectional_navigation_equals_brute_force(detector):
    """config.bidirectional = 1 (rules N3''): tips that leave a barrel module INWARD cross the inner layers against
    their normals, pass the beam line and leave through the far side -- the visited-module sequence equals the brute
    force; with the flag off (reading A7, BASELINE configs) the same tips stop NOT_OUTGOING."""
    det = detector
    kw = dict(max_rk_steps_per_surface=100000)
    on = oracle.Setup(det, synth.uniform_field(), CKFSettings(bidirectional=1, rk_tolerance_mm=1e-6, surface_tolerance_mm=1e-8, **kw))
    off = oracle.Setup(det, synth.uniform_field(), CKFSettings(rk_tolerance_mm=1e-6, surface_tolerance_mm=1e-8, **kw))
    stt = oracle.Setup(det, synth.uniform_field(), CKFSettings(rk_tolerance_mm=1e-8, surface_tolerance_mm=1e-10, **kw))
    rng = np.random.default_rng(9)
    n_cmp = n_inward_visits = n_turned = 0
    for trial in range(10):
        layer = int(rng.integers(0, 6))
        m = int(det.module_offset[layer] + rng.integers(0, det.n_phi[layer]) * det.n_z[layer] + det.n_z[layer] // 2 +
                rng.integers(-3, 4))
        n = np.cross(det.axis_u[m], det.axis_v[m])
        # pointing inward: opposite to the module normal, up to 1.2 rad off (so that some tips miss the inner layers)
        phi = math.atan2(-n[1], -n[0]) + rng.uniform(-1.2, 1.2)
        theta = rng.uniform(1.0, 2.1)
        pt = math.exp(rng.uniform(math.log(5.0), math.log(50.0)))     # stiff: the pre-filter is a tube around a line
        q = 1.0 if rng.random() < 0.5 else -1.0
        x = np.array([rng.uniform(-5, 5), rng.uniform(-10, 10), phi, theta, q * math.sin(theta) / pt, 0.0])
        d0 = np.array([math.sin(theta) * math.cos(phi), math.sin(theta) * math.sin(phi), math.cos(theta)])
        r0 = det.center[m] + x[0] * det.axis_u[m] + x[1] * det.axis_v[m]
        y0 = np.concatenate([r0, [0.0], d0, [x[4]]])
        want, near_edge = _crossings_any_direction(det, stt, y0, m)
        if near_edge:
            continue
        code0, *_ = oracle.move(off, m, x, np.eye(6) * 1e-6)
        assert oracle.STOP_NAMES[code0] == "NOT_OUTGOING"          # reading A7 without the flag
        visited, mm, xm = [], m, x
        while True:
            code, tg, xp, Cp, _ = oracle.move(on, mm, xm, np.eye(6) * 1e-6)
            if code != 0:
                assert oracle.STOP_NAMES[code] == "EXIT", (trial, oracle.STOP_NAMES[code])
                break
            visited.append(tg)
            xm, mm = xp, tg
        assert visited == want, (trial, layer, visited, want)
        n_cmp += 1
        normals = np.cross(det.axis_u[want], det.axis_v[want]) if want else np.zeros((0, 3))
        lay = det.module_layer[np.array(want, int)] if want else np.zeros(0, int)
        n_inward_visits += int(np.sum(lay < layer)) if want else 0
        n_turned += int(want != [] and lay.min() >= layer)          # turned inside its shell: left through the far side
    print("bidirectional pin: compared", n_cmp, "inward visits", n_inward_visits, "turned", n_turned)
    assert n_cmp >= 8 and n_inward_visits >= 10 and n_turned >= 1
