"""CPU oracle of the CKF hot path — TEST INFRASTRUCTURE, not the product.

ctypes binding of oracle/ckf_oracle.cpp (plain double-precision C++; see its header for the
citations and the list of pins).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package; paper_2505_22822_b200/ never does.
All arrays are widened to float64 here: for the fp32 configs the oracle computes in double on the
same float32-rounded inputs.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass
from typing import Optional

import numpy as np

from . import build as _build

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_fp = C.POINTER(C.c_float)


class OGeometry(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("layer_r", _dp), ("layer_half_z", _dp), ("n_phi", _ip), ("n_z", _ip),
                ("module_offset", _ip), ("n_modules", C.c_int32), ("center", _dp), ("axis_u", _dp), ("axis_v", _dp),
                ("half_u", _dp), ("half_v", _dp), ("x_over_x0", _dp), ("layer_kind", _ip), ("layer_r_min", _dp)]


class OField(C.Structure):
    _fields_ = [("kind", C.c_int32), ("uniform_b", C.c_double * 3), ("n", C.c_int32 * 3), ("origin", C.c_double * 3),
                ("spacing", C.c_double * 3), ("grid", _fp)]


class OConfig(C.Structure):
    _fields_ = [("chi2_max", C.c_double), ("max_branches_per_surface", C.c_int32),
                ("max_candidates_per_seed", C.c_int32), ("max_holes", C.c_int32), ("min_measurements", C.c_int32),
                ("rk_tolerance_mm", C.c_double), ("surface_tolerance_mm", C.c_double), ("h_max_mm", C.c_double),
                ("particle_mass_gev", C.c_double), ("max_rk_steps_per_surface", C.c_int32), ("max_levels", C.c_int32),
                ("energy_loss", C.c_int32), ("field_gradient", C.c_int32), ("bidirectional", C.c_int32)]


class OSeedConfig(C.Structure):
    _fields_ = [("layer_b", C.c_int32), ("layer_m", C.c_int32), ("layer_t", C.c_int32), ("dphi_max", C.c_double),
                ("cot_max", C.c_double), ("z0_max", C.c_double), ("dcot_max", C.c_double), ("pt_min", C.c_double),
                ("d0_max", C.c_double), ("sigma_angle", C.c_double), ("rel_sigma_qop", C.c_double),
                ("cov_scale", C.c_double)]


STOP_NAMES = {0: "NONE", 1: "EXIT", 2: "HOLES", 3: "NOT_OUTGOING", 4: "STEP_LIMIT", 5: "NUMERIC", 6: "LEVEL_LIMIT"}

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.oracle_ckf_find.restype = C.c_void_p
        L.oracle_ckf_find.argtypes = [C.POINTER(OGeometry), C.POINTER(OField), C.POINTER(OConfig), C.c_int32, _ip, _dp,
                                      _dp, C.c_int32, _ip, _dp, _dp, C.c_int32]
        L.oracle_result_n_tracks.restype = C.c_int32
        L.oracle_result_n_tracks.argtypes = [C.c_void_p]
        L.oracle_result_n_entries.restype = C.c_int64
        L.oracle_result_n_entries.argtypes = [C.c_void_p]
        L.oracle_result_counters.argtypes = [C.c_void_p, C.POINTER(C.c_int64)]
        L.oracle_result_copy.argtypes = [C.c_void_p, _ip, _ip, _dp, _ip, _ip, _ip, _ip, _dp, _dp, _dp]
        L.oracle_result_free.argtypes = [C.c_void_p]
        L.oracle_field_at.argtypes = [C.POINTER(OField), _dp, _dp]
        L.oracle_set_n3_literal_walk.argtypes = [C.c_int32]
        L.oracle_resolve_ambiguity.restype = None
        L.oracle_resolve_ambiguity.argtypes = [C.c_int32, _ip, _ip, _dp, C.c_int32, C.c_int32, C.c_double, _ip, _ip]
        L.oracle_propagate_free.restype = C.c_int32
        L.oracle_propagate_free.argtypes = [C.POINTER(OField), C.POINTER(OConfig), C.c_int32, _dp, _dp, C.c_double, _dp,
                                            _dp, _ip]
        L.oracle_move.restype = C.c_int32
        L.oracle_move.argtypes = [C.POINTER(OGeometry), C.POINTER(OField), C.POINTER(OConfig), C.c_int32, _dp, _dp, _ip,
                                  _dp, _dp, _dp]
        L.oracle_last_move_trials.restype = C.c_int64
        L.oracle_seed_find.restype = C.c_void_p
        L.oracle_seed_find.argtypes = [C.POINTER(OGeometry), C.POINTER(OField), C.POINTER(OSeedConfig), C.c_int32, _ip,
                                       _dp, _dp, C.c_int32]
        L.oracle_seed_count.restype = C.c_int32
        L.oracle_seed_count.argtypes = [C.c_void_p]
        L.oracle_seed_copy.argtypes = [C.c_void_p, _ip, _ip, _dp, _dp]
        L.oracle_seed_free.argtypes = [C.c_void_p]
        L.oracle_bound_to_bound.restype = C.c_int32
        L.oracle_bound_to_bound.argtypes = [C.POINTER(OGeometry), C.POINTER(OField), C.POINTER(OConfig), C.c_int32,
                                            C.c_int32, _dp, _dp, _dp]
        L.oracle_transport_cov.argtypes = [_dp, _dp, _dp]
        L.oracle_predicted_chi2.restype = C.c_double
        L.oracle_predicted_chi2.argtypes = [_dp, _dp, _dp, _dp]
        L.oracle_kalman_update.argtypes = [_dp, _dp, _dp, _dp, _dp, _dp]
        L.oracle_highland_theta0.restype = C.c_double
        L.oracle_highland_theta0.argtypes = [C.c_double, C.c_double, C.c_double]
        L.oracle_add_material.argtypes = [C.POINTER(OGeometry), C.POINTER(OConfig), C.c_int32, _dp, _dp]
        L.oracle_bethe_dedx.restype = C.c_double
        L.oracle_bethe_dedx.argtypes = [C.c_double, C.c_double]
        L.oracle_energy_loss.restype = C.c_double
        L.oracle_energy_loss.argtypes = [C.POINTER(OGeometry), C.POINTER(OConfig), C.c_int32, _dp, _dp, _dp]
        L.oracle_kf_fit.restype = None
        L.oracle_kf_fit.argtypes = [C.POINTER(OGeometry), C.POINTER(OField), C.POINTER(OConfig), _ip, _dp, _dp, _ip, _dp,
                                    _dp, C.c_int32, _ip, _ip, _ip, C.c_int32, _ip, _ip, _dp, _dp, _dp, _dp, _dp, C.c_int32]
        L.oracle_kf_fit_states.restype = C.c_int32
        L.oracle_kf_fit_states.argtypes = [C.POINTER(OGeometry), C.POINTER(OField), C.POINTER(OConfig), _ip, _dp, _dp,
                                           C.c_int32, _dp, _dp, C.c_int32, _ip, C.c_int32, _ip, _ip, _dp, _dp, _dp, _dp,
                                           _dp, _dp, _dp, C.c_int32]
        L.oracle_rts_smooth.restype = C.c_int32
        L.oracle_rts_smooth.argtypes = [C.c_int32, _dp, _dp, _dp, _dp, _dp, _dp, _dp]
        _lib = L
    return _lib


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _pd(a):
    return a.ctypes.data_as(_dp)


def _pi(a):
    return a.ctypes.data_as(_ip)


class Setup:
    """Holds the geometry / field / config structs (and keeps their numpy buffers alive)."""

    def __init__(self, det, fld, ckf):
        self._keep = []
        k = self._keep
        g = OGeometry()
        g.n_layers = int(det.n_layers)
        g.n_modules = int(det.n_modules)
        for name, conv in (("layer_r", _d), ("layer_half_z", _d), ("n_phi", _i), ("n_z", _i), ("module_offset", _i),
                           ("center", _d), ("axis_u", _d), ("axis_v", _d), ("half_u", _d), ("half_v", _d),
                           ("x_over_x0", _d)):
            arr = conv(getattr(det, name))
            k.append(arr)
            setattr(g, name, _pd(arr) if conv is _d else _pi(arr))
        if getattr(det, "layer_kind", None) is not None:      # endcap discs (row f3)
            lk, rm = _i(det.layer_kind), _d(det.layer_r_min)
            k.extend([lk, rm])
            g.layer_kind, g.layer_r_min = _pi(lk), _pd(rm)
        f = OField()
        f.kind = int(fld.kind)
        for a in range(3):
            f.uniform_b[a] = float(fld.uniform_b[a])
            f.n[a] = int(fld.n[a])
            f.origin[a] = float(fld.origin[a])
            f.spacing[a] = float(fld.spacing[a])
        if fld.grid is not None:
            grid = np.ascontiguousarray(fld.grid, dtype=np.float32)
            k.append(grid)
            f.grid = grid.ctypes.data_as(_fp)
        c = OConfig()
        for name, _t in OConfig._fields_:
            setattr(c, name, getattr(ckf, name, 0))
        self.geometry, self.field, self.config = g, f, c
        self.det = det


@dataclass
class Tracks:
    """Track candidates in the layout of `ckf_tracks` (include/ckf.h), all float64 / int32."""
    n_tracks: int
    track_offsets: np.ndarray
    meas_idx: np.ndarray
    entry_chi2: np.ndarray
    seed_id: np.ndarray
    n_holes: np.ndarray
    last_module: np.ndarray
    stop_reason: np.ndarray
    params: np.ndarray
    cov: np.ndarray
    chi2_sum: np.ndarray
    counters: Optional[dict] = None

    def meas_list(self, t: int):
        return self.meas_idx[self.track_offsets[t]:self.track_offsets[t + 1]]


def ckf_find(setup: Setup, module_offsets, loc, var, seed_module, seed_params, seed_cov, n_threads: int = 1) -> Tracks:
    L = lib()
    mo, lo, va = _i(module_offsets), _d(loc), _d(var)
    sm, sp, sc = _i(seed_module), _d(seed_params), _d(seed_cov)
    r = L.oracle_ckf_find(C.byref(setup.geometry), C.byref(setup.field), C.byref(setup.config), lo.shape[0], _pi(mo),
                          _pd(lo), _pd(va), sm.shape[0], _pi(sm), _pd(sp), _pd(sc), int(n_threads))
    try:
        nt = L.oracle_result_n_tracks(r)
        ne = L.oracle_result_n_entries(r)
        out = Tracks(nt, np.zeros(nt + 1, np.int32), np.zeros(ne, np.int32), np.zeros(ne), np.zeros(nt, np.int32),
                     np.zeros(nt, np.int32), np.zeros(nt, np.int32), np.zeros(nt, np.int32), np.zeros((nt, 6)),
                     np.zeros((nt, 36)), np.zeros(nt))
        L.oracle_result_copy(r, _pi(out.track_offsets), _pi(out.meas_idx), _pd(out.entry_chi2), _pi(out.seed_id),
                             _pi(out.n_holes), _pi(out.last_module), _pi(out.stop_reason), _pd(out.params),
                             _pd(out.cov), _pd(out.chi2_sum))
        cnt = (C.c_int64 * 6)()
        L.oracle_result_counters(r, cnt)
        out.counters = dict(zip(("visits", "rk_trials", "rk_accepted", "gate_tests", "updates", "tips"), list(cnt)))
    finally:
        L.oracle_result_free(r)
    return out


def find_event(setup: Setup, ev, n_threads: int = 1) -> Tracks:
    return ckf_find(setup, ev.module_offsets, ev.loc, ev.var, ev.seed_module, ev.seed_params, ev.seed_cov, n_threads)


# ------------------------------------------------------------------ pieces for the pins
def set_n3_literal_walk(on: bool):
    """Pin hook: navigate past the barrel ends as SURVEY.md N3 words it (True) instead of reading D11 (False, default)."""
    lib().oracle_set_n3_literal_walk(1 if on else 0)


def field_at(setup: Setup, r):
    r = _d(r)
    b = np.zeros(3)
    lib().oracle_field_at(C.byref(setup.field), _pd(r), _pd(b))
    return b


def propagate_free(setup: Setup, y, plane=None, cylinder_r=None):
    """y = (r[3], t, d[3], q/p).  Returns (status, y', D[8,8], n_steps)."""
    y = _d(y).copy()
    D = np.zeros((8, 8))
    ns = C.c_int32(0)
    if plane is not None:
        c, n = _d(plane[0]), _d(plane[1])
        st = lib().oracle_propagate_free(C.byref(setup.field), C.byref(setup.config), 0, _pd(c), _pd(n), 0.0, _pd(y),
                                         _pd(D), C.byref(ns))
    else:
        st = lib().oracle_propagate_free(C.byref(setup.field), C.byref(setup.config), 1, None, None,
                                         float(cylinder_r), _pd(y), _pd(D), C.byref(ns))
    return st, y, D, ns.value


def move(setup: Setup, module, x, Cov):
    x, Cov = _d(x), _d(Cov).reshape(36)
    xp, Cp, J = np.zeros(6), np.zeros(36), np.zeros(36)
    tg = C.c_int32(-1)
    st = lib().oracle_move(C.byref(setup.geometry), C.byref(setup.field), C.byref(setup.config), int(module), _pd(x),
                           _pd(Cov), C.byref(tg), _pd(xp), _pd(Cp), _pd(J))
    return st, tg.value, xp, Cp.reshape(6, 6), J.reshape(6, 6)


def last_move_trials() -> int:
    """RKN4 trials of this thread's last `move` (also of moves that ended in a stop)."""
    return int(lib().oracle_last_move_trials())


def bound_to_bound(setup: Setup, m_from, m_to, x):
    x = _d(x)
    xp, J = np.zeros(6), np.zeros(36)
    st = lib().oracle_bound_to_bound(C.byref(setup.geometry), C.byref(setup.field), C.byref(setup.config), int(m_from),
                                     int(m_to), _pd(x), _pd(xp), _pd(J))
    return st, xp, J.reshape(6, 6)


def transport_cov(J, Cov):
    J, Cov = _d(J).reshape(36), _d(Cov).reshape(36)
    o = np.zeros(36)
    lib().oracle_transport_cov(_pd(J), _pd(Cov), _pd(o))
    return o.reshape(6, 6)


def predicted_chi2(x, Cov, loc, var):
    x, Cov, loc, var = _d(x), _d(Cov).reshape(36), _d(loc), _d(var)
    return lib().oracle_predicted_chi2(_pd(x), _pd(Cov), _pd(loc), _pd(var))


def kalman_update(x, Cov, loc, var):
    x, Cov, loc, var = _d(x), _d(Cov).reshape(36), _d(loc), _d(var)
    xo, Co = np.zeros(6), np.zeros(36)
    lib().oracle_kalman_update(_pd(x), _pd(Cov), _pd(loc), _pd(var), _pd(xo), _pd(Co))
    return xo, Co.reshape(6, 6)


def highland_theta0(p, x_eff, mass):
    return lib().oracle_highland_theta0(float(p), float(x_eff), float(mass))


def add_material(setup: Setup, module, x, Cov):
    x, Cov = _d(x), _d(Cov).reshape(36).copy()
    lib().oracle_add_material(C.byref(setup.geometry), C.byref(setup.config), int(module), _pd(x), _pd(Cov))
    return Cov.reshape(6, 6)


def bethe_dedx(p, mass):
    """Mean stopping power [GeV cm^2 / g] of the oracle's rule E (silicon, no density correction)."""
    return lib().oracle_bethe_dedx(float(p), float(mass))


def energy_loss(setup: Setup, module, x):
    """Rule E on leaving `module`: (dE [GeV], parameters after the loss, g = d(q/p)'/d(q/p))."""
    x = _d(x)
    xo, g = np.zeros(6), C.c_double(1.0)
    dE = lib().oracle_energy_loss(C.byref(setup.geometry), C.byref(setup.config), int(module), _pd(x), _pd(xo), C.byref(g))
    return dE, xo, g.value


# ------------------------------------------------------------------ K: KF fit + RTS smoother
@dataclass
class Fits:
    """Result of the KF fit + RTS smoother over a CSR list of candidates (layout of `ckf_fits`, include/ckf.h)."""
    n_tracks: int
    status: np.ndarray        # [n_tracks] 0 = fitted, else stop reason
    n_states: np.ndarray      # [n_tracks] visited modules of the forward pass
    chi2_sum: np.ndarray      # [n_tracks] forward (predicted-residual) chi2 sum
    last_params: np.ndarray   # [n_tracks, 6] forward-filtered state at the last measurement
    last_cov: np.ndarray      # [n_tracks, 36]
    first_cov: np.ndarray     # [n_tracks, 36] smoothed covariance at the first measurement
    entry_params: np.ndarray  # [n_entries, 6] smoothed parameters at every measurement of the list


def kf_fit(setup: Setup, ev, track_offsets, meas_idx, seed_id, n_threads: int = 1, smoother: int = 0) -> Fits:
    """smoother: 0 = RTS recursion (K4), 1 = two-filter 'optimal' smoother (K4')."""
    L = lib()
    mo, lo, va = _i(ev.module_offsets), _d(ev.loc), _d(ev.var)
    sm, sp, sc = _i(ev.seed_module), _d(ev.seed_params), _d(ev.seed_cov)
    to, mi, si = _i(track_offsets), _i(meas_idx), _i(seed_id)
    nt = si.shape[0]
    ne = int(to[nt]) if nt else 0
    out = Fits(nt, np.zeros(nt, np.int32), np.zeros(nt, np.int32), np.zeros(nt), np.zeros((nt, 6)), np.zeros((nt, 36)),
               np.zeros((nt, 36)), np.zeros((ne, 6)))
    L.oracle_kf_fit(C.byref(setup.geometry), C.byref(setup.field), C.byref(setup.config), _pi(mo), _pd(lo), _pd(va),
                    _pi(sm), _pd(sp), _pd(sc), nt, _pi(to), _pi(mi), _pi(si), int(n_threads), _pi(out.status),
                    _pi(out.n_states), _pd(out.chi2_sum), _pd(out.last_params), _pd(out.last_cov), _pd(out.first_cov),
                    _pd(out.entry_params), int(smoother))
    return out


def kf_fit_states(setup: Setup, ev, seed: int, meas, max_states: int = 64, smoother: int = 0):
    """Every state of one track's fit: dict of module, meas, xp, Cp, xf, Cf, J, xs, Cs (arrays over states)."""
    mo, lo, va = _i(ev.module_offsets), _d(ev.loc), _d(ev.var)
    sx, sC = _d(ev.seed_params[seed]), _d(ev.seed_cov[seed]).reshape(36)
    me = _i(meas)
    n = max_states
    mod, mu = np.zeros(n, np.int32), np.zeros(n, np.int32)
    xp, xf, xs = np.zeros((n, 6)), np.zeros((n, 6)), np.zeros((n, 6))
    Cp, Cf, J, Cs = np.zeros((n, 36)), np.zeros((n, 36)), np.zeros((n, 36)), np.zeros((n, 36))
    ns = lib().oracle_kf_fit_states(C.byref(setup.geometry), C.byref(setup.field), C.byref(setup.config), _pi(mo),
                                    _pd(lo), _pd(va), int(ev.seed_module[seed]), _pd(sx), _pd(sC), me.shape[0], _pi(me),
                                    n, _pi(mod), _pi(mu), _pd(xp), _pd(Cp), _pd(xf), _pd(Cf), _pd(J), _pd(xs), _pd(Cs),
                                    int(smoother))
    if ns < 0:
        return {"status": -ns}
    ns = min(ns, n)
    r6 = lambda a: a[:ns].reshape(ns, 6, 6)
    return {"status": 0, "module": mod[:ns], "meas": mu[:ns], "xp": xp[:ns], "xf": xf[:ns], "xs": xs[:ns],
            "Cp": r6(Cp), "Cf": r6(Cf), "J": r6(J), "Cs": r6(Cs)}


def rts_smooth(xp, Cp, xf, Cf, J):
    """The RTS recursion alone on given states ([n,6] / [n,6,6]; J[k] leads into state k)."""
    xp, xf = _d(xp), _d(xf)
    n = xp.shape[0]
    Cp, Cf, J = _d(Cp).reshape(n, 36), _d(Cf).reshape(n, 36), _d(J).reshape(n, 36)
    xs, Cs = np.zeros((n, 6)), np.zeros((n, 36))
    rc = lib().oracle_rts_smooth(n, _pd(xp), _pd(Cp), _pd(xf), _pd(Cf), _pd(J), _pd(xs), _pd(Cs))
    return rc, xs, Cs.reshape(n, 6, 6)


# ------------------------------------------------------------------ AR: ambiguity resolution
def resolve_ambiguity(track_offsets, meas_idx, chi2_sum, n_measurements: int, max_shared_hits: int = 1,
                      max_shared_fraction: float = 1.0):
    """Greedy shared-hit resolver (rules AR1-AR3).  Returns (accepted[n_tracks] in {0,1}, n_shared[n_tracks])."""
    to, mi, c2 = _i(track_offsets), _i(meas_idx), _d(chi2_sum)
    nt = c2.shape[0]
    acc, ns = np.zeros(nt, np.int32), np.zeros(nt, np.int32)
    lib().oracle_resolve_ambiguity(nt, _pi(to), _pi(mi), _pd(c2), int(n_measurements), int(max_shared_hits),
                                   float(max_shared_fraction), _pi(acc), _pi(ns))
    return acc, ns


# ------------------------------------------------------------------ S: triplet seeding + parameter estimation
def seed_find(setup: Setup, seeding, module_offsets, loc, var, n_threads: int = 1):
    """Rules S0-S6 over all combinations.  Returns dict(triplets [n,3] measurement indices (bottom, middle, top),
    module [n], params [n,6], cov [n,36]), ordered by (bottom, middle, top)."""
    c = OSeedConfig()
    for name, _t in OSeedConfig._fields_:
        setattr(c, name, getattr(seeding, name))
    mo, lo, va = _i(module_offsets), _d(loc), _d(var)
    r = lib().oracle_seed_find(C.byref(setup.geometry), C.byref(setup.field), C.byref(c), lo.shape[0], _pi(mo), _pd(lo),
                               _pd(va), int(n_threads))
    try:
        n = lib().oracle_seed_count(r)
        out = dict(triplets=np.zeros((n, 3), np.int32), module=np.zeros(n, np.int32), params=np.zeros((n, 6)),
                   cov=np.zeros((n, 36)))
        lib().oracle_seed_copy(r, _pi(out["triplets"]), _pi(out["module"]), _pd(out["params"]), _pd(out["cov"]))
    finally:
        lib().oracle_seed_free(r)
    return out
