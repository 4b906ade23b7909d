"""Thin Python binding of the C ABI in include/ckf.h — argument marshalling only.

Every step of the CKF runs in the CUDA kernels of libckf.so; PyTorch provides device memory and streams.
There is no CPU fallback: if libckf.so is missing or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_fp = C.POINTER(C.c_float)
_vp = C.c_void_p

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libckf.so")

EXPORTS = ("ckf_create", "ckf_find", "ckf_find_host", "ckf_fit", "ckf_get_counters", "ckf_get_launch_info", "ckf_destroy",
           "ckf_set_timing", "ckf_get_timing", "ckf_measure_alu_peak", "ckf_resolve", "ckf_resolve_static", "ckf_seed",
           "ckf_last_error", "ckf_abi_version")


class ckf_geometry(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("layer_r", _dp), ("layer_half_z", _dp), ("n_phi", _ip), ("n_z", _ip),
                ("module_offset", _ip), ("n_modules", C.c_int32), ("center", _dp), ("axis_u", _dp), ("axis_v", _dp),
                ("half_u", _dp), ("half_v", _dp), ("x_over_x0", _dp), ("layer_kind", _ip), ("layer_r_min", _dp)]


class ckf_field(C.Structure):
    _fields_ = [("kind", C.c_int32), ("uniform_b", C.c_double * 3), ("n", C.c_int32 * 3), ("origin", C.c_double * 3),
                ("spacing", C.c_double * 3), ("grid", _fp)]


class ckf_config(C.Structure):
    _fields_ = [("precision", C.c_int32), ("chi2_max", C.c_double), ("max_branches_per_surface", C.c_int32),
                ("max_candidates_per_seed", C.c_int32), ("max_holes", C.c_int32), ("min_measurements", C.c_int32),
                ("rk_tolerance_mm", C.c_double), ("surface_tolerance_mm", C.c_double), ("h_max_mm", C.c_double),
                ("particle_mass_gev", C.c_double), ("max_rk_steps_per_surface", C.c_int32), ("max_levels", C.c_int32),
                ("max_seeds", C.c_int32), ("max_measurements", C.c_int32), ("max_tracks", C.c_int32),
                ("max_track_entries", C.c_int32), ("max_links", C.c_int32), ("max_tips_per_level", C.c_int32),
                ("n_streams", C.c_int32), ("max_events_per_find", C.c_int32), ("energy_loss", C.c_int32),
                ("field_gradient", C.c_int32), ("bidirectional", C.c_int32), ("max_seed_doublets", C.c_int32), ("max_fit_tracks", C.c_int32)]


class ckf_measurements(C.Structure):
    _fields_ = [("n", C.c_int32), ("module_offsets", _vp), ("loc", _vp), ("var", _vp), ("n_events", C.c_int32)]


class ckf_seeds(C.Structure):
    _fields_ = [("n", C.c_int32), ("module_id", _vp), ("params", _vp), ("cov", _vp)]


class ckf_tracks(C.Structure):
    _fields_ = [("n_tracks", _vp), ("status", _vp), ("track_offsets", _vp), ("meas_idx", _vp), ("seed_id", _vp),
                ("n_holes", _vp), ("last_module", _vp), ("stop_reason", _vp), ("params", _vp), ("cov", _vp),
                ("chi2_sum", _vp), ("entry_chi2", _vp)]


class ckf_fits(C.Structure):
    _fields_ = [("status", _vp), ("n_states", _vp), ("chi2_sum", _vp), ("last_params", _vp), ("last_cov", _vp),
                ("first_cov", _vp), ("entry_params", _vp), ("work", _vp), ("smoother_precision", C.c_int32),
                ("n_tracks_upper", C.c_int32), ("smoother", C.c_int32)]


class ckf_resolution(C.Structure):
    _fields_ = [("accepted", _vp), ("n_shared", _vp), ("summary", _vp), ("max_shared_hits", C.c_int32),
                ("max_shared_fraction", C.c_double)]


class ckf_seeding(C.Structure):
    _fields_ = [("layer_b", C.c_int32), ("layer_m", C.c_int32), ("layer_t", C.c_int32), ("dphi_max", C.c_double),
                ("cot_max", C.c_double), ("z0_max", C.c_double), ("dcot_max", C.c_double), ("pt_min", C.c_double),
                ("d0_max", C.c_double), ("sigma_angle", C.c_double), ("rel_sigma_qop", C.c_double),
                ("cov_scale", C.c_double)]


class ckf_seed_out(C.Structure):
    _fields_ = [("n_seeds", _vp), ("status", _vp), ("module_id", _vp), ("params", _vp), ("cov", _vp), ("triplets", _vp),
                ("capacity", C.c_int32)]


class ckf_timing(C.Structure):
    _fields_ = [("init_ms", C.c_float), ("sort_ms", C.c_float), ("step_ms", C.c_float), ("visit_ms", C.c_float),
                ("scan_ms", C.c_float), ("update_ms", C.c_float), ("emit_ms", C.c_float), ("launches", C.c_int32)]


class ckf_counters(C.Structure):
    _fields_ = [("tips", C.c_int64), ("visits", C.c_int64), ("rk_trials", C.c_int64), ("rk_accepted", C.c_int64),
                ("gate_tests", C.c_int64), ("updates", C.c_int64), ("links", C.c_int64), ("iterations", C.c_int64),
                ("gate_tests_executed", C.c_int64)]


_lib = None


def load_library():
    """Loads libckf.so (built in-tree by `_build.py`).  Raises if it is missing: no fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2505_22822_b200._build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.ckf_create.restype = C.c_int
        L.ckf_create.argtypes = [C.POINTER(ckf_geometry), C.POINTER(ckf_field), C.POINTER(ckf_config), C.POINTER(_vp)]
        for name in ("ckf_find", "ckf_find_host"):
            fn = getattr(L, name)
            fn.restype = C.c_int
            fn.argtypes = [_vp, C.POINTER(ckf_measurements), C.POINTER(ckf_seeds), C.POINTER(ckf_tracks), _vp]
        L.ckf_fit.restype = C.c_int
        L.ckf_fit.argtypes = [_vp, C.POINTER(ckf_measurements), C.POINTER(ckf_seeds), C.POINTER(ckf_tracks),
                              C.POINTER(ckf_fits), _vp]
        L.ckf_resolve.restype = C.c_int
        L.ckf_resolve.argtypes = [_vp, C.POINTER(ckf_tracks), C.c_int32, C.POINTER(ckf_resolution), _vp]
        L.ckf_resolve_static.restype = C.c_int
        L.ckf_resolve_static.argtypes = [C.POINTER(ckf_tracks), C.c_int32, C.c_int32, C.c_int32, C.POINTER(ckf_resolution), _vp]
        L.ckf_seed.restype = C.c_int
        L.ckf_seed.argtypes = [_vp, C.POINTER(ckf_measurements), C.POINTER(ckf_seeding), C.POINTER(ckf_seed_out), _vp]
        L.ckf_set_timing.restype = C.c_int
        L.ckf_set_timing.argtypes = [_vp, C.c_int]
        L.ckf_get_timing.restype = C.c_int
        L.ckf_get_timing.argtypes = [_vp, _vp, C.POINTER(ckf_timing)]
        L.ckf_get_counters.restype = C.c_int
        L.ckf_get_counters.argtypes = [_vp, _vp, C.POINTER(ckf_counters)]
        L.ckf_get_launch_info.restype = C.c_int
        L.ckf_get_launch_info.argtypes = [_vp, _ip, _ip, _ip, _ip]
        L.ckf_destroy.restype = C.c_int
        L.ckf_destroy.argtypes = [_vp]
        L.ckf_last_error.restype = C.c_char_p
        L.ckf_last_error.argtypes = [_vp]
        L.ckf_abi_version.restype = C.c_int
        L.ckf_measure_alu_peak.restype = C.c_int
        L.ckf_measure_alu_peak.argtypes = [C.c_int, C.c_double, _dp, _dp, _dp, _dp]
        _lib = L
    return _lib


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def make_geometry(det, keep: list) -> ckf_geometry:
    g = ckf_geometry()
    g.n_layers = int(det.n_layers)
    g.n_modules = int(det.n_modules)
    for name, conv, pt in (("layer_r", _d, _dp), ("layer_half_z", _d, _dp), ("n_phi", _i, _ip), ("n_z", _i, _ip),
                           ("module_offset", _i, _ip), ("center", _d, _dp), ("axis_u", _d, _dp), ("axis_v", _d, _dp),
                           ("half_u", _d, _dp), ("half_v", _d, _dp), ("x_over_x0", _d, _dp)):
        arr = conv(getattr(det, name))
        keep.append(arr)
        setattr(g, name, arr.ctypes.data_as(pt))
    if getattr(det, "layer_kind", None) is not None:      # endcap discs
        lk, rm = _i(det.layer_kind), _d(det.layer_r_min)
        keep.extend([lk, rm])
        g.layer_kind, g.layer_r_min = lk.ctypes.data_as(_ip), rm.ctypes.data_as(_dp)
    return g


def make_field(fld, keep: list) -> ckf_field:
    f = ckf_field()
    f.kind = int(fld.kind)
    for a in range(3):
        f.uniform_b[a] = float(fld.uniform_b[a])
        f.n[a] = int(fld.n[a])
        f.origin[a] = float(fld.origin[a])
        f.spacing[a] = float(fld.spacing[a])
    if fld.grid is not None:
        grid = np.ascontiguousarray(fld.grid, dtype=np.float32)
        keep.append(grid)
        f.grid = grid.ctypes.data_as(_fp)
    return f


def make_config(ckf, precision: int, max_seeds: int, max_measurements: int, max_tracks: int, max_track_entries: int,
                max_links: int = 0, n_streams: int = 1, max_tips_per_level: int = 0,
                max_events_per_find: int = 1, max_fit_tracks: int = 0, max_seed_doublets: int = 0) -> ckf_config:
    c = ckf_config()
    c.precision = int(precision)
    for name in ("chi2_max", "max_branches_per_surface", "max_candidates_per_seed", "max_holes", "min_measurements",
                 "rk_tolerance_mm", "surface_tolerance_mm", "h_max_mm", "particle_mass_gev",
                 "max_rk_steps_per_surface", "max_levels"):
        setattr(c, name, getattr(ckf, name))
    c.max_seeds, c.max_measurements = int(max_seeds), int(max_measurements)
    c.max_tracks, c.max_track_entries = int(max_tracks), int(max_track_entries)
    c.max_links, c.n_streams = int(max_links), int(n_streams)
    c.max_tips_per_level = int(max_tips_per_level)
    c.max_events_per_find = int(max_events_per_find)
    c.max_fit_tracks = int(max_fit_tracks)
    c.max_seed_doublets = int(max_seed_doublets)
    c.energy_loss = int(getattr(ckf, "energy_loss", 0))
    c.field_gradient = int(getattr(ckf, "field_gradient", 0))
    c.bidirectional = int(getattr(ckf, "bidirectional", 0))
    return c


def measure_alu_peak(mix: int, seconds: float = 1.0) -> dict:
    """ckf_measure_alu_peak: FMA-chain throughput of the current device (mix 0 float32, 1 float64, 2 both)."""
    v = [C.c_double(0.0) for _ in range(4)]
    rc = load_library().ckf_measure_alu_peak(int(mix), float(seconds), *[C.byref(x) for x in v])
    if rc != 0:
        raise RuntimeError("ckf_measure_alu_peak failed (%d): %s" % (rc, load_library().ckf_last_error(None).decode()))
    return dict(tflops_f32=v[0].value, tflops_f64=v[1].value, best_f32=v[2].value, best_f64=v[3].value)


RESOLVE_STATIC_MAX_TRACKS = 65536           # CKF_RESOLVE_STATIC_MAX_TRACKS
RESOLVE_STATIC_MAX_MEASUREMENTS = 131072    # CKF_RESOLVE_STATIC_MAX_MEASUREMENTS


def resolve_static(tracks: dict, n_measurements: int, res: dict, precision: int, max_shared_hits: int = 1,
                   max_shared_fraction: float = 1.0, stream=None):
    """ckf_resolve_static: ambiguity resolution of the candidates in `tracks` (device tensors filled by CKF.find) with no
    handle and no allocation inside the library; scratch in a static device array, so sizes are limited (see ckf.h).
    `res` as from CKF.alloc_resolution; its length is the capacity passed as max_tracks."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream()
    lib = load_library()
    o = ckf_tracks(*[tracks[k].data_ptr() for k in ("n_tracks", "status", "track_offsets", "meas_idx", "seed_id",
                                                    "n_holes", "last_module", "stop_reason", "params", "cov",
                                                    "chi2_sum", "entry_chi2")])
    r = ckf_resolution(res["accepted"].data_ptr(), res["n_shared"].data_ptr(), res["summary"].data_ptr(),
                       int(max_shared_hits), float(max_shared_fraction))
    cap = min(int(res["accepted"].shape[0]), int(tracks["chi2_sum"].shape[0]))
    rc = lib.ckf_resolve_static(C.byref(o), cap, int(n_measurements), int(precision), C.byref(r), _vp(st.cuda_stream))
    if rc != 0:
        raise RuntimeError("ckf_resolve_static failed (%d): %s" % (rc, lib.ckf_last_error(None).decode()))


@dataclass
class EventBatch:
    """B events concatenated for one ckf_find (include/ckf.h, ckf_measurements): virtual module ids
    event * n_modules + module in `module_offsets` and `seed_module`; `seed_ranges` / `meas_ranges` split the results."""
    n_events: int
    module_offsets: np.ndarray
    loc: np.ndarray
    var: np.ndarray
    seed_module: np.ndarray
    seed_params: np.ndarray
    seed_cov: np.ndarray
    seed_ranges: list
    meas_ranges: list

    @property
    def n_seeds(self) -> int:
        return int(self.seed_module.shape[0])

    @property
    def n_measurements(self) -> int:
        return int(self.loc.shape[0])


def concat_events(evs, n_modules: int) -> EventBatch:
    """Argument marshalling only: concatenates the arrays of independent events into one batch."""
    offs, mo, so = [], 0, 0
    seed_ranges, meas_ranges, smod = [], [], []
    for e, ev in enumerate(evs):
        off = np.asarray(ev.module_offsets, np.int64)
        offs.append(off[:-1] + mo if e < len(evs) - 1 else off + mo)
        meas_ranges.append((mo, mo + ev.n_measurements))
        seed_ranges.append((so, so + ev.n_seeds))
        smod.append(np.asarray(ev.seed_module, np.int64) + e * n_modules)
        mo += ev.n_measurements
        so += ev.n_seeds
    return EventBatch(len(evs), np.concatenate(offs).astype(np.int32), np.concatenate([ev.loc for ev in evs]),
                      np.concatenate([ev.var for ev in evs]), np.concatenate(smod).astype(np.int32),
                      np.concatenate([ev.seed_params for ev in evs]), np.concatenate([ev.seed_cov for ev in evs]),
                      seed_ranges, meas_ranges)


@dataclass
class TrackArrays:
    """Host copy of `ckf_tracks` (numpy)."""
    n_tracks: int
    status: int
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

    def meas_list(self, t: int):
        return self.meas_idx[self.track_offsets[t]:self.track_offsets[t + 1]]


class CKF:
    """ckf_create / ckf_find / ckf_find_host / ckf_destroy with torch tensors as device memory."""

    def __init__(self, det, fld, ckf, precision: int, max_seeds: int, max_measurements: int,
                 max_tracks: Optional[int] = None, max_track_entries: Optional[int] = None, max_links: int = 0,
                 n_streams: int = 1, max_tips_per_level: int = 0, max_events_per_find: int = 1,
                 max_fit_tracks: Optional[int] = None, max_seed_doublets: int = 0):
        """max_fit_tracks: candidates per ckf_fit pass (sizes the state store reserved by ckf_create); None = all of
        max_tracks up to the library's pass limit, 0 = this handle never fits."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: paper_2505_22822_b200 has no CPU fallback")
        self.torch = torch
        self.lib = load_library()
        self.precision = int(precision)
        self.tdtype = torch.float32 if precision == 32 else torch.float64
        self.ndtype = np.float32 if precision == 32 else np.float64
        self.n_modules = int(det.n_modules)
        self.max_tracks = int(max_tracks if max_tracks is not None else 8 * max_seeds)
        self.max_track_entries = int(max_track_entries if max_track_entries is not None else 16 * self.max_tracks)
        keep = []
        g = make_geometry(det, keep)
        f = make_field(fld, keep)
        self.config = make_config(ckf, precision, max_seeds, max_measurements, self.max_tracks, self.max_track_entries,
                                  max_links, n_streams, max_tips_per_level, max_events_per_find,
                                  self.max_tracks if max_fit_tracks is None else max_fit_tracks, max_seed_doublets)
        h = _vp()
        rc = self.lib.ckf_create(C.byref(g), C.byref(f), C.byref(self.config), C.byref(h))
        if rc != 0:
            raise RuntimeError("ckf_create failed (%d): %s" % (rc, self.lib.ckf_last_error(None).decode()))
        self.handle = h

    # ------------------------------------------------------------------ device-resident path
    def alloc_tracks(self, device="cuda"):
        t = self.torch
        i32 = dict(dtype=t.int32, device=device)
        T = dict(dtype=self.tdtype, device=device)
        nt, ne = self.max_tracks, self.max_track_entries
        return dict(n_tracks=t.zeros(1, **i32), status=t.zeros(1, **i32), track_offsets=t.zeros(nt + 1, **i32),
                    meas_idx=t.zeros(ne, **i32), seed_id=t.zeros(nt, **i32), n_holes=t.zeros(nt, **i32),
                    last_module=t.zeros(nt, **i32), stop_reason=t.zeros(nt, **i32), params=t.zeros(nt, 6, **T),
                    cov=t.zeros(nt, 36, **T), chi2_sum=t.zeros(nt, **T), entry_chi2=t.zeros(ne, **T))

    def upload_event(self, ev, device="cuda"):
        t = self.torch
        return dict(
            n_events=int(getattr(ev, "n_events", 1)),
            module_offsets=t.from_numpy(np.ascontiguousarray(ev.module_offsets, np.int32)).to(device),
            loc=t.from_numpy(np.ascontiguousarray(ev.loc, self.ndtype)).to(device),
            var=t.from_numpy(np.ascontiguousarray(ev.var, self.ndtype)).to(device),
            seed_module=t.from_numpy(np.ascontiguousarray(ev.seed_module, np.int32)).to(device),
            seed_params=t.from_numpy(np.ascontiguousarray(ev.seed_params, self.ndtype)).to(device),
            seed_cov=t.from_numpy(np.ascontiguousarray(ev.seed_cov, self.ndtype)).to(device))

    def _structs(self, d, out, ptr):
        m = ckf_measurements(int(d["loc"].shape[0]), ptr(d["module_offsets"]), ptr(d["loc"]), ptr(d["var"]),
                             int(d.get("n_events", 1)))
        s = ckf_seeds(int(d["seed_module"].shape[0]), ptr(d["seed_module"]), ptr(d["seed_params"]), ptr(d["seed_cov"]))
        o = ckf_tracks(*[ptr(out[k]) for k in ("n_tracks", "status", "track_offsets", "meas_idx", "seed_id", "n_holes",
                                               "last_module", "stop_reason", "params", "cov", "chi2_sum",
                                               "entry_chi2")])
        return m, s, o

    def find(self, dev_event: dict, out: dict, stream=None):
        """Asynchronous ckf_find on device tensors; `stream` is a torch.cuda.Stream (default: current)."""
        st = stream if stream is not None else self.torch.cuda.current_stream()
        m, s, o = self._structs(dev_event, out, lambda x: x.data_ptr())
        rc = self.lib.ckf_find(self.handle, C.byref(m), C.byref(s), C.byref(o), _vp(st.cuda_stream))
        if rc != 0:
            raise RuntimeError("ckf_find failed (%d): %s" % (rc, self.lib.ckf_last_error(self.handle).decode()))

    # ------------------------------------------------------------------ KF fit + RTS smoother (ckf_fit)
    def alloc_fits(self, device="cuda"):
        t = self.torch
        i32 = dict(dtype=t.int32, device=device)
        T = dict(dtype=self.tdtype, device=device)
        nt, ne = self.max_tracks, self.max_track_entries
        return dict(status=t.zeros(nt, **i32), n_states=t.zeros(nt, **i32), chi2_sum=t.zeros(nt, **T),
                    last_params=t.zeros(nt, 6, **T), last_cov=t.zeros(nt, 36, **T), first_cov=t.zeros(nt, 36, **T),
                    entry_params=t.zeros(ne, 6, **T), work=t.zeros(4, dtype=t.int64, device=device))

    def fit(self, dev_event: dict, tracks: dict, fits: dict, stream=None, smoother_precision: int = 0, smoother: int = 0,
            n_tracks_upper: int = 0):
        """Asynchronous ckf_fit of the candidates in `tracks` (device tensors filled by `find`)."""
        st = stream if stream is not None else self.torch.cuda.current_stream()
        m, s, o = self._structs(dev_event, tracks, lambda x: x.data_ptr())
        f = ckf_fits(*[fits[k].data_ptr() for k in ("status", "n_states", "chi2_sum", "last_params", "last_cov",
                                                    "first_cov", "entry_params", "work")],
                     int(smoother_precision), int(n_tracks_upper), int(smoother))
        rc = self.lib.ckf_fit(self.handle, C.byref(m), C.byref(s), C.byref(o), C.byref(f), _vp(st.cuda_stream))
        if rc != 0:
            raise RuntimeError("ckf_fit failed (%d): %s" % (rc, self.lib.ckf_last_error(self.handle).decode()))

    def download_fits(self, fits: dict, n_tracks: int, n_entries: int) -> dict:
        out = {}
        for k, v in fits.items():
            a = v.cpu().numpy()
            if k != "work":
                a = a[:n_entries] if k == "entry_params" else a[:n_tracks]
            out[k] = a.astype(np.float64) if a.dtype.kind == "f" else a.copy()
        return out

    # ------------------------------------------------------------------ seeding + parameter estimation (ckf_seed)
    def alloc_seeds(self, capacity: int, device="cuda"):
        t = self.torch
        i32 = dict(dtype=t.int32, device=device)
        T = dict(dtype=self.tdtype, device=device)
        return dict(n_seeds=t.zeros(1, **i32), status=t.zeros(1, **i32), module_id=t.zeros(capacity, **i32),
                    params=t.zeros(capacity, 6, **T), cov=t.zeros(capacity, 36, **T), triplets=t.zeros(capacity, 3, **i32))

    def seed(self, dev_event: dict, seeding, seeds: dict, stream=None):
        """Asynchronous ckf_seed on the measurements of `dev_event` (device tensors); `seeding` = synth.SeedSettings."""
        st = stream if stream is not None else self.torch.cuda.current_stream()
        m = ckf_measurements(int(dev_event["loc"].shape[0]), dev_event["module_offsets"].data_ptr(),
                             dev_event["loc"].data_ptr(), dev_event["var"].data_ptr(), 1)
        sc = ckf_seeding(*[getattr(seeding, n) for n, _ in ckf_seeding._fields_])
        o = ckf_seed_out(*[seeds[k].data_ptr() for k in ("n_seeds", "status", "module_id", "params", "cov", "triplets")],
                         int(seeds["module_id"].shape[0]))
        rc = self.lib.ckf_seed(self.handle, C.byref(m), C.byref(sc), C.byref(o), _vp(st.cuda_stream))
        if rc != 0:
            raise RuntimeError("ckf_seed failed (%d): %s" % (rc, self.lib.ckf_last_error(self.handle).decode()))

    # ------------------------------------------------------------------ ambiguity resolution (ckf_resolve)
    def alloc_resolution(self, device="cuda"):
        t = self.torch
        i32 = dict(dtype=t.int32, device=device)
        return dict(accepted=t.zeros(self.max_tracks, **i32), n_shared=t.zeros(self.max_tracks, **i32),
                    summary=t.zeros(2, **i32))

    def resolve(self, tracks: dict, n_measurements: int, res: dict, max_shared_hits: int = 1,
                max_shared_fraction: float = 1.0, stream=None):
        """Asynchronous ckf_resolve of the candidates in `tracks` (device tensors filled by `find`)."""
        st = stream if stream is not None else self.torch.cuda.current_stream()
        o = ckf_tracks(*[tracks[k].data_ptr() for k in ("n_tracks", "status", "track_offsets", "meas_idx", "seed_id",
                                                        "n_holes", "last_module", "stop_reason", "params", "cov",
                                                        "chi2_sum", "entry_chi2")])
        r = ckf_resolution(res["accepted"].data_ptr(), res["n_shared"].data_ptr(), res["summary"].data_ptr(),
                           int(max_shared_hits), float(max_shared_fraction))
        rc = self.lib.ckf_resolve(self.handle, C.byref(o), int(n_measurements), C.byref(r), _vp(st.cuda_stream))
        if rc != 0:
            raise RuntimeError("ckf_resolve failed (%d): %s" % (rc, self.lib.ckf_last_error(self.handle).decode()))

    def find_host(self, host_event: dict, host_out: dict, stream=None):
        """ckf_find_host on (pinned) host tensors: H2D, find, D2H inside; synchronous on return."""
        st = stream if stream is not None else self.torch.cuda.current_stream()
        m, s, o = self._structs(host_event, host_out, lambda x: x.data_ptr())
        rc = self.lib.ckf_find_host(self.handle, C.byref(m), C.byref(s), C.byref(o), _vp(st.cuda_stream))
        if rc != 0:
            raise RuntimeError("ckf_find_host failed (%d): %s" % (rc, self.lib.ckf_last_error(self.handle).decode()))

    def pinned_event(self, ev):
        d = self.upload_event(ev, device="cpu")
        return {k: (v.pin_memory() if hasattr(v, "pin_memory") else v) for k, v in d.items()}

    def pinned_tracks(self):
        d = self.alloc_tracks(device="cpu")
        return {k: v.pin_memory() for k, v in d.items()}

    def download(self, out: dict) -> TrackArrays:
        cpu = {k: v.cpu().numpy() for k, v in out.items()} if out["n_tracks"].is_cuda else \
            {k: v.numpy() for k, v in out.items()}
        nt = int(cpu["n_tracks"][0])
        ne = int(cpu["track_offsets"][nt]) if nt > 0 else 0
        return TrackArrays(nt, int(cpu["status"][0]), cpu["track_offsets"][:nt + 1].copy(), cpu["meas_idx"][:ne].copy(),
                           cpu["entry_chi2"][:ne].astype(np.float64), cpu["seed_id"][:nt].copy(),
                           cpu["n_holes"][:nt].copy(), cpu["last_module"][:nt].copy(), cpu["stop_reason"][:nt].copy(),
                           cpu["params"][:nt].astype(np.float64), cpu["cov"][:nt].astype(np.float64),
                           cpu["chi2_sum"][:nt].astype(np.float64))

    def set_timing(self, on: bool) -> None:
        self.lib.ckf_set_timing(self.handle, 1 if on else 0)

    def timing(self, stream=None) -> dict:
        st = stream if stream is not None else self.torch.cuda.current_stream()
        t = ckf_timing()
        rc = self.lib.ckf_get_timing(self.handle, _vp(st.cuda_stream), C.byref(t))
        if rc != 0:
            raise RuntimeError("ckf_get_timing failed: %s" % self.lib.ckf_last_error(self.handle).decode())
        return {k: getattr(t, k) for k, _ in ckf_timing._fields_}

    def counters(self, stream=None) -> dict:
        st = stream if stream is not None else self.torch.cuda.current_stream()
        c = ckf_counters()
        rc = self.lib.ckf_get_counters(self.handle, _vp(st.cuda_stream), C.byref(c))
        if rc != 0:
            raise RuntimeError("ckf_get_counters failed: %s" % self.lib.ckf_last_error(self.handle).decode())
        return {k: int(getattr(c, k)) for k, _ in ckf_counters._fields_}

    def launch_info(self) -> dict:
        v = [C.c_int32(0) for _ in range(4)]
        self.lib.ckf_get_launch_info(self.handle, *[C.byref(x) for x in v])
        return dict(blocks=v[0].value, threads=v[1].value, smem_bytes=v[2].value, regs=v[3].value)

    def close(self):
        if getattr(self, "handle", None):
            self.lib.ckf_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
