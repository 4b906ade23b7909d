"""-m gpu: ckf_resolve_static, the entry point that allocates nothing (scratch in a static __device__ array of the
library, include/ckf.h), against the existing path ckf_resolve on the same candidates.  Integer work: the accepted flags,
the shared-hit counts and the summary must be identical.  Two calls in a row on DIFFERENT candidate sets and limits, so
that whatever the first call left in the shared array would show in the second.  Collected last on purpose (the suite
runs with pytest -x); passes alone in a fresh process and after the other GPU tests."""
import ctypes as C

import pytest

import synth

pytestmark = pytest.mark.gpu


def _find(config, n_particles, n_fake, event_index=0):
    import torch
    from paper_2505_22822_b200 import CKF
    det, fld, cfg = synth.config_bundle(config)
    ev = synth.make_event(config, event_index=event_index, det=det, n_particles=n_particles, n_fake_seeds=n_fake)
    ckf = CKF(det, fld, cfg.ckf, cfg.precision, max_seeds=ev.n_seeds, max_measurements=ev.n_measurements, max_fit_tracks=0)
    dev, out = ckf.upload_event(ev), ckf.alloc_tracks()
    ckf.find(dev, out)
    torch.cuda.synchronize()
    return ckf, ev, out, cfg.precision, int(out["n_tracks"][0])


def test_resolve_static_equals_resolve_on_two_calls_in_a_row():
    import torch
    from paper_2505_22822_b200 import binding as B
    cases = [_find(1, 1500, 1500), _find(2, 3000, 400, event_index=1)]       # fp64 uniform field, fp32 grid field
    limits = [(1, 1.0), (2, 0.25)]
    want = []
    for (ckf, ev, out, precision, n), lim in zip(cases, limits):
        assert 1000 < n and ckf.max_tracks <= B.RESOLVE_STATIC_MAX_TRACKS
        assert ev.n_measurements <= B.RESOLVE_STATIC_MAX_MEASUREMENTS
        ref = ckf.alloc_resolution()
        ckf.resolve(out, ev.n_measurements, ref, *lim)                        # the existing path: workspace of the handle
        torch.cuda.synchronize()
        want.append(ref)
        assert 0 < int(ref["summary"][0]) < n                                 # something is removed, something is kept
    # the new entry point: two calls in a row on one stream, then the same two in the other order (the array then holds
    # the LARGER problem's leftovers when the smaller one runs)
    for order in ((0, 1), (1, 0)):
        got = {}
        for i in order:
            ckf, ev, out, precision, n = cases[i]
            res = ckf.alloc_resolution()
            res["accepted"].fill_(-7)
            res["n_shared"].fill_(-7)
            B.resolve_static(out, ev.n_measurements, res, precision, *limits[i])
            got[i] = res
        torch.cuda.synchronize()
        for i in order:
            n = cases[i][4]
            assert torch.equal(got[i]["summary"], want[i]["summary"]), (order, i)
            assert torch.equal(got[i]["accepted"][:n], want[i]["accepted"][:n]), (order, i)
            assert torch.equal(got[i]["n_shared"][:n], want[i]["n_shared"][:n]), (order, i)
            assert bool((got[i]["accepted"][n:] == -7).all())                 # nothing beyond the candidates is written
    for c in cases:
        c[0].close()


def test_resolve_static_rejects_sizes_beyond_the_static_array():
    import torch
    from paper_2505_22822_b200 import binding as B
    lib = B.load_library()
    ckf, ev, out, precision, n = _find(1, 200, 0)
    res = ckf.alloc_resolution()
    with pytest.raises(RuntimeError, match="n_measurements .* outside"):
        B.resolve_static(out, B.RESOLVE_STATIC_MAX_MEASUREMENTS + 1, res, precision)
    o = B.ckf_tracks(*[out[k].data_ptr() for k in ("n_tracks", "status", "track_offsets", "meas_idx", "seed_id", "n_holes",
                                                   "last_module", "stop_reason", "params", "cov", "chi2_sum", "entry_chi2")])
    r = B.ckf_resolution(res["accepted"].data_ptr(), res["n_shared"].data_ptr(), res["summary"].data_ptr(), 1, 1.0)
    st = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    rc = lib.ckf_resolve_static(C.byref(o), B.RESOLVE_STATIC_MAX_TRACKS + 1, ev.n_measurements, precision, C.byref(r), st)
    assert rc == -3 and b"max_tracks" in lib.ckf_last_error(None) and b"use ckf_resolve" in lib.ckf_last_error(None)
    assert lib.ckf_resolve_static(C.byref(o), ckf.max_tracks, ev.n_measurements, 16, C.byref(r), st) == -1
    # and a call inside the limits still works afterwards
    B.resolve_static(out, ev.n_measurements, res, precision)
    ref = ckf.alloc_resolution()
    ckf.resolve(out, ev.n_measurements, ref)
    torch.cuda.synchronize()
    assert torch.equal(res["summary"], ref["summary"]) and torch.equal(res["accepted"][:n], ref["accepted"][:n])
    ckf.close()
