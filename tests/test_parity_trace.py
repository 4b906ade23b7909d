"""CPU test of the mismatch tracer used by the fp32 parity tests (tests/parity.py): gate-edge differences are
explained, a fabricated difference is not."""
import copy

import numpy as np

import oracle
import synth
from tests import parity


def test_gate_edge_mismatches_are_traced_and_fabricated_ones_are_not():
    det, fld, cfg = synth.config_bundle(1)
    ev = synth.make_event(1, det=det, n_particles=1500)
    a = oracle.find_event(oracle.Setup(det, fld, cfg.ckf), ev, n_threads=8)
    ckf2 = copy.copy(cfg.ckf)
    ckf2.chi2_max = cfg.ckf.chi2_max + 0.6
    b = oracle.find_event(oracle.Setup(det, fld, ckf2), ev, n_threads=8)
    r = parity.compare_fp32(a, b, ev.n_seeds)
    assert len(r["bad_seeds"]) >= 1                       # a 0.6-wide band at the gate does catch a few hits
    traced = parity.trace_mismatches(a, b, r["bad_seeds"], cfg.ckf.chi2_max, tol=0.65)
    assert all(why is not None for _, why in traced), traced
    # the same mismatches are NOT explained at the real tolerance unless they sit within 1e-3 of the gate
    tight = parity.trace_mismatches(a, b, r["bad_seeds"], cfg.ckf.chi2_max, tol=1e-3)
    assert any(why is None for _, why in tight)
    # a fabricated discrepancy: one candidate's last measurement replaced -- nothing near the gate, no tie
    c = copy.deepcopy(a)
    t = int(np.argmax((a.track_offsets[1:] - a.track_offsets[:-1]) >= 8))
    e = int(a.track_offsets[t + 1]) - 1
    assert abs(a.entry_chi2[e] - cfg.ckf.chi2_max) > 0.5
    c.meas_idx[e] += 1
    c.entry_chi2[e] += 1.5 if a.entry_chi2[e] < 8.0 else -1.5
    r2 = parity.compare_fp32(c, a, ev.n_seeds)
    assert r2["bad_seeds"] == [int(a.seed_id[t])]
    tr2 = parity.trace_mismatches(c, a, r2["bad_seeds"], cfg.ckf.chi2_max)
    assert tr2[0][1] is None
