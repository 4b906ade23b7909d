"""Timing report of ckf_find on one synthetic event: `python -m paper_2505_22822_b200.probe --config 3`.

For a user who wants to know where the time of a find goes on their GPU: the median device time of repeated finds
(CUDA events on the launching stream), the per-kernel breakdown of one find (ckf_set_timing: an event after every
launch, so every launch carries a few microseconds of bracketing), and the work counters.  The tables of
profiles/r02_launch_overlap.md and profiles/r02_latency_floor.md are printed by this module.  Environment switches read
by ckf_create apply: CKF_CHAIN_OVERLAP=<mask> (which kernels are launched with programmatic stream serialisation),
CKF_GRAPH=1 (replay a find that repeats the previous call's arguments from a CUDA graph).  Needs a CUDA device; inputs are synthetic (synth/)."""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs[i] recipe (0-3)")
    ap.add_argument("--particles", type=int, default=None, help="override the number of particles (seeds)")
    ap.add_argument("--fake-seeds", type=int, default=None, help="override the number of fake seeds")
    ap.add_argument("--batch", type=int, default=1, help="independent events per ckf_find")
    ap.add_argument("--calls", type=int, default=15, help="timed finds (median / min reported)")
    ap.add_argument("--alternate", action="store_true",
                    help="alternate between two events of different sizes, so that no call repeats the previous one's "
                         "arguments (with CKF_GRAPH=1 a repeated call is replayed from a CUDA graph; this avoids it)")
    args = ap.parse_args(argv)
    import torch
    import synth
    from . import CKF, concat_events

    det, fld, cfg = synth.config_bundle(args.config)
    n_ev = args.batch * (2 if args.alternate else 1)
    evs = [synth.make_event(args.config, event_index=i, det=det, n_particles=args.particles, n_fake_seeds=args.fake_seeds)
           for i in range(n_ev)]
    if args.batch > 1:
        evs = [concat_events(evs[k * args.batch:(k + 1) * args.batch], det.n_modules) for k in range(n_ev // args.batch)]
    ms, mm = max(e.n_seeds for e in evs), max(e.n_measurements for e in evs)
    ckf = CKF(det, fld, cfg.ckf, cfg.precision, max_seeds=max(1, ms), max_measurements=max(1, mm), max_fit_tracks=0,
              max_events_per_find=args.batch, max_tracks=8 * max(1, ms), max_track_entries=80 * max(1, ms))
    devs = [ckf.upload_event(e) for e in evs]
    out = ckf.alloc_tracks()
    for i in range(4):
        ckf.find(devs[i % len(devs)], out)
    torch.cuda.synchronize()
    ts = []
    for i in range(args.calls):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        ckf.find(devs[i % len(devs)], out)
        b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    ckf.set_timing(True)
    ckf.find(devs[0], out)
    torch.cuda.synchronize()
    t = ckf.timing()
    ckf.set_timing(False)
    cnt = ckf.counters()
    live = max(1, cnt["iterations"])
    rep = {"config": args.config, "events_per_find": args.batch, "seeds": int(evs[0].n_seeds),
           "measurements": int(evs[0].n_measurements), "candidates": int(out["n_tracks"][0]),
           "find_ms_median": float(np.median(ts)), "find_ms_min": float(min(ts)),
           "call_pattern": "alternating arguments" if args.alternate else "repeated arguments",
           "per_kernel_ms_timing_mode": {k: round(v, 4) for k, v in t.items() if k.endswith("_ms")},
           "launches_per_find": int(t["launches"]), "live_levels": int(cnt["iterations"]), "tips": cnt["tips"],
           "rk_trials": cnt["rk_trials"], "rk_trials_per_tip": cnt["rk_trials"] / max(1, cnt["tips"]),
           "ckf_step_us_per_live_level": 1e3 * t["step_ms"] / live,
           "env": {k: os.environ.get(k) for k in ("CKF_CHAIN_OVERLAP", "CKF_GRAPH") if os.environ.get(k) is not None}}
    print(json.dumps(rep))
    ckf.close()
    return rep


if __name__ == "__main__":
    main()
