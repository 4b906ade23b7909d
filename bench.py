#!/usr/bin/env python
"""bench.py — CKF track-finding throughput on B200 (BASELINE.json metric: seeds/s on the 40k-particle event).

A step = one pass of the whole hot path (ckf_find: init, level loop, emission) over one synthetic event of
BASELINE.json configs[3] (40,000 particles + 4,000 fake seeds, fp32 arrays, grid field).  `value` is device
timed with the inputs resident in HBM; `e2e` goes through ckf_find_host with pinned HOST buffers on 4 streams
(H2D + D2H inside the timed region, the shape of configs[4]).  See DESIGN.md §7 for the roofline accounting.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import synth  # noqa: E402

CONFIG = 3
N_EVENTS = 4            # distinct events rotated through the timed loop (working set >> L2)
E2E_STREAMS = 4

# Algorithmic flops per unit of work (counted from the formulas of §3, not from SASS)
F_FIELD_GRID = 75       # one trilinear read
F_TRIAL = 108           # one RKN4 trial without the three field reads
F_ACCEPT = 500          # state update 50 + four Jacobian columns 450
F_NAV = 600             # navigation of one visit (ckf_step): ~1.7 module choices x 9 modules x 35 + targeting
F_VISIT = 1450          # navigation 600 + arrival Jacobian, covariance transport, bound parameters 850
F_GATE = 17             # one chi2 actually evaluated (inside a loc0 window)
F_UPDATE = 155          # one gain-form update
F_RTS = 1950            # one RTS step (ckf_fit_smooth): J Cf 300, scaled Cholesky 150, 6 column solves 430, gain products 1070
# plain-ALU peaks from the guide's unit counts: 148 SMs x 128 FP32 (64 FP64) lanes x 2 flop x 1.965 GHz
PEAK_FP32_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12
PEAK_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12


def algorithmic_flops(cnt: dict, grid_field: bool):
    """(total flop, flop the design computes in float64) for one launch, from the library's work counters."""
    f_trial = F_TRIAL + (3 * F_FIELD_GRID if grid_field else 0)
    traj = cnt["rk_trials"] * f_trial + cnt["rk_accepted"] * 50 + cnt["visits"] * 700   # float64 in both modes
    cov = cnt["rk_accepted"] * 450 + cnt["visits"] * 750 + cnt["gate_tests_executed"] * F_GATE + cnt["updates"] * F_UPDATE
    return float(traj + cov), float(traj)


def algorithmic_bytes(ev, n_tracks, n_entries, tsize):
    """Compulsory HBM bytes of one step: inputs read once, candidates written once."""
    inp = ev.n_measurements * 4 * tsize + (ev.module_offsets.size) * 4 + ev.n_seeds * (42 * tsize + 4)
    out = n_tracks * (43 * tsize + 5 * 4) + n_entries * (4 + tsize)
    return inp, out


class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index=0):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for ln in self.lines:
            p = [x.strip() for x in ln.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0]))
                mx.append(float(p[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), p[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def make_events(n, first_index=0):
    det, fld, cfg = synth.config_bundle(CONFIG)
    from concurrent.futures import ProcessPoolExecutor
    with ProcessPoolExecutor(max_workers=min(n, os.cpu_count() or 1)) as ex:
        evs = list(ex.map(_make_one, range(first_index, first_index + n)))
    return det, fld, cfg, evs


def _make_one(i):
    return synth.make_event(CONFIG, event_index=i)


def run_reference(args, rank, world):
    """--impl reference: the oracle as it stands, timed on the host cores (rank 0 only)."""
    if rank != 0:
        return
    import oracle
    det, fld, cfg = synth.config_bundle(CONFIG)
    ev = synth.make_event(CONFIG, det=det)
    st = oracle.Setup(det, fld, cfg.ckf)
    cores = os.cpu_count() or 1
    for _ in range(max(1, min(args.warmup, 1))):
        oracle.find_event(st, ev, n_threads=cores)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.find_event(st, ev, n_threads=cores)
    dt = time.perf_counter() - t0
    v = ev.n_seeds * args.steps / dt
    print(json.dumps({
        "impl": "reference", "metric": "CKF seeds/sec (40k-particle event)", "value": v, "unit": "seeds/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[3]: 40,000 particles + 4,000 fake seeds, 1 event, grid field", "seeds": ev.n_seeds,
                   "measurements": ev.n_measurements},
        "cpu_baseline": {"value": v, "unit": "seeds/s", "cores": cores, "kind": "oracle",
                         "sample": "the full configs[3] event per step, all host threads"},
        "e2e": {"value": v, "unit": "seeds/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--streams", type=int, default=2, help="batches kept in flight (CUDA streams) for `value`")
    ap.add_argument("--batch", type=int, default=4, help="independent events per ckf_find (one step = one batch)")
    ap.add_argument("--e2e-batch", type=int, default=4, help="events per ckf_find_host call of the e2e leg")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_2505_22822_b200 import CKF
    from paper_2505_22822_b200.dist import aggregate_throughput
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    # weak scaling: every rank owns its own events (events are independent: no data-path collective)
    det, fld, cfg, evs = make_events(N_EVENTS, first_index=rank * N_EVENTS)
    max_s = max(e.n_seeds for e in evs)
    max_m = max(e.n_measurements for e in evs)
    S = max(1, args.streams)
    B = max(1, min(args.batch, N_EVENTS))
    # one step = one ckf_find over a BATCH of B independent events (include/ckf.h, ckf_measurements.n_events): the
    # level loop then runs over the tips of all B events, which shares its per-level cost
    from paper_2505_22822_b200 import concat_events
    batches = [concat_events([evs[(i + j) % N_EVENTS] for j in range(B)], det.n_modules) for i in range(N_EVENTS)]
    ckf = CKF(det, fld, cfg.ckf, cfg.precision, max_seeds=B * max_s, max_measurements=B * max_m, max_tracks=8 * B * max_s,
              max_track_entries=80 * B * max_s, n_streams=max(S, E2E_STREAMS) + 1, max_events_per_find=B)
    devs = [ckf.upload_event(e) for e in evs]
    bdevs = [ckf.upload_event(b) for b in batches]
    stream = torch.cuda.current_stream()
    work = [torch.cuda.Stream() for _ in range(S)]
    outs = [ckf.alloc_tracks() for _ in range(S)]
    out = outs[0]

    # the K steps are independent batches, kept S at a time in flight on S CUDA streams (the paper's own throughput
    # mode: one event pipeline per stream)
    def run_steps(k):
        for i in range(k):
            ckf.find(bdevs[i % N_EVENTS], outs[i % S], work[i % S])

    W = max(3, args.warmup)
    ev_last = evs[(W - 1) % N_EVENTS]
    ckf.find(devs[(W - 1) % N_EVENTS], out, stream)  # that event alone: parity check and e2e byte counts below
    torch.cuda.synchronize()
    res1 = ckf.download(out)
    for i in range(W):
        ckf.find(bdevs[i % N_EVENTS], out, stream)
    torch.cuda.synchronize()
    cnt = ckf.counters(stream)                      # of batch (warmup-1) % N: the B events starting at ev_last
    res = ckf.download(out)
    run_steps(S)                                    # warm the per-stream workspaces
    torch.cuda.synchronize()

    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = torch.cuda.Event(enable_timing=True)
    t1 = torch.cuda.Event(enable_timing=True)
    t0.record(stream)
    for w in work:
        w.wait_stream(stream)
    run_steps(args.steps)
    for w in work:
        stream.wait_stream(w)
    t1.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ms_total = t0.elapsed_time(t1)
    seeds_done = sum(batches[i % N_EVENTS].n_seeds for i in range(args.steps))

    # single-event latency (one stream, finds back to back) and the per-kernel device times of the dominant
    # kernel, ckf_step, measured live with CUDA events on the launching stream (ckf_set_timing)
    per = []
    for i in range(min(args.steps, 8)):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        ckf.find(devs[i % N_EVENTS], out, stream)
        b.record(stream)
        torch.cuda.synchronize()
        per.append(a.elapsed_time(b))
    ckf.set_timing(True)
    tim = []
    for i in range(min(args.steps, 8)):
        ckf.find(bdevs[(W - 1) % N_EVENTS], out, stream)
        torch.cuda.synchronize()
        tim.append(ckf.timing(stream))
    ckf.set_timing(False)
    # ---- next row: KF fit + RTS smoother of that event's candidates (ckf_fit)
    fits = ckf.alloc_fits()
    dev_last = bdevs[(W - 1) % N_EVENTS]
    for _ in range(2):
        ckf.fit(dev_last, out, fits, stream)
    torch.cuda.synchronize()
    n_fit = 5
    fa, fb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    fa.record(stream)
    for _ in range(n_fit):
        ckf.fit(dev_last, out, fits, stream)
    fb.record(stream)
    torch.cuda.synchronize()
    fit_ms = fa.elapsed_time(fb) / n_fit
    fa.record(stream)
    for _ in range(n_fit):
        ckf.fit(dev_last, out, fits, stream, smoother=1)
    fb.record(stream)
    torch.cuda.synchronize()
    fit_tf_ms = fa.elapsed_time(fb) / n_fit
    ckf.fit(dev_last, out, fits, stream)            # leave the RTS result in `fits` for the counts below
    torch.cuda.synchronize()
    fit_ok = int((fits["status"][:res.n_tracks] == 0).sum().item())
    fit_work = [int(v) // (2 * n_fit + 3) for v in fits["work"].cpu().tolist()]   # trials, accepted, moves, updates per call
    fit_states = int(fits["n_states"][:res.n_tracks].sum().item())
    clocks = sampler.stop()
    launches_per_find = int(tim[0]["launches"])

    # ---- e2e: host buffers through ckf_find_host on 4 streams / 4 host threads (configs[4] shape)
    EB = max(1, min(args.e2e_batch, B))
    e2e_src = evs if EB == 1 else [concat_events([evs[(i + j) % N_EVENTS] for j in range(EB)], det.n_modules)
                                   for i in range(N_EVENTS)]
    hevs = [ckf.pinned_event(e) for e in e2e_src]
    houts = [ckf.pinned_tracks() for _ in range(E2E_STREAMS)]
    streams = [torch.cuda.Stream() for _ in range(E2E_STREAMS)]
    n_e2e = max(E2E_STREAMS * 2, min(args.steps, 16))

    def worker(k, lo, hi):
        torch.cuda.set_device(local)
        for i in range(lo, hi):
            ckf.find_host(hevs[i % N_EVENTS], houts[k], streams[k])

    def run_e2e(n):
        ths = [threading.Thread(target=worker, args=(k, k * n // E2E_STREAMS, (k + 1) * n // E2E_STREAMS))
               for k in range(E2E_STREAMS)]
        torch.cuda.synchronize()
        t = time.perf_counter()
        for th in ths:
            th.start()
        for th in ths:
            th.join()
        torch.cuda.synchronize()
        return time.perf_counter() - t

    run_e2e(E2E_STREAMS)
    dt_e2e = run_e2e(n_e2e)
    e2e_seeds = sum(e2e_src[i % N_EVENTS].n_seeds for i in range(n_e2e))
    tsize = 4 if cfg.precision == 32 else 8
    bi, bo = algorithmic_bytes(ev_last, res1.n_tracks, int(res1.meas_idx.size), tsize)

    value, ms_step = aggregate_throughput(seeds_done, ms_total, args.steps, world)
    e2e_value, _ = aggregate_throughput(e2e_seeds, dt_e2e * 1e3, n_e2e, world)

    if rank == 0:
        flop, flop64 = algorithmic_flops(cnt, grid_field=cfg.inhomogeneous)
        k_ms = float(np.mean(per))
        # dominant kernel: ckf_step (navigation + RKN4 trials + Jacobian columns), all its launches of one find
        step_ms = float(np.mean([t["step_ms"] for t in tim]))
        f_trial = F_TRIAL + (3 * F_FIELD_GRID if cfg.inhomogeneous else 0)
        step64 = cnt["rk_trials"] * f_trial + cnt["rk_accepted"] * 50 + cnt["visits"] * F_NAV
        step32 = cnt["rk_accepted"] * 450
        step_flop = float(step64 + step32)
        achieved = step_flop / (step_ms * 1e-3) / 1e12
        # serial-pipe peak for this kernel's fp32/fp64 mix
        f64_share = step64 / step_flop if cfg.precision == 32 else 1.0
        peak = 1.0 / (f64_share / PEAK_FP64_TFLOPS + (1.0 - f64_share) / PEAK_FP32_TFLOPS)
        step_launches = sum(1 for _ in range(cfg.ckf.max_levels))
        fit_flop = float(fit_work[0] * f_trial + fit_work[1] * F_ACCEPT + fit_work[2] * F_VISIT + fit_work[3] * F_UPDATE +
                         max(fit_states - res.n_tracks, 0) * F_RTS)
        line = {
            "metric": "CKF seeds/sec (40k-particle event)", "value": value, "unit": "seeds/s", "n_gpus": world,
            "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32 covariance/Jacobian + f64 trajectory",
            "data": "synthetic",
            "config": {"workload": "configs[3]: 40,000 particles + 4,000 fake seeds per event, %d independent events per "
                                   "step (one batched ckf_find), fp32 arrays, " % B +
                                   "float32 grid field, k=10, cap=100", "seeds_per_event": ev_last.n_seeds,
                       "measurements_per_event": ev_last.n_measurements, "distinct_events_rotated": N_EVENTS,
                       "l2": "4 events rotated; each step writes a >190 MB link buffer (> 126 MB L2)",
                       "events_per_step": B, "batches_in_flight": S,
                       "how": "K independent batches of B events, S at a time on S CUDA streams, device "
                       "timed from the first launch to the last completion", "launch": ckf.launch_info()},
            "latency_ms_single_event": k_ms, "seeds_per_s_single_stream": ev_last.n_seeds / (k_ms * 1e-3),
            "events_per_s": value / ev_last.n_seeds,
            "e2e": {"value": e2e_value, "unit": "seeds/s", "h2d_bytes_per_step": int(bi), "d2h_bytes_per_step": int(bo),
                    "streams": E2E_STREAMS, "calls": n_e2e, "events_per_call": EB, "events": n_e2e * EB, "events_per_s": e2e_value / ev_last.n_seeds,
                    "how": "ckf_find_host on batches of events_per_call events, pinned host buffers, 4 host threads x 4 CUDA "
                           "streams (configs[4]: 64 events over 4 streams), H2D and D2H inside, wall clock"},
            "fit": {"what": "ckf_fit: Kalman-filter fit + RTS smoother of every candidate of one step's batch of configs[3] "
                            "events (next row, SURVEY.md 8(f) rank 1); device-resident, CUDA events, mean of 5",
                    "value": res.n_tracks / (fit_ms * 1e-3), "unit": "tracks/s", "ms_per_event": fit_ms / B,
                    "ms_per_step": fit_ms, "ms_per_event_two_filter_smoother": fit_tf_ms / B,
                    "tracks": res.n_tracks, "fitted": fit_ok, "entries": int(res.meas_idx.size),
                    "work": dict(zip(("rk_trials", "rk_accepted", "moves", "updates"), fit_work)), "states": fit_states,
                    "flop_per_event": fit_flop, "achieved_tflops": fit_flop / (fit_ms * 1e-3) / 1e12,
                    "launches": "per pass of 262,144 candidates: ckf_step + ckf_fit_level per level, then ckf_fit_smooth"},
            "ms_per_event": ms_step / B,
            "gpu_launches": launches_per_find * args.steps,
            "clocks": clocks,
            "roofline": {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                         # DRAM bytes of ONE ckf_step launch (level 4 of a batched find of 4 events, ~360,000 tips), from the
                         # committed ncu --set full capture; only valid for the default batch of 4
                         "traffic": 139.1e6 if (B == 4 and cfg.precision == 32) else None,
                         "traffic_source": "profiles/r01i_step_and_launches.md: dram__bytes_read.sum + dram__bytes_write.sum "
                                           "of one ckf_step launch (level 4 of a batched find, ~360,000 tips); its algorithmic "
                                           "bytes (tip state in and out: 8 + 8 float64 and 25 float32 per tip) are 228 B x "
                                           "360,000 = 82 MB",
                         "kernel": "ckf_step (all %d launches of one find)" % step_launches,
                         "flop_per_find_this_kernel": step_flop, "kernel_ms_per_find": step_ms,
                         "share_of_find": step_ms / max(sum(v for k, v in tim[0].items() if k.endswith("_ms")), 1e-9),
                         "whole_path_flop_per_find": flop,
                         "whole_path_tflops": flop / max(sum(v for k, v in tim[0].items() if k.endswith("_ms")) * 1e-3, 1e-12) / 1e12,
                         "kernel_ms_by_phase": {k: float(np.mean([t[k] for t in tim])) for k in tim[0] if k.endswith("_ms")},
                         "fp64_share_of_flop": f64_share, "peak_fp32": PEAK_FP32_TFLOPS, "peak_fp64": PEAK_FP64_TFLOPS,
                         "peak_source": "derived from the guide's unit counts and max clock (DESIGN.md §7); "
                                        "MEASURED_PEAKS.json has no ALU peak",
                         "hbm_gbs_achieved": (bi + bo) / (k_ms * 1e-3) / 1e9,
                         "counters": cnt},
        }
        if not args.no_cpu_baseline:
            import oracle
            cores = os.cpu_count() or 1
            st = oracle.Setup(det, fld, cfg.ckf)
            t = time.perf_counter()
            ora = oracle.find_event(st, ev_last, n_threads=cores)
            dt = time.perf_counter() - t
            line["cpu_baseline"] = {"value": ev_last.n_seeds / dt, "unit": "seeds/s", "cores": cores, "kind": "oracle",
                                    "sample": "one full configs[3] event (%d seeds), %d host threads, %.2f s" %
                                              (ev_last.n_seeds, cores, dt)}
            line["parity_in_bench"] = {"n_tracks_gpu": res1.n_tracks, "n_tracks_oracle": ora.n_tracks,
                                       "index_lists_identical": bool(res1.n_tracks == ora.n_tracks and
                                                                     np.array_equal(res1.meas_idx, ora.meas_idx))}
        print(json.dumps(line))
    ckf.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
