#!/usr/bin/env python
"""bench.py — CKF track-finding throughput on B200 (BASELINE.json metric: seeds/s on the 40k-particle event).

A step = one pass of the whole hot path (ckf_find: init, gate index, level loop, emission) over ONE synthetic event of
BASELINE.json configs[3] (40,000 particles + 4,000 fake seeds, fp32 arrays, float32 grid field), inputs resident in HBM.
`value` is SURVEY.md 8(d)'s quantity: seeds of the event / MEDIAN device time of the K timed single ckf_find calls
(CUDA events on the launching stream; min and mean beside it).  Further blocks of the same line:
  throughput_batched  events kept in flight (batches of B events per ckf_find, S batches on S streams)
  e2e                 BASELINE.json configs[4]: 64 DISTINCT events through ckf_find_host, pinned host buffers, 4 host
                      threads x 4 CUDA streams, H2D + D2H inside, wall clock
  roofline            the dominant kernel (ckf_step) against the MEASURED plain-ALU peak (ckf_measure_alu_peak)
  fit                 ckf_fit (KF fit + RTS smoother) on the candidates of one event
  cpu_baseline        the oracle as it stands on the host cores (a baseline, not the target)
See DESIGN.md 7 for the accounting.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
"""
from __future__ import annotations

import argparse
import csv
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
N_EVENTS = 4            # distinct events rotated through the timed single-event loop (working set >> L2)
E2E_EVENTS = 64         # configs[4]: 64 distinct events
E2E_STREAMS = 4

# Algorithmic flops per unit of work (counted from the formulas of 3, an FMA = 2)
F_FIELD_GRID = 75       # one trilinear read
F_TRIAL = 108           # one RKN4 trial without the three field reads
F_ACCEPT = 500          # state update 50 + four Jacobian columns 450
F_NAV = 600             # navigation of one visit (ckf_step): ~1.7 module choices x 9 modules x 35 + targeting
F_VISIT = 1450          # navigation 600 + arrival Jacobian, covariance transport, bound parameters 850
F_GATE = 17             # one chi2 actually evaluated (inside a loc0 window)
F_UPDATE = 155          # one gain-form update
F_RTS = 1950            # one RTS step (ckf_fit_smooth)
# nominal plain-ALU peaks (148 SMs x 128 FP32 / 64 FP64 lanes x 2 flop x 1.965 GHz): context beside the measured ones
NOMINAL_FP32_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12
NOMINAL_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
DRAM_PROFILE = os.path.join(ROOT, "profiles", "r02_find_dram_per_launch.csv")


def algorithmic_flops(cnt: dict, grid_field: bool):
    """(total flop, flop the design computes in float64) of one ckf_find, from the library's work counters.  Since r02
    the arrival algebra, J C J^T, the gate's final evaluation and the update are float64 in both modes; float32 is the
    25-number transport Jacobian (450 flop per accepted step) and the chi2 pre-filter."""
    f_trial = F_TRIAL + (3 * F_FIELD_GRID if grid_field else 0)
    f64 = cnt["rk_trials"] * f_trial + cnt["rk_accepted"] * 50 + cnt["visits"] * F_VISIT + cnt["updates"] * F_UPDATE
    f32 = cnt["rk_accepted"] * 450 + cnt["gate_tests_executed"] * F_GATE
    return float(f64 + f32), float(f64)


def step_kernel_flops(cnt: dict, grid_field: bool):
    """Algorithmic flop of ckf_step alone (navigation + RKN4 trials + Jacobian columns): (float64, float32)."""
    f_trial = F_TRIAL + (3 * F_FIELD_GRID if grid_field else 0)
    return (float(cnt["rk_trials"] * f_trial + cnt["rk_accepted"] * 50 + cnt["visits"] * F_NAV),
            float(cnt["rk_accepted"] * 450))


def event_bytes(ev, tsize):
    """Input bytes of one event as ckf_find_host copies them host -> device."""
    return ev.n_measurements * 4 * tsize + ev.module_offsets.size * 4 + ev.n_seeds * (42 * tsize + 4)


def result_bytes(n_tracks, n_entries, tsize):
    """Candidate bytes of one result (device -> host): 5 int32 + 43 T per track, (int32 + T) per entry, + 2 int32."""
    return n_tracks * (43 * tsize + 5 * 4) + 4 + n_entries * (4 + tsize) + 8


def dram_traffic_from_profile(kernel_prefix="ckf_step"):
    """DRAM bytes (read + write) of all launches of `kernel_prefix` in ONE single-event ckf_find of configs[3], summed
    from the committed ncu launch list (profiles/r02_find_dram_per_launch.md names the command).  None if absent."""
    if not os.path.exists(DRAM_PROFILE):
        return None, None
    tot_k = tot_all = 0.0
    with open(DRAM_PROFILE) as f:
        rows = [r for r in csv.reader(f) if r]
    hdr = next((r for r in rows if "Kernel Name" in r and "Metric Name" in r), None)
    if hdr is None:
        return None, None
    ik, im, iv, iu = hdr.index("Kernel Name"), hdr.index("Metric Name"), hdr.index("Metric Value"), hdr.index("Metric Unit")
    for r in rows:
        if len(r) <= max(ik, im, iv) or r is hdr or not r[im].startswith("dram__bytes_"):
            continue
        try:
            v = float(r[iv].replace(",", ""))
        except ValueError:
            continue
        v *= {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(r[iu], 1.0)
        tot_all += v
        if kernel_prefix in r[ik]:
            tot_k += v
    return (tot_k or None), (tot_all or None)


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
        sm, mx, pw, reasons = [], [], [], set()
        for ln in self.lines:
            p = [x.strip() for x in ln.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0]))
                mx.append(float(p[1]))
                pw.append(float(p[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), p[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "reasons": sorted(reasons), "samples": len(sm)}


def _make_one(args):
    cfg, i = args
    return synth.make_event(cfg, event_index=i)


def make_events(config, indices):
    from concurrent.futures import ProcessPoolExecutor
    with ProcessPoolExecutor(max_workers=min(len(indices), os.cpu_count() or 1)) as ex:
        return list(ex.map(_make_one, [(config, i) for i in indices]))


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
    ts = []
    for _ in range(args.steps):
        t0 = time.perf_counter()
        oracle.find_event(st, ev, n_threads=cores)
        ts.append(time.perf_counter() - t0)
    dt = float(np.median(ts))
    v = ev.n_seeds / dt
    print(json.dumps({
        "impl": "reference", "metric": "CKF seeds/sec (40k-particle event)", "value": v, "unit": "seeds/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[3]: 40,000 particles + 4,000 fake seeds, 1 event, grid field", "seeds": ev.n_seeds,
                   "measurements": ev.n_measurements},
        "cpu_baseline": {"value": v, "unit": "seeds/s", "cores": cores, "kind": "oracle",
                         "sample": "the full configs[3] event per step, all host threads, median of the steps"},
        "e2e": {"value": v, "unit": "seeds/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--streams", type=int, default=2, help="throughput_batched: batches kept in flight (CUDA streams)")
    ap.add_argument("--batch", type=int, default=4, help="throughput_batched: independent events per ckf_find")
    ap.add_argument("--e2e-batch", type=int, default=4, help="events per ckf_find_host call of the e2e leg's batched run")
    ap.add_argument("--e2e-events", type=int, default=E2E_EVENTS)
    ap.add_argument("--peak-seconds", type=float, default=1.0, help="duration of each ALU-peak measurement")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_2505_22822_b200 import CKF, concat_events, measure_alu_peak
    from paper_2505_22822_b200.dist import aggregate_throughput
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    # weak scaling: every rank owns its own events (events are independent: no data-path collective)
    det, fld, cfg = synth.config_bundle(CONFIG)
    n_e2e_ev = 0 if args.no_e2e else max(E2E_STREAMS, args.e2e_events)
    n_gen = max(N_EVENTS, n_e2e_ev)
    all_evs = make_events(4 if n_e2e_ev else CONFIG, [rank * n_gen + i for i in range(n_gen)])   # configs[4] = configs[3]'s recipe
    evs = all_evs[:N_EVENTS]
    max_s = max(e.n_seeds for e in all_evs)
    max_m = max(e.n_measurements for e in all_evs)
    S = max(1, args.streams)
    B = max(1, min(args.batch, N_EVENTS))
    EB = max(1, min(args.e2e_batch, B))
    batches = [concat_events([evs[(i + j) % N_EVENTS] for j in range(B)], det.n_modules) for i in range(N_EVENTS)]
    ckf = CKF(det, fld, cfg.ckf, cfg.precision, max_seeds=B * max_s, max_measurements=B * max_m, max_tracks=8 * B * max_s,
              max_track_entries=80 * B * max_s, n_streams=max(S, E2E_STREAMS) + 1, max_events_per_find=B)
    devs = [ckf.upload_event(e) for e in evs]
    bdevs = [ckf.upload_event(b) for b in batches]
    stream = torch.cuda.current_stream()
    out = ckf.alloc_tracks()
    tsize = 4 if cfg.precision == 32 else 8
    W = max(3, args.warmup)

    # ---- warm-up (W single-event finds), result and counters of the event the parity check below uses
    for i in range(W):
        ckf.find(devs[i % N_EVENTS], out, stream)
    torch.cuda.synchronize()
    ev_chk = evs[(W - 1) % N_EVENTS]
    res1 = ckf.download(out)
    cnt1 = ckf.counters(stream)

    # ---- ALU peak, measured (the roofline denominator) -- before the timed region so the clocks are warm
    peak32 = measure_alu_peak(0, args.peak_seconds)
    peak64 = measure_alu_peak(1, args.peak_seconds)
    peakmix = measure_alu_peak(2, max(0.25, args.peak_seconds / 2))

    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()

    # ---- `value`: K single-event ckf_find calls back to back on one stream, each bracketed by CUDA events
    marks = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    marks[0].record(stream)
    for i in range(args.steps):
        ckf.find(devs[i % N_EVENTS], out, stream)
        marks[i + 1].record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    per = np.array([marks[i].elapsed_time(marks[i + 1]) for i in range(args.steps)])
    ms_total = marks[0].elapsed_time(marks[-1])
    seeds_per_step = float(np.mean([evs[i % N_EVENTS].n_seeds for i in range(args.steps)]))
    med_ms, min_ms, mean_ms = float(np.median(per)), float(per.min()), float(ms_total / args.steps)
    clocks = sampler.stop()
    value, _ = aggregate_throughput(seeds_per_step, med_ms, 1, world)

    # ---- per-kernel device times of one single-event find (ckf_set_timing: an event after every launch)
    ckf.set_timing(True)
    tim = []
    for i in range(8):
        ckf.find(devs[(W - 1) % N_EVENTS], out, stream)
        torch.cuda.synchronize()
        tim.append(ckf.timing(stream))
    ckf.set_timing(False)
    launches_per_find = int(tim[0]["launches"])
    phase_ms = {k: float(np.median([t[k] for t in tim])) for k in tim[0] if k.endswith("_ms")}

    # ---- throughput_batched: K batches of B events, S at a time on S streams (events are independent)
    work = [torch.cuda.Stream() for _ in range(S)]
    outs = [ckf.alloc_tracks() for _ in range(S)]

    def run_batches(k):
        for i in range(k):
            ckf.find(bdevs[i % N_EVENTS], outs[i % S], work[i % S])

    run_batches(2 * S)
    torch.cuda.synchronize()
    cntb = ckf.counters(work[(2 * S - 1) % S])
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record(stream)
    for w in work:
        w.wait_stream(stream)
    run_batches(args.steps)
    for w in work:
        stream.wait_stream(w)
    t1.record(stream)
    torch.cuda.synchronize()
    ms_batched = t0.elapsed_time(t1)
    seeds_batched = sum(batches[i % N_EVENTS].n_seeds for i in range(args.steps))
    ckf.set_timing(True)
    timb = []
    for i in range(4):
        ckf.find(bdevs[0], outs[0], stream)
        torch.cuda.synchronize()
        timb.append(ckf.timing(stream))
    ckf.set_timing(False)
    bphase_ms = {k: float(np.median([t[k] for t in timb])) for k in timb[0] if k.endswith("_ms")}
    torch.cuda.synchronize()
    cntb = ckf.counters(stream)

    # ---- next row: KF fit + RTS smoother of one event's candidates (ckf_fit)
    ckf.find(devs[(W - 1) % N_EVENTS], out, stream)
    fits = ckf.alloc_fits()
    for _ in range(2):
        ckf.fit(devs[(W - 1) % N_EVENTS], out, fits, stream, n_tracks_upper=res1.n_tracks)
    torch.cuda.synchronize()
    n_fit = 5
    fa, fb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    fa.record(stream)
    for _ in range(n_fit):
        ckf.fit(devs[(W - 1) % N_EVENTS], out, fits, stream, n_tracks_upper=res1.n_tracks)
    fb.record(stream)
    torch.cuda.synchronize()
    fit_ms = fa.elapsed_time(fb) / n_fit
    fa.record(stream)
    for _ in range(n_fit):
        ckf.fit(devs[(W - 1) % N_EVENTS], out, fits, stream, smoother=1, n_tracks_upper=res1.n_tracks)
    fb.record(stream)
    torch.cuda.synchronize()
    fit_tf_ms = fa.elapsed_time(fb) / n_fit
    ckf.fit(devs[(W - 1) % N_EVENTS], out, fits, stream, n_tracks_upper=res1.n_tracks)       # leave the RTS result in `fits` for the counts below
    torch.cuda.synchronize()
    fit_ok = int((fits["status"][:res1.n_tracks] == 0).sum().item())
    fit_work = [int(v) // (2 * n_fit + 3) for v in fits["work"].cpu().tolist()]   # trials, accepted, moves, updates per call
    fit_states = int(fits["n_states"][:res1.n_tracks].sum().item())

    # ---- row f4: shared-hit ambiguity resolution of the same candidates (ckf_resolve)
    ckf.find(devs[(W - 1) % N_EVENTS], out, stream)
    reso = ckf.alloc_resolution()
    ckf.resolve(out, ev_chk.n_measurements, reso, 1, 1.0, stream)
    torch.cuda.synchronize()
    fa.record(stream)
    for _ in range(n_fit):
        ckf.resolve(out, ev_chk.n_measurements, reso, 1, 1.0, stream)
    fb.record(stream)
    torch.cuda.synchronize()
    resolve_ms = fa.elapsed_time(fb) / n_fit
    resolve_kept, resolve_rounds = [int(v) for v in reso["summary"].cpu()]

    # ---- e2e = BASELINE.json configs[4]: 64 distinct events, pinned host buffers, 4 host threads x 4 streams
    e2e = None
    if n_e2e_ev:
        e_evs = all_evs[:n_e2e_ev]
        streams = [torch.cuda.Stream() for _ in range(E2E_STREAMS)]
        houts = [ckf.pinned_tracks() for _ in range(E2E_STREAMS)]

        def run_e2e(hevs, n_calls):
            d2h = [0] * E2E_STREAMS

            def worker(k):
                torch.cuda.set_device(local)
                for i in range(k, n_calls, E2E_STREAMS):
                    ckf.find_host(hevs[i % len(hevs)], houts[k], streams[k])
                    nt = int(houts[k]["n_tracks"][0])
                    d2h[k] += result_bytes(nt, int(houts[k]["track_offsets"][nt]) if nt else 0, tsize)

            ths = [threading.Thread(target=worker, args=(k,)) for k in range(E2E_STREAMS)]
            torch.cuda.synchronize()
            t = time.perf_counter()
            for th in ths:
                th.start()
            for th in ths:
                th.join()
            torch.cuda.synchronize()
            return time.perf_counter() - t, sum(d2h)

        # (a) as configs[4] words it: one event per call
        hev1 = [ckf.pinned_event(e) for e in e_evs]
        run_e2e(hev1[:2 * E2E_STREAMS], 2 * E2E_STREAMS)
        dt1, d2h1 = run_e2e(hev1, len(hev1))
        # (b) the same 64 events as ckf_find_host calls of EB batched events
        nb = len(e_evs) // EB
        hevb = [ckf.pinned_event(concat_events(e_evs[i * EB:(i + 1) * EB], det.n_modules)) for i in range(nb)]
        run_e2e(hevb[:E2E_STREAMS], E2E_STREAMS)
        dtb, d2hb = run_e2e(hevb, nb)
        seeds1 = sum(e.n_seeds for e in e_evs)
        seedsb = sum(e.n_seeds for e in e_evs[:nb * EB])
        h2d = sum(event_bytes(e, tsize) for e in e_evs)
        v1, _ = aggregate_throughput(seeds1, dt1 * 1e3, 1, world)
        vb, _ = aggregate_throughput(seedsb, dtb * 1e3, 1, world)
        best_b = vb >= v1
        e2e = {"value": vb if best_b else v1, "unit": "seeds/s",
               "h2d_bytes_per_step": int(h2d / len(e_evs)), "d2h_bytes_per_step": int((d2hb if best_b else d2h1) / len(e_evs)),
               "bytes_are": "per event (a step of `value` is one event): inputs copied host->device and candidates copied "
                            "device->host, counted from the tensors; the library copies up to 1/8 more (size guess)",
               "events": len(e_evs), "distinct_events": len(e_evs), "streams": E2E_STREAMS, "host_threads": E2E_STREAMS,
               "events_per_s": (vb if best_b else v1) / (seeds1 / len(e_evs)),
               "events_per_call": EB if best_b else 1,
               "single_event_calls": {"seeds_per_s": v1, "events_per_s": len(e_evs) / dt1 * world, "wall_s": dt1, "calls": len(hev1)},
               "batched_calls": {"seeds_per_s": vb, "events_per_s": nb * EB / dtb * world, "wall_s": dtb, "calls": nb,
                                 "events_per_call": EB},
               "how": "BASELINE.json configs[4]: 64 distinct events (event_index 0..63) through ckf_find_host, pinned host "
                      "buffers, 4 host threads x 4 CUDA streams, H2D and D2H inside the timed region, wall clock"}

    if rank == 0:
        grid = bool(cfg.inhomogeneous)
        flop, flop64 = algorithmic_flops(cnt1, grid)
        s64, s32 = step_kernel_flops(cnt1, grid)
        step_ms = phase_ms["step_ms"]
        achieved = (s64 + s32) / (step_ms * 1e-3) / 1e12
        f64_share = s64 / (s64 + s32)
        p32, p64 = peak32["tflops_f32"], peak64["tflops_f64"]
        peak = 1.0 / (f64_share / p64 + (1.0 - f64_share) / p32)      # pipes assumed serial: conservative
        find_ms = sum(phase_ms.values())
        b64, b32 = step_kernel_flops(cntb, grid)
        bstep_ms = bphase_ms["step_ms"]
        traffic_step, traffic_find = dram_traffic_from_profile()
        bi = event_bytes(ev_chk, tsize)
        bo = result_bytes(res1.n_tracks, int(res1.meas_idx.size), tsize)
        f_trial = F_TRIAL + (3 * F_FIELD_GRID if grid else 0)
        fit_flop = float(fit_work[0] * f_trial + fit_work[1] * F_ACCEPT + fit_work[2] * F_VISIT + fit_work[3] * F_UPDATE +
                         max(fit_states - res1.n_tracks, 0) * F_RTS)
        line = {
            "metric": "CKF seeds/sec (40k-particle event)", "value": value, "unit": "seeds/s", "n_gpus": world,
            "steps": args.steps, "warmup": W, "ms_per_step": med_ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64 trajectory + covariance, f32 transport Jacobian, f32 I/O arrays",
            "data": "synthetic",
            "config": {"workload": "configs[3]: 40,000 particles + 4,000 fake seeds, ONE event per step (one ckf_find), fp32 "
                                   "arrays, float32 grid field, k=10, cap=100", "seeds_per_event": ev_chk.n_seeds,
                       "measurements_per_event": ev_chk.n_measurements, "distinct_events_rotated": N_EVENTS,
                       "l2": "4 events rotated; each find writes a > 300 MB link buffer (> 126 MB L2)",
                       "how": "SURVEY.md 8(d): seeds / MEDIAN device time of the K timed single ckf_find calls, CUDA events "
                              "on the launching stream", "launch": ckf.launch_info()},
            "value_is": "median", "ms_per_step_min": min_ms, "ms_per_step_mean": mean_ms,
            "seeds_per_s_at_min": seeds_per_step / (min_ms * 1e-3) * world, "events_per_s": value / seeds_per_step,
            "throughput_batched": {"events_per_step": B, "batches_in_flight": S, "steps": args.steps,
                                   "seeds_per_s": seeds_batched / (ms_batched * 1e-3) * world,
                                   "events_per_s": seeds_batched / (ms_batched * 1e-3) / seeds_per_step * world,
                                   "ms_per_event": ms_batched / args.steps / B,
                                   "ckf_step": {"kernel_ms_per_find": bstep_ms, "tflops": (b64 + b32) / (bstep_ms * 1e-3) / 1e12,
                                                "frac_of_measured_peak": (b64 + b32) / (bstep_ms * 1e-3) / 1e12 /
                                                                         (1.0 / ((b64 / (b64 + b32)) / p64 + (b32 / (b64 + b32)) / p32))},
                                   "kernel_ms_by_phase": bphase_ms,
                                   "how": "K batched ckf_find calls of B independent events, S at a time on S CUDA streams, "
                                          "device time from the first launch to the last completion"},
            "fit": {"what": "ckf_fit: Kalman-filter fit + RTS smoother of every candidate of ONE configs[3] event (next row, "
                            "SURVEY.md 8(f) rank 1); device-resident, CUDA events, mean of 5",
                    "value": res1.n_tracks / (fit_ms * 1e-3), "unit": "tracks/s", "ms_per_event": fit_ms,
                    "ms_per_event_two_filter_smoother": fit_tf_ms, "tracks": res1.n_tracks, "fitted": fit_ok,
                    "entries": int(res1.meas_idx.size), "states": fit_states,
                    "work_per_event": dict(zip(("rk_trials", "rk_accepted", "moves", "updates"), fit_work)),
                    "flop_per_event": fit_flop, "achieved_tflops": fit_flop / (fit_ms * 1e-3) / 1e12,
                    "launches_per_call": "per pass of <= 262,144 candidates: 4 memsets + (ckf_step + ckf_fit_level) per level "
                                         "(max_levels = %d) + 2; passes bounded by the host hint n_tracks_upper (one "
                                         "pass here)" % cfg.ckf.max_levels},
            "resolve": {"what": "ckf_resolve: greedy shared-hit ambiguity resolution (PAPER.md:98, rules AR1-AR3) of ONE "
                                "configs[3] event's candidates, max_shared_hits = 1; one cooperative launch",
                        "ms_per_event": resolve_ms, "candidates": res1.n_tracks, "kept": resolve_kept,
                        "rounds": resolve_rounds, "value": res1.n_tracks / (resolve_ms * 1e-3), "unit": "candidates/s"},
            "gpu_launches": launches_per_find * args.steps,
            "gpu_launches_per_find": launches_per_find,
            "clocks": clocks,
            "roofline": {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                         "traffic": traffic_step,
                         "traffic_source": "profiles/r02_find_dram_per_launch.csv: dram__bytes_read.sum + dram__bytes_write.sum "
                                           "summed over the ckf_step launches of one single-event configs[3] ckf_find "
                                           "(ncu, one pass per launch)" if traffic_step else None,
                         "traffic_whole_find": traffic_find, "compulsory_bytes_per_find": int(bi + bo),
                         "kernel": "ckf_step (all %d launches of one single-event find)" % cfg.ckf.max_levels,
                         "flop_per_find_this_kernel": s64 + s32, "kernel_ms_per_find": step_ms,
                         "share_of_find": step_ms / max(find_ms, 1e-9),
                         "whole_path_flop_per_find": flop, "whole_path_tflops": flop / max(find_ms * 1e-3, 1e-12) / 1e12,
                         "kernel_ms_by_phase": phase_ms,
                         "fp64_share_of_flop": f64_share, "peak_fp32": p32, "peak_fp64": p64,
                         "peak_source": "measured: ckf_measure_alu_peak (FMA chains in registers, all SMs, %.1f s each, run "
                                        "average); mix peak = 1 / (f64_share / fp64 + (1 - f64_share) / fp32)" % args.peak_seconds,
                         "peak_measured": {"fp32_only": peak32, "fp64_only": peak64, "fp32_and_fp64_together": peakmix},
                         "peak_nominal": {"fp32": NOMINAL_FP32_TFLOPS, "fp64": NOMINAL_FP64_TFLOPS,
                                          "what": "148 SMs x 128 / 64 lanes x 2 x 1.965 GHz"},
                         "hbm_gbs_achieved": (bi + bo) / (med_ms * 1e-3) / 1e9,
                         "counters": cnt1},
        }
        if e2e is not None:
            line["e2e"] = e2e
        if not args.no_cpu_baseline:
            import oracle
            cores = os.cpu_count() or 1
            st = oracle.Setup(det, fld, cfg.ckf)
            t = time.perf_counter()
            ora = oracle.find_event(st, ev_chk, n_threads=cores)
            dt = time.perf_counter() - t
            line["cpu_baseline"] = {"value": ev_chk.n_seeds / dt, "unit": "seeds/s", "cores": cores, "kind": "oracle",
                                    "sample": "one full configs[3]-recipe event (%d seeds), %d host threads, %.2f s" %
                                              (ev_chk.n_seeds, cores, dt)}
            line["parity_in_bench"] = {"n_tracks_gpu": res1.n_tracks, "n_tracks_oracle": ora.n_tracks,
                                       "index_lists_identical": bool(res1.n_tracks == ora.n_tracks and
                                                                     np.array_equal(res1.meas_idx, ora.meas_idx)),
                                       "max_entry_chi2_abs_diff": float(np.max(np.abs(res1.entry_chi2 - ora.entry_chi2)))
                                       if res1.n_tracks == ora.n_tracks and res1.meas_idx.size == ora.meas_idx.size else None}
        print(json.dumps(line))
    ckf.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
