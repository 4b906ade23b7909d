"""Comparison of CUDA-path candidates with the oracle's (metric definitions: Table 1 caption —
patterns match iff all measurements are identical; parameters by maximum relative difference; A15)."""
import numpy as np

FLOOR = np.array([1.0, 1.0, 1.0, 1.0, 0.0, 1.0])   # mm, mm, rad, rad, (none for q/p), mm


def param_rel_diff(a, b, qop_floor=0.0):
    """A15: |a-b| / max(|a|, |b|, floor); angles compared after wrapping the difference.  qop_floor: a floor for q/p
    (A15 has none: the workloads' |q/p| >= 0.0126 / GeV; seeds ESTIMATED from fake triplets can be straight lines)."""
    d = a - b
    d[..., 2] = (d[..., 2] + np.pi) % (2 * np.pi) - np.pi
    floor = FLOOR.copy()
    floor[4] = qop_floor
    den = np.maximum(np.maximum(np.abs(a), np.abs(b)), floor)
    den = np.where(den == 0.0, 1.0, den)     # both exactly zero (q/p has no floor): difference 0
    return np.abs(d) / den


def assert_bit_exact_lists(gpu, ora):
    assert gpu.n_tracks == ora.n_tracks, (gpu.n_tracks, ora.n_tracks)
    assert np.array_equal(gpu.seed_id, ora.seed_id)
    assert np.array_equal(gpu.track_offsets, ora.track_offsets)
    assert np.array_equal(gpu.meas_idx, ora.meas_idx)
    assert np.array_equal(gpu.n_holes, ora.n_holes)
    assert np.array_equal(gpu.stop_reason, ora.stop_reason)
    assert np.array_equal(gpu.last_module, ora.last_module)


def max_param_diffs(gpu, ora):
    rel = param_rel_diff(gpu.params.copy(), ora.params.copy())
    chi2 = np.abs(gpu.chi2_sum - ora.chi2_sum)
    scale = np.sqrt(np.abs(ora.cov[:, [0, 7, 14, 21, 28, 35]]))
    sc = (scale[:, :, None] * scale[:, None, :]).reshape(-1, 36)
    cov = np.abs(gpu.cov - ora.cov) / np.maximum(sc, 1e-300)
    return float(rel.max(initial=0.0)), float(chi2.max(initial=0.0)), float(cov.max(initial=0.0))


def by_seed(tr):
    """seed -> {tuple(meas list): track index}"""
    out = {}
    for t in range(tr.n_tracks):
        out.setdefault(int(tr.seed_id[t]), {})[tuple(int(i) for i in tr.meas_list(t))] = t
    return out


def compare_fp32(gpu, ora, n_seeds, qop_floor=0.0):
    """Returns dict: frac_identical seeds, mismatching seed ids, max param rel diff / chi2 abs diff on matched tracks."""
    if (gpu.n_tracks == ora.n_tracks and np.array_equal(gpu.seed_id, ora.seed_id) and
            np.array_equal(gpu.track_offsets, ora.track_offsets) and np.array_equal(gpu.meas_idx, ora.meas_idx)):
        # the common case: same candidates in the same order -> everything vectorised, every entry compared
        rel = param_rel_diff(gpu.params.copy(), ora.params.copy(), qop_floor)
        chi2 = np.abs(gpu.chi2_sum - ora.chi2_sum)
        emax = float(np.max(np.abs(gpu.entry_chi2 - ora.entry_chi2), initial=0.0))
        return dict(frac_identical=1.0, bad_seeds=[], n_matched=int(gpu.n_tracks),
                    max_param_rel=float(rel.max(initial=0.0)), max_chi2_sum_abs=float(chi2.max(initial=0.0)),
                    max_entry_chi2_abs=emax,
                    table1=[float(np.mean(rel.max(axis=1) <= tol)) if gpu.n_tracks else 1.0 for tol in (1e-4, 1e-3, 1e-2, 5e-2)])
    g, o = by_seed(gpu), by_seed(ora)
    bad = []
    gi, oi = [], []
    for s in range(n_seeds):
        gs, os_ = g.get(s, {}), o.get(s, {})
        if set(gs) != set(os_):
            bad.append(s)
        for k in set(gs) & set(os_):
            gi.append(gs[k])
            oi.append(os_[k])
    gi, oi = np.array(gi, int), np.array(oi, int)
    rel = param_rel_diff(gpu.params[gi].copy(), ora.params[oi].copy(), qop_floor) if gi.size else np.zeros((0, 6))
    chi2 = np.abs(gpu.chi2_sum[gi] - ora.chi2_sum[oi]) if gi.size else np.zeros(0)
    # per-entry chi2 on matched tracks
    emax = 0.0
    for a, b in zip(gi[:20000], oi[:20000]):
        ea = gpu.entry_chi2[gpu.track_offsets[a]:gpu.track_offsets[a + 1]]
        eb = ora.entry_chi2[ora.track_offsets[b]:ora.track_offsets[b + 1]]
        if ea.size:
            emax = max(emax, float(np.max(np.abs(ea - eb))))
    return dict(frac_identical=1.0 - len(bad) / max(1, n_seeds), bad_seeds=bad, n_matched=int(gi.size),
                max_param_rel=float(rel.max(initial=0.0)), max_chi2_sum_abs=float(chi2.max(initial=0.0)),
                max_entry_chi2_abs=emax,
                table1=[float(np.mean(rel.max(axis=1) <= tol)) if gi.size else 1.0 for tol in (1e-4, 1e-3, 1e-2, 5e-2)])


def compare_fits(gpu: dict, ora, track_offsets):
    """CUDA ckf_fit (dict of arrays from CKF.download_fits) against oracle.kf_fit on the SAME candidate lists.
    Integer results must be equal; returns the maximum A15 relative differences of the forward state at the last
    measurement and of the smoothed parameters, the scaled covariance difference at the first measurement, and the
    Table-1-style matching ratios of the smoothed parameters (fitted parameters at 0.01/0.1/1/5 %)."""
    # The one tolerated difference (counted, asserted by the callers): a track whose forward pass succeeded on both
    # sides but whose float32-STORED predicted covariance is no longer positive definite, so that the CUDA smoother
    # flags it NUMERIC (5) and reports zeros while the all-float64 oracle fits it.
    diff = gpu["status"] != ora.status
    only_gpu = diff & (gpu["status"] == 5) & (ora.status == 0)
    assert np.array_equal(diff, only_gpu), np.flatnonzero(diff & ~only_gpu)[:10]
    assert np.array_equal(gpu["n_states"], ora.n_states)
    if only_gpu.any():   # compare the rest: blank the oracle's values for those tracks like the CUDA path does
        import copy
        ora = copy.deepcopy(ora)
        for t in np.flatnonzero(only_gpu):
            ora.status[t] = 5
            ora.chi2_sum[t] = 0.0; ora.last_params[t] = 0.0; ora.last_cov[t] = 0.0; ora.first_cov[t] = 0.0
            ora.entry_params[track_offsets[t]:track_offsets[t + 1]] = 0.0
    ok = ora.status == 0
    last = param_rel_diff(gpu["last_params"][ok].copy(), ora.last_params[ok].copy())
    ent = param_rel_diff(gpu["entry_params"].copy(), ora.entry_params.copy())
    scale = np.sqrt(np.abs(ora.first_cov[:, [0, 7, 14, 21, 28, 35]]))
    sc = (scale[:, :, None] * scale[:, None, :]).reshape(-1, 36)
    cov = (np.abs(gpu["first_cov"] - ora.first_cov) / np.maximum(sc, 1e-300))[ok]
    first = track_offsets[:-1][ok]
    rel_first = ent[first].max(axis=1) if first.size else np.zeros(0)
    return dict(n_fitted=int(ok.sum()), n_failed=int((~ok).sum()), n_not_pd_gpu_only=int(only_gpu.sum()),
                max_last_rel=float(last.max(initial=0.0)), max_smoothed_rel=float(ent.max(initial=0.0)),
                max_first_cov_scaled=float(cov.max(initial=0.0)),
                max_chi2_abs=float(np.abs(gpu["chi2_sum"] - ora.chi2_sum).max(initial=0.0)),
                table1_first=[float(np.mean(rel_first <= tol)) if first.size else 1.0 for tol in (1e-4, 1e-3, 1e-2, 5e-2)])


def split_batch(tr, batch):
    """Per-event views of the candidates of a batched ckf_find (paper_2505_22822_b200.EventBatch): seed ids, entry
    offsets and measurement indices rebased to the event's own arrays.  Returns [(TrackArrays-like, t0, t1, e0)]."""
    from types import SimpleNamespace
    out = []
    for (s0, s1), (m0, _m1) in zip(batch.seed_ranges, batch.meas_ranges):
        t0 = int(np.searchsorted(tr.seed_id, s0, side="left"))
        t1 = int(np.searchsorted(tr.seed_id, s1, side="left"))
        e0, e1 = int(tr.track_offsets[t0]), int(tr.track_offsets[t1])
        v = SimpleNamespace(n_tracks=t1 - t0, track_offsets=tr.track_offsets[t0:t1 + 1] - e0,
                            meas_idx=tr.meas_idx[e0:e1] - m0, entry_chi2=tr.entry_chi2[e0:e1],
                            seed_id=tr.seed_id[t0:t1] - s0, n_holes=tr.n_holes[t0:t1], last_module=tr.last_module[t0:t1],
                            stop_reason=tr.stop_reason[t0:t1], params=tr.params[t0:t1], cov=tr.cov[t0:t1],
                            chi2_sum=tr.chi2_sum[t0:t1])
        v.meas_list = lambda t, v=v: v.meas_idx[v.track_offsets[t]:v.track_offsets[t + 1]]
        out.append((v, t0, t1, e0))
    return out


def trace_mismatches(gpu, ora, bad_seeds, chi2_max, tol=1e-3):
    """north_star: every seed whose candidate lists differ must be traced to a chi2 within `tol` of the gate or to a
    branch-ranking tie.  For every list that exists on one side only, the list of the other side with the longest
    common prefix is found; at the first differing position the cause must show:
      gate  -- a measurement attached there (on either side) has |chi2 - chi2_max| < tol: one side let it pass;
      tie   -- two different measurements attached there after the same prefix (any list, either side) have chi2 values
               closer than tol: their rank, hence what the k-best cut or the per-seed cap kept, may legitimately swap.
    Returns [(seed, reason or None)], one entry per bad seed; None = unexplained (a real discrepancy)."""
    out = []
    for s in bad_seeds:
        sides = []
        for tr in (gpu, ora):
            idx = np.flatnonzero(tr.seed_id == s)
            sides.append([(tuple(int(i) for i in tr.meas_list(t)),
                           np.asarray(tr.entry_chi2[tr.track_offsets[t]:tr.track_offsets[t + 1]], np.float64)) for t in idx])
        reason = "gate/tie"
        for a, b in ((0, 1), (1, 0)):
            have = {l for l, _ in sides[b]}
            for L, cL in sides[a]:
                if L in have:
                    continue
                # longest common prefix with any list of the other side
                best, Mb, cMb = -1, (), np.zeros(0)
                for M, cM in sides[b]:
                    c = 0
                    while c < len(L) and c < len(M) and L[c] == M[c]:
                        c += 1
                    if c > best:
                        best, Mb, cMb = c, M, cM
                c = max(best, 0)
                here = [float(x[c]) for l, x in ((L, cL), (Mb, cMb)) if len(l) > c]
                gate = any(abs(v - chi2_max) < tol for v in here)
                # all continuations of the common prefix, both sides
                cont = {}
                for side in sides:
                    for M, cM in side:
                        if len(M) > c and M[:c] == L[:c]:
                            cont[M[c]] = float(cM[c])
                vals = sorted(cont.values())
                tie = any(v2 - v1 < tol for v1, v2 in zip(vals, vals[1:]))
                if not (gate or tie):
                    reason = None
        out.append((int(s), reason))
    return out


def assert_fp32_parity(gpu, ora, n_seeds, chi2_max, what="", qop_floor=0.0):
    """The fp32 bar of north_star in one place: >= 99.9 % of seeds with identical lists, EVERY mismatch traced,
    parameters 1e-4 relative, chi2 1e-3 absolute."""
    r = compare_fp32(gpu, ora, n_seeds, qop_floor)
    traced = trace_mismatches(gpu, ora, r["bad_seeds"], chi2_max)
    untraced = [s for s, why in traced if why is None]
    assert r["frac_identical"] >= 0.999, (what, r["frac_identical"])
    assert not untraced, (what, "mismatching seeds not explained by a gate-edge chi2 or a ranking tie", untraced[:10])
    assert r["max_param_rel"] < 1e-4, (what, r["max_param_rel"])
    assert r["max_chi2_sum_abs"] < 1e-3, (what, r["max_chi2_sum_abs"])
    assert r["max_entry_chi2_abs"] < 1e-3, (what, r["max_entry_chi2_abs"])
    r["n_mismatch_traced"] = len(traced)
    return r
