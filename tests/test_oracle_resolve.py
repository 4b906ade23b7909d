"""Pins of the oracle's ambiguity resolution (rules AR1-AR3): the greedy shared-hit resolver.

The greedy result is the UNIQUE subset A of the candidates with the property
    t in A   <=>   |hits(t) & union of hits(u), u in A ranked better than t| <= limit(t)
(induction over the rank order), so it can be pinned without re-typing the loop: brute force over all 2^n subsets of
a small candidate set must find exactly one subset with that property, and it must be the oracle's."""
import itertools

import numpy as np
import pytest

import oracle
import synth


def _csr(lists):
    off = np.zeros(len(lists) + 1, np.int32)
    off[1:] = np.cumsum([len(l) for l in lists])
    return off, np.array([m for l in lists for m in l], np.int32)


def _rank_key(lists, chi2, t):
    return (-len(lists[t]), np.float32(chi2[t]), t)


def _fixed_points(lists, chi2, k, frac):
    n = len(lists)
    order = sorted(range(n), key=lambda t: _rank_key(lists, chi2, t))
    pos = {t: i for i, t in enumerate(order)}
    sets = [set(l) for l in lists]
    found = []
    for bits in itertools.product((0, 1), repeat=n):
        ok = True
        for t in range(n):
            better = set()
            for u in range(n):
                if bits[u] and pos[u] < pos[t]:
                    better |= sets[u]
            s = len(sets[t] & better)
            want = 1 if (s <= k and s <= frac * len(lists[t])) else 0
            if want != bits[t]:
                ok = False
                break
        if ok:
            found.append(bits)
    return found


@pytest.mark.parametrize("k,frac", [(0, 1.0), (1, 1.0), (2, 1.0), (3, 0.3), (100, 1.0)])
def test_greedy_is_the_unique_fixed_point(k, frac):
    rng = np.random.default_rng(5 + k)
    for trial in range(6):
        n = 11
        # candidates that overlap a lot: random subsets of a small pool of measurements, distinct lengths and chi2
        lists = [sorted(rng.choice(14, size=rng.integers(3, 8), replace=False).tolist()) for _ in range(n)]
        chi2 = rng.uniform(1.0, 30.0, n)
        chi2[3] = chi2[7]                                       # an exact chi2 tie: the index decides
        off, mi = _csr(lists)
        acc, ns = oracle.resolve_ambiguity(off, mi, chi2, 14, k, frac)
        fps = _fixed_points(lists, chi2, k, frac)
        assert len(fps) == 1
        assert tuple(int(a) for a in acc) == fps[0]
        # the reported shared count is the one the decision used
        for t in range(n):
            assert (ns[t] <= k and ns[t] <= frac * len(lists[t])) == bool(acc[t])


def test_limits_and_duplicates():
    lists = [[0, 1, 2, 3], [0, 1, 2, 3], [0, 1, 2, 3, 4], [5, 6, 7], [3, 5, 6]]
    chi2 = np.array([4.0, 3.0, 9.0, 1.0, 2.0])
    off, mi = _csr(lists)
    # k = 0: hit-disjoint survivors; the 5-hit list wins over its sub-lists; [5,6,7] beats [3,5,6] only through rank
    acc, _ = oracle.resolve_ambiguity(off, mi, chi2, 8, 0, 1.0)
    assert acc.tolist() == [0, 0, 1, 1, 0]
    # exact duplicates: the better chi2 survives, not both
    acc, _ = oracle.resolve_ambiguity(*_csr(lists[:2]), chi2[:2], 8, 0, 1.0)
    assert acc.tolist() == [0, 1]
    # no limit: everything is accepted
    acc, _ = oracle.resolve_ambiguity(off, mi, chi2, 8, 1000, 1.0)
    assert acc.tolist() == [1, 1, 1, 1, 1]
    # empty input
    acc, ns = oracle.resolve_ambiguity(np.zeros(1, np.int32), np.zeros(0, np.int32), np.zeros(0), 8, 1, 1.0)
    assert acc.size == 0 and ns.size == 0


def _double_matching(ev, tr, keep):
    """a candidate's major particle contributes N of its N_t hits and has N_p hits in the event;
    matched iff N > N_t / 2 and N > N_p / 2.  Returns (matched particle or -1) per kept candidate."""
    n_p = np.bincount(ev.meas_particle[ev.meas_particle >= 0], minlength=ev.particle_q.size)
    out = []
    for t in np.flatnonzero(keep):
        pid = ev.meas_particle[tr.meas_list(t)]
        pid = pid[pid >= 0]
        if pid.size == 0:
            out.append(-1)
            continue
        vals, cnt = np.unique(pid, return_counts=True)
        j = int(np.argmax(cnt))
        N, Nt, Np = int(cnt[j]), int(tr.track_offsets[t + 1] - tr.track_offsets[t]), int(n_p[vals[j]])
        out.append(int(vals[j]) if (2 * N > Nt and 2 * N > Np) else -1)
    return np.array(out, int)


def test_resolution_removes_duplicates_and_keeps_efficiency():
    """Physics sanity on synthetic truth (not a parity pin): with the paper's double-matching definition the duplicate
    rate collapses while the efficiency stays."""
    det, fld, cfg = synth.config_bundle(1)
    ev = synth.make_event(1, det=det, n_particles=800)
    tr = oracle.find_event(oracle.Setup(det, fld, cfg.ckf), ev, n_threads=8)
    acc, _ = oracle.resolve_ambiguity(tr.track_offsets, tr.meas_idx, tr.chi2_sum, ev.n_measurements, 1, 1.0)
    n_part = int(np.sum(ev.seed_particle >= 0))
    before = _double_matching(ev, tr, np.ones(tr.n_tracks, bool))
    after = _double_matching(ev, tr, acc.astype(bool))
    eff_b, eff_a = np.unique(before[before >= 0]).size / n_part, np.unique(after[after >= 0]).size / n_part
    dup_b = 1.0 - np.unique(before[before >= 0]).size / max(1, np.sum(before >= 0))
    dup_a = 1.0 - np.unique(after[after >= 0]).size / max(1, np.sum(after >= 0))
    print("efficiency %.4f -> %.4f, duplicate rate %.4f -> %.4f, candidates %d -> %d" %
          (eff_b, eff_a, dup_b, dup_a, tr.n_tracks, int(acc.sum())))
    assert eff_a >= eff_b - 0.01 and eff_a > 0.97
    assert dup_a < 0.01 and (dup_b == 0.0 or dup_a <= 0.2 * dup_b)
