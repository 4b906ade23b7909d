// ckf_level_loop.cuh — the persistent, warp-autonomous level-loop kernel (a3-a11).  See ckf_kernels.cuh.
#pragma once
#include "ckf_kernels.cuh"

namespace ckf {

// ---- P2 (a7, a8): gate of the <= 32 tips of a chunk.  Lane = tip for the window search and the ranking; the
// chi2 tests run over the FLATTENED (tip, measurement) pairs of all windows, 32 pairs per round, so the
// lanes stay full whatever the individual window lengths are.  Passers of a tip are collected in any order
// (shared-memory counter) and then ranked by (chi2, index), which makes the result order-independent.
// Returns the number of selected measurements of this lane's tip, written in rank order to sel*[rank][lane].
template <typename T>
__device__ __forceinline__ int gate_chunk(const KParams<T>& p, const WSmem<T>& s, int lane, bool visit, int K,
                                          unsigned long long& n_exec) {
  const T chi2_max = (T)p.cfg.chi2_max;
  int lo = 0, len = 0;
  if (visit) {
    const int m = s.target[lane];
    const int beg = __ldg(p.moff + m), end = __ldg(p.moff + m + 1);
    int hi = end;
    lo = beg;
    if (end > beg) {
      const T v0max = p.s_v0max[m];
      const T C00 = s.pC[tri(0, 0) * 32 + lane], C01 = s.pC[tri(0, 1) * 32 + lane], C11 = s.pC[tri(1, 1) * 32 + lane];
      if (v0max >= T(0) && C00 > T(0) && C11 > T(0) && C00 * C11 - C01 * C01 > T(0)) {
        // chi2 >= r0^2 / S00 and S00 <= C00 + v0max: nothing outside |loc0 - l0| <= w can pass
        const double w = sqrt(p.cfg.chi2_max * ((double)C00 + (double)v0max)) * (1.0 + 1e-6) + 1e-9;
        if (isfinite(w)) {
          const double l0 = s.px[0 * 32 + lane];
          const double a = l0 - w, b = l0 + w;
          int x0 = beg, x1 = end;  // first k with loc0[k] >= a
          while (x0 < x1) {
            const int mid = (x0 + x1) >> 1;
            if ((double)p.s_loc[mid].x < a) x0 = mid + 1; else x1 = mid;
          }
          lo = x0;
          x1 = end;  // first k with loc0[k] > b
          while (x0 < x1) {
            const int mid = (x0 + x1) >> 1;
            if ((double)p.s_loc[mid].x <= b) x0 = mid + 1; else x1 = mid;
          }
          hi = x0;
        }
      }
    }
    len = hi - lo;
  }
  const int inc = warp_incl_scan(len, lane);
  const int total = __shfl_sync(0xffffffffu, inc, 31);
  s.off[lane] = inc - len;
  s.lo[lane] = lo;
  s.cnt[lane] = 0;
  __syncwarp();
  for (int q0 = 0; q0 < total; q0 += 32) {
    const int q = q0 + lane;
    if (q < total) {
      int t = 0;  // last tip with off[t] <= q (tips with an empty window share off with their successor)
#pragma unroll
      for (int b = 16; b > 0; b >>= 1)
        if (s.off[t + b] <= q) t += b;
      const int k = s.lo[t] + (q - s.off[t]);
      const auto lc = p.s_loc[k];
      const auto vr = p.s_var[k];
      T c2 = T(0);
      const bool pass = gate_chi2<T>(s.px[0 * 32 + t], s.px[1 * 32 + t], s.pC[tri(0, 0) * 32 + t],
                                     s.pC[tri(0, 1) * 32 + t], s.pC[tri(1, 1) * 32 + t], lc.x, lc.y, vr.x, vr.y,
                                     chi2_max, c2);
      if (pass) {
        const int pos = atomicAdd(&s.cnt[t], 1);
        if (pos < CAND) { s.candchi2[pos * 32 + t] = c2; s.candidx[pos * 32 + t] = p.s_idx[k]; }
      }
    }
  }
  if (lane == 0) n_exec += (unsigned long long)total;
  __syncwarp();
  int nsel = 0;
  if (visit) {
    const int count = s.cnt[lane];
    if (count <= CAND) {
      // fast path: rank the passers by (chi2, index)
      for (int a = 0; a < count; ++a) {
        const T mc = s.candchi2[a * 32 + lane];
        const int mi = s.candidx[a * 32 + lane];
        int rank = 0;
        for (int b = 0; b < count; ++b) rank += key_less<T>(s.candchi2[b * 32 + lane], s.candidx[b * 32 + lane], mc, mi) ? 1 : 0;
        if (rank < K) { s.selchi2[rank * 32 + lane] = mc; s.selidx[rank * 32 + lane] = mi; }
      }
      nsel = count < K ? count : K;
    } else {
      // rare: more than CAND passers.  K rounds of "smallest key above the last one" over the window.
      const double l0 = s.px[0 * 32 + lane], l1 = s.px[1 * 32 + lane];
      const T C00 = s.pC[tri(0, 0) * 32 + lane], C01 = s.pC[tri(0, 1) * 32 + lane], C11 = s.pC[tri(1, 1) * 32 + lane];
      T last_c = T(-1);
      int last_i = -1;
      nsel = count < K ? count : K;
      for (int r = 0; r < nsel; ++r) {
        T bc = T(0);
        int bi = 0x7fffffff;
        for (int k = lo; k < lo + len; ++k) {
          const auto lc = p.s_loc[k];
          const auto vr = p.s_var[k];
          T c2 = T(0);
          const bool ok = gate_chi2<T>(l0, l1, C00, C01, C11, lc.x, lc.y, vr.x, vr.y, chi2_max, c2);
          const int id = p.s_idx[k];
          if (ok && key_less<T>(last_c, last_i, c2, id) && (bi == 0x7fffffff || key_less<T>(c2, id, bc, bi))) {
            bc = c2; bi = id;
          }
        }
        s.selchi2[r * 32 + lane] = bc;
        s.selidx[r * 32 + lane] = bi;
        last_c = bc; last_i = bi;
      }
    }
  }
  return nsel;
}

// ---- P1 scratch of one warp (aliases the P2-P4 arrays of WSmem: the two phases never overlap in time)
struct P1Smem {
  double* hit;     // [9][32] path length of each (tip, neighbour) test; NaN = no hit
  double* rd;      // [6][32] position and direction of the requesting tips
  int32_t* hid;    // [9][32] module id of each test
  int32_t *rl, *ri, *rj, *rx, *list;  // [32] request: layer (-1 none), iphi, iz, exclude | s_min sign, compacted lanes
  static constexpr size_t bytes() { return 8 * 9 * 32 + 8 * 6 * 32 + 4 * 9 * 32 + 4 * 5 * 32; }
  __device__ void carve(unsigned char* raw) {
    unsigned char* p = raw;
    hit = (double*)p; p += 8 * 9 * 32;
    rd = (double*)p; p += 8 * 6 * 32;
    hid = (int32_t*)p; p += 4 * 9 * 32;
    rl = (int32_t*)p; p += 4 * 32;
    ri = (int32_t*)p; p += 4 * 32;
    rj = (int32_t*)p; p += 4 * 32;
    rx = (int32_t*)p; p += 4 * 32;
    list = (int32_t*)p; p += 4 * 32;
  }
};

// ---- a4: module choice for all lanes in PH_START / PH_LANDED at once.  The nine straight-line tests of each
// requesting tip are spread over the 32 lanes as flattened (tip, neighbour) pairs; the owning lane then
// scans its nine results in the order of the sequential rule (nearest first, tie -> lower id).
template <typename T>
__device__ __forceinline__ void pick_warp(const KParams<T>& p, const P1Smem& ps, Move<T>& m, int lane) {
  const bool need = m.phase == PH_START || m.phase == PH_LANDED;
  PickRequest q;
  bool ok = false;
  if (need) ok = move_pick_request(m, p.geo, q);
  const unsigned breq = __ballot_sync(0xffffffffu, ok);
  if (ok) {
    ps.rl[lane] = q.layer; ps.ri[lane] = q.iphi; ps.rj[lane] = q.iz;
    ps.rx[lane] = (q.exclude < 0 ? 0 : q.exclude + 1) * 2 + (q.s_min > 0.0 ? 1 : 0);
#pragma unroll
    for (int i = 0; i < 3; ++i) { ps.rd[i * 32 + lane] = m.y.r[i]; ps.rd[(3 + i) * 32 + lane] = m.y.d[i]; }
    ps.list[__popc(breq & ((1u << lane) - 1u))] = lane;
  }
  __syncwarp();
  const int total = 9 * __popc(breq);
  for (int q0 = 0; q0 < total; q0 += 32) {
    const int pr = q0 + lane;
    if (pr < total) {
      const int t = ps.list[pr / 9], nb = pr % 9;
      const LayerRec L = p.geo.layer[ps.rl[t]];
      int ii = ps.ri[t] + (nb / 3 - 1);
      ii = ii < 0 ? ii + L.n_phi : (ii >= L.n_phi ? ii - L.n_phi : ii);
      const int jj = ps.rj[t] + (nb % 3 - 1);
      const int rx = ps.rx[t];
      double sres = __longlong_as_double(0x7ff8000000000000LL);
      int id = -1;
      if (jj >= 0 && jj < L.n_z) {
        id = L.offset + ii * L.n_z + jj;
        if (id != (rx >> 1) - 1) {
          const double r[3] = {ps.rd[0 * 32 + t], ps.rd[1 * 32 + t], ps.rd[2 * 32 + t]};
          const double d[3] = {ps.rd[3 * 32 + t], ps.rd[4 * 32 + t], ps.rd[5 * 32 + t]};
          double sv;
          if (line_hits_module(p.geo.mod[id], r, d, (rx & 1) ? 1e-3 : -1e-3, sv)) sres = sv;
        }
      }
      ps.hit[nb * 32 + t] = sres;
      ps.hid[nb * 32 + t] = id;
    }
  }
  __syncwarp();
  if (need) {
    int best = -1;
    double best_s = 0.0;
    if (ok) {
#pragma unroll 1
      for (int nb = 0; nb < 9; ++nb) {
        const double sv = ps.hit[nb * 32 + lane];
        const int id = ps.hid[nb * 32 + lane];
        if (sv == sv && (best < 0 || sv < best_s || (sv == best_s && id < best))) { best = id; best_s = sv; }
      }
    }
    move_pick_apply(m, p.geo, best);
  }
  __syncwarp();
}

// Predictions of one sub-wave of a warp, in global memory (written by P1, read by the P2-P4 chunks)
template <typename T>
struct Pred {
  double* x;        // [6][SUBW]
  T* C;             // [21][SUBW]
  int32_t* target;  // [SUBW]
  int32_t* stop;    // [SUBW]
};

// ---- P1 (a3-a6) for tips [w0, w1) of the warp's wave.  Every lane owns one Move at a time and pulls the next
// tip when its move is done (persistent lanes), so lanes do not idle while a neighbour needs more RKN4
// trials.  The heavy non-trial code runs at SERVICE points, converged: lanes that finished (arrival
// algebra), lanes without a tip (fetch + departure state) and lanes that need a module choice wait until
// SERVICE_MIN of them have gathered, or until no lane can step.
template <typename T>
__device__ __forceinline__ void propagate_wave(const KParams<T>& p, const P1Smem& ps, const int2* Qin, int w0, int w1,
                                               const Pred<T>& pred, int lane, unsigned long long& my_trials,
                                               unsigned long long& my_accepted) {
  Move<T> m;
  m.phase = PH_IDLE; m.stop = STOP_NONE; m.from = 0; m.tgt = -1; m.lp = 0; m.n_steps = 0; m.retry = false;
  m.h = 0.0; m.h_ctrl = 0.0; m.R = 0.0; m.y.qop = 0.0;
  int tip = -1, link = -1, nt = 0, na = 0;
  int next = w0;
  for (;;) {
    const unsigned bI = __ballot_sync(0xffffffffu, m.phase == PH_IDLE);
    const unsigned bP = __ballot_sync(0xffffffffu, m.phase == PH_START || m.phase == PH_LANDED);
    const unsigned bS = __ballot_sync(0xffffffffu, m.phase == PH_CYL || m.phase == PH_PLANE);
    const unsigned bF = __ballot_sync(0xffffffffu, m.phase == PH_FIN);
    const int R = w1 - next;
    if (!bP && !bS && !bF && R <= 0) break;
    const int waiting = __popc(bF) + __popc(bP) + (R > 0 ? __popc(bI) : 0);
    if (bS == 0u || waiting >= SERVICE_MIN) {
      // ---- arrival (J4, J5), covariance transport, prediction record
      if (bF) {
        if (m.phase == PH_FIN) {
          const int slot = tip - w0;
          int stop = m.stop;
          if (stop == STOP_NONE) {
            double xp[6];
            T J[5][5];
            stop = move_arrive<T>(m, p.geo, p.fld, p.cfg, xp, J);
            if (stop == STOP_NONE) {
              T C[21], Co[21];
#pragma unroll
              for (int i = 0; i < 21; ++i) C[i] = p.lk_C[(size_t)i * p.max_links + link];
              C[tri(2, 2)] += m.q_phi;
              C[tri(3, 3)] += m.q_theta;
              transport_cov<T>(J, C, Co);
              bool fin = true;
#pragma unroll
              for (int i = 0; i < 21; ++i) { pred.C[i * SUBW + slot] = Co[i]; fin = fin && isfinite(Co[i]); }
#pragma unroll
              for (int i = 0; i < 6; ++i) pred.x[i * SUBW + slot] = xp[i];
              if (!fin) stop = STOP_NUMERIC;
            }
          }
          pred.target[slot] = m.tgt;
          pred.stop[slot] = stop;
          m.phase = PH_IDLE;
        }
        __syncwarp();
      }
      // ---- fetch: idle lanes take the next tips of the wave, in order
      const unsigned idle = __ballot_sync(0xffffffffu, m.phase == PH_IDLE);
      if (idle && next < w1) {
        const int t = next + __popc(idle & ((1u << lane) - 1u));
        const bool got = m.phase == PH_IDLE && t < w1;
        next += min(__popc(idle), w1 - next);
        if (got) {
          tip = t;
          const int2 e = Qin[t];
          link = e.x;
          const int seed = e.y, slot = t - w0;
          if (link < 0) {
            // fresh seed: level 0 visits the seed's own module with identity transport (N6)
            bool ok = true;
#pragma unroll
            for (int i = 0; i < 6; ++i) {
              const double v = (double)p.seed_x[(size_t)seed * 6 + i];
              ok = ok && isfinite(v);
              if (i == 3) ok = ok && (v > 0.0 && v < PI_D);
              pred.x[i * SUBW + slot] = v;
            }
#pragma unroll
            for (int i = 0; i < 6; ++i)
#pragma unroll
              for (int j = i; j < 6; ++j) pred.C[tri(i, j) * SUBW + slot] = p.seed_C[(size_t)seed * 36 + i * 6 + j];
            pred.target[slot] = p.seed_module[seed];
            pred.stop[slot] = ok ? STOP_NONE : STOP_NUMERIC;
          } else {
            const int counts = p.lk_counts[link];
            if ((counts & 0xffff) + (counts >> 16) >= p.cfg.max_levels) {
              pred.target[slot] = -1;
              pred.stop[slot] = STOP_LEVEL_LIMIT;
            } else {
              double x[6];
#pragma unroll
              for (int i = 0; i < 6; ++i) x[i] = p.lk_x[(size_t)i * p.max_links + link];
              move_init<T>(m, p.geo, p.cfg, p.lk_module[link], x);
            }
          }
        }
        __syncwarp();
      }
      // ---- module choice for every lane that needs one
      if (__ballot_sync(0xffffffffu, m.phase == PH_START || m.phase == PH_LANDED)) pick_warp<T>(p, ps, m, lane);
    }
    // ---- one step: targeting + landing, else one RKN4 trial
    if (m.phase == PH_CYL || m.phase == PH_PLANE) move_step<T>(m, p.fld, p.cfg, nt, na);
    __syncwarp();
  }
  my_trials += (unsigned long long)nt;
  my_accepted += (unsigned long long)na;
}

template <typename T, int MINB>
__global__ void __launch_bounds__(NT, MINB) ckf_level_loop(const KParams<T> p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int K = p.cfg.max_branches;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  WSmem<T> s;
  s.carve(smem_raw + (size_t)wib * WSmem<T>::bytes(K), K);
  P1Smem ps;
  ps.carve(smem_raw + (size_t)wib * WSmem<T>::bytes(K));
  const int gw = blockIdx.x * WPB + wib, nw = gridDim.x * WPB;
  const int cap = p.cfg.max_cands;
  Pred<T> pred;
  pred.x = p.pred_x + (size_t)gw * 6 * SUBW;
  pred.C = p.pred_C + (size_t)gw * 21 * SUBW;
  pred.target = p.pred_ts + (size_t)gw * 2 * SUBW;
  pred.stop = pred.target + SUBW;
  int2* Q0 = p.queue + (size_t)gw * 2 * p.qcap;
  int2* Q1 = Q0 + p.qcap;
  int fair = (p.n_seeds + nw - 1) / nw;
  fair = fair < 1 ? 1 : fair;
  unsigned long long my_trials = 0, my_accepted = 0, my_gate = 0, my_visits = 0, my_updates = 0;
  unsigned long long w_tips = 0, w_links = 0, w_iter = 0, w_exec = 0;  // lane 0 only
  int n_live = 0, seeds_bound = 0;

  for (int wave = 0;; ++wave) {
    int2* Qin = (wave & 1) ? Q1 : Q0;
    int2* Qout = (wave & 1) ? Q0 : Q1;
    // ---------------- refill: pull seeds while the last chunk has free lanes (continuous batching)
    {
      int want = n_live == 0 ? 32 : ((32 - (n_live & 31)) & 31);
      want = want > fair ? fair : want;
      const int room = MAX_LIVE_SEEDS - seeds_bound;
      want = want > room ? room : want;
      int pb = 0, pn = 0;
      if (lane == 0 && want > 0 && *(volatile int32_t*)p.g_seed_cursor < p.n_seeds) {
        pb = atomicAdd(p.g_seed_cursor, want);
        pn = pb < p.n_seeds ? min(want, p.n_seeds - pb) : 0;
      }
      pb = __shfl_sync(0xffffffffu, pb, 0);
      pn = __shfl_sync(0xffffffffu, pn, 0);
      if (lane < pn) Qin[n_live + lane] = make_int2(-(pb + lane) - 1, pb + lane);
      n_live += pn;
      __syncwarp();
    }
    if (n_live == 0) break;  // the pull returned nothing and nothing is alive: all seeds are taken

    int n_out = 0, seeds_seen = 0;
    // R10 state of a seed whose tips straddle two chunks (warp-uniform)
    int carry_seed = -1, carry_E = 0, carry_extra0 = 0, carry_K = 0;

    for (int w0 = 0; w0 < n_live; w0 += SUBW) {
    const int w1 = min(n_live, w0 + SUBW);
    // ======== P1: persistent lanes over the sub-wave — load, navigate, propagate, predict (a3-a6)
    propagate_wave<T>(p, ps, Qin, w0, w1, pred, lane, my_trials, my_accepted);
    __syncwarp();
    for (int base = w0; base < w1; base += 32) {
      const int n = min(32, n_live - base);
      const bool act = lane < n;
      int2 e = make_int2(0, -2);
      if (act) e = Qin[base + lane];
      const int seed = e.y;
      int link = e.x;
      int next_seed = -3;
      if (base + 32 < n_live) next_seed = Qin[base + 32].y;

      // predictions of this chunk's tips -> shared memory
      int stop = STOP_NONE, target = -1, counts = 0, lastmeas = -1;
      T c2s = T(0);
      if (act) {
        const int slot = base + lane - w0;
        stop = pred.stop[slot];
        target = pred.target[slot];
        if (link >= 0) {
          counts = p.lk_counts[link];
          lastmeas = p.lk_lastmeas[link];
          c2s = p.lk_chi2sum[link];
        } else link = -1;
        if (stop == STOP_NONE) {
#pragma unroll
          for (int i = 0; i < 6; ++i) s.px[i * 32 + lane] = pred.x[i * SUBW + slot];
#pragma unroll
          for (int i = 0; i < 21; ++i) s.pC[i * 32 + lane] = pred.C[i * SUBW + slot];
        }
      }
      s.link[lane] = link; s.seed[lane] = seed; s.target[lane] = target;
      s.lastmeas[lane] = lastmeas; s.chi2sum[lane] = c2s;
      __syncwarp();

      // ======== P2: chi2 gate over the loc0 windows, k best (a7, a8)
      const bool visit = act && stop == STOP_NONE;
      if (visit) {
        const int m = target;
        my_gate += (unsigned long long)(__ldg(p.moff + m + 1) - __ldg(p.moff + m));
        my_visits += 1ull;
      }
      const int nsel = gate_chunk<T>(p, s, lane, visit, K, w_exec);
      int want = 0;
      if (visit) {
        if (nsel == 0) {
          const int nh = (counts >> 16) + 1;
          if (nh > p.cfg.max_holes) { stop = STOP_HOLES; counts += (1 << 16); }
          else want = 1;
        } else want = nsel;
      }
      s.nsel[lane] = nsel;
      s.counts[lane] = counts;

      // ======== P3: per-seed cap R10 + warp prefix sums (a10)
      const int my_nm = counts & 0xffff;
      const int my_emit = (act && stop != STOP_NONE && my_nm >= p.cfg.min_meas) ? 1 : 0;
      const int prev_seed = __shfl_up_sync(0xffffffffu, seed, 1);
      const int succ_seed = __shfl_down_sync(0xffffffffu, seed, 1);
      const bool is_head = act && (lane == 0 || prev_seed != seed);
      const bool is_tail = act && (lane == n - 1 || succ_seed != seed);
      const int head = warp_incl_max(is_head ? lane : 0, lane);
      const bool cont_prev = act && head == 0 && seed == carry_seed;
      seeds_seen += __popc(__ballot_sync(0xffffffffu, is_head && !cont_prev));
      const int ev = want > 0 ? want - 1 : 0;
      const int Ein = warp_incl_scan(ev, lane);
      const int Ehead = __shfl_sync(0xffffffffu, Ein - ev, head);
      int extra0 = 0, sd_nemit = 0, sd_nent = 0;
      if (act) {
        extra0 = cont_prev ? carry_extra0 : p.sd_extra[seed];
        sd_nemit = p.sd_nemit[seed];
        sd_nent = p.sd_nentries[seed];
      }
      int keep = 0;
      if (want > 0) {
        const int Rm = cap - (1 + extra0);
        const int Pex = (Ein - ev) - Ehead + (cont_prev ? carry_E : 0);
        const int room = Rm - Pex;
        keep = 1 + min(ev, room > 0 ? room : 0);
      }
      const int Kin = warp_incl_scan(keep, lane);
      const int tot = __shfl_sync(0xffffffffu, Kin, 31);
      const int km1 = keep > 1 ? keep - 1 : 0;
      const int KMin = warp_incl_scan(km1, lane);
      const int KMhead = __shfl_sync(0xffffffffu, KMin - km1, head);
      const int mval = (my_emit << 16) | (my_emit ? my_nm : 0);
      const int Min = warp_incl_scan(mval, lane);
      const int Mhead = __shfl_sync(0xffffffffu, Min - mval, head);
      const int totE = (Ein - Ehead) + (cont_prev ? carry_E : 0);
      const int totK = (KMin - KMhead) + (cont_prev ? carry_K : 0);
      const bool cont_next = is_tail && n == 32 && lane == 31 && next_seed == seed;
      s.Kex[lane] = Kin - keep;
      if (lane == 31) s.Kex[32] = tot;
      int lb = 0, allowed = 0;
      if (lane == 0) {
        if (tot > 0) {
          lb = atomicAdd(p.g_link_count, tot);
          allowed = p.max_links - lb;
          allowed = allowed < 0 ? 0 : (allowed > tot ? tot : allowed);
          if (allowed < tot) atomicOr(p.o_status, 4);
          const int qroom = p.qcap - n_out;
          if (allowed > qroom) { allowed = qroom; atomicOr(p.o_status, 4); }
        }
        w_tips += (unsigned long long)n;
        w_links += (unsigned long long)allowed;
        w_iter += 1ull;
      }
      lb = __shfl_sync(0xffffffffu, lb, 0);
      allowed = __shfl_sync(0xffffffffu, allowed, 0);
      // emission records (a11) for tips that stopped at this level, in tip order within the seed
      if (my_emit) {
        const int slot = sd_nemit + ((Min - mval) >> 16) - (Mhead >> 16);
        const int eoff = sd_nent + ((Min - mval) & 0xffff) - (Mhead & 0xffff);
        if (slot < cap) {
          const size_t li = (size_t)seed * cap + slot;
          p.leaf_link[li] = link;
          p.leaf_meta[li] = stop | ((counts >> 16) << 8);
          p.leaf_entry[li] = eoff;
        }
      }
      __syncwarp();  // every lane has read its seed's counters; Kex is visible
      if (is_tail) {
        const int seg = Min - Mhead;
        if (seg != 0) {
          p.sd_nemit[seed] = sd_nemit + (seg >> 16);
          p.sd_nentries[seed] = sd_nent + (seg & 0xffff);
        }
        if (!cont_next && totK != 0) p.sd_extra[seed] = extra0 + totK;
      }
      {
        const int cn = __shfl_sync(0xffffffffu, cont_next ? 1 : 0, 31);
        const int cE = __shfl_sync(0xffffffffu, totE, 31);
        const int cK = __shfl_sync(0xffffffffu, totK, 31);
        const int cX = __shfl_sync(0xffffffffu, extra0, 31);
        const int cS = __shfl_sync(0xffffffffu, seed, 31);
        carry_seed = cn ? cS : -1;
        carry_E = cE; carry_K = cK; carry_extra0 = cX;
      }

      // ======== P4: lane per child — Kalman update or hole, link append, next queue (a9, a10)
      for (int c = lane; c < allowed; c += 32) {
        int par = 0;  // last tip with Kex <= c (tips that keep nothing share Kex with their successor)
#pragma unroll
        for (int b = 16; b > 0; b >>= 1)
          if (s.Kex[par + b] <= c) par += b;
        const int j = c - s.Kex[par];
        const int nl = lb + c;
        const int pc = s.counts[par];
        double x[6];
        T C[21];
#pragma unroll
        for (int i = 0; i < 6; ++i) x[i] = s.px[i * 32 + par];
#pragma unroll
        for (int i = 0; i < 21; ++i) C[i] = s.pC[i * 32 + par];
        int meas = -1, ncounts, nlast = s.lastmeas[par];
        T chi2 = T(0), nc2s = s.chi2sum[par];
        if (s.nsel[par] == 0) {
          ncounts = pc + (1 << 16);
#pragma unroll
          for (int i = 0; i < 6; ++i) p.lk_x[(size_t)i * p.max_links + nl] = x[i];
#pragma unroll
          for (int i = 0; i < 21; ++i) p.lk_C[(size_t)i * p.max_links + nl] = C[i];
        } else {
          meas = s.selidx[j * 32 + par];
          chi2 = s.selchi2[j * 32 + par];
          const auto lc = __ldg(p.loc + meas);
          const auto vr = __ldg(p.var + meas);
          double xo[6];
          T Co[21];
          kalman_update<T>(x, C, lc.x, lc.y, vr.x, vr.y, xo, Co);
          ncounts = pc + 1;
          nlast = nl;
          my_updates += 1ull;
          nc2s += chi2;
#pragma unroll
          for (int i = 0; i < 6; ++i) p.lk_x[(size_t)i * p.max_links + nl] = xo[i];
#pragma unroll
          for (int i = 0; i < 21; ++i) p.lk_C[(size_t)i * p.max_links + nl] = Co[i];
        }
        p.lk_module[nl] = s.target[par];
        p.lk_parent[nl] = s.link[par];
        p.lk_meas[nl] = meas;
        p.lk_chi2[nl] = chi2;
        p.lk_chi2sum[nl] = nc2s;
        p.lk_counts[nl] = ncounts;
        p.lk_lastmeas[nl] = nlast;
        Qout[n_out + c] = make_int2(nl, s.seed[par]);
      }
      n_out += allowed;
      __syncwarp();
    }
    }
    n_live = n_out;
    seeds_bound = seeds_seen;
  }

  // ---------------- work counters
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    my_trials += __shfl_xor_sync(0xffffffffu, my_trials, o);
    my_accepted += __shfl_xor_sync(0xffffffffu, my_accepted, o);
    my_gate += __shfl_xor_sync(0xffffffffu, my_gate, o);
    my_visits += __shfl_xor_sync(0xffffffffu, my_visits, o);
    my_updates += __shfl_xor_sync(0xffffffffu, my_updates, o);
  }
  if (lane == 0) {
    if (my_trials) atomicAdd(p.counters + CNT_TRIALS, my_trials);
    if (my_accepted) atomicAdd(p.counters + CNT_ACCEPTED, my_accepted);
    if (my_gate) atomicAdd(p.counters + CNT_GATE, my_gate);
    if (my_visits) atomicAdd(p.counters + CNT_VISITS, my_visits);
    if (my_updates) atomicAdd(p.counters + CNT_UPDATES, my_updates);
    if (w_tips) atomicAdd(p.counters + CNT_TIPS, w_tips);
    if (w_links) atomicAdd(p.counters + CNT_LINKS, w_links);
    if (w_iter) atomicAdd(p.counters + CNT_ITER, w_iter);
    if (w_exec) atomicAdd(p.counters + CNT_GATE_EXEC, w_exec);
  }
}

}  // namespace ckf
