// ckf_level_loop.cuh — the persistent level-loop kernel (a3-a11).  See ckf_kernels.cuh for the design.
#pragma once
#include "ckf_kernels.cuh"

namespace ckf {

// ---- P2: gate of one tip by one warp (a7, a8).  Returns the number of selected measurements (<= K), written
// in (chi2, index) rank order to sel*[rank][slot].  `count_out` = number of chi2 evaluations.
template <typename T>
__device__ __forceinline__ int gate_tip(const KParams<T>& p, const Smem<T>& s, int slot, int warp, int lane, int K) {
  const int m = s.target[slot];
  const int beg = __ldg(p.moff + m), end = __ldg(p.moff + m + 1);
  const double l0 = s.px[0 * NT + slot], l1 = s.px[1 * NT + slot];
  const T C00 = s.pC[tri(0, 0) * NT + slot], C01 = s.pC[tri(0, 1) * NT + slot], C11 = s.pC[tri(1, 1) * NT + slot];
  const T chi2_max = (T)p.cfg.chi2_max;
  T* cc = s.candchi2 + warp * CAND;
  int32_t* ci = s.candidx + warp * CAND;
  int count = 0;
  for (int k0 = beg; k0 < end; k0 += 32) {
    const int k = k0 + lane;
    bool pass = false;
    T c2 = T(0);
    if (k < end) {
      const auto lc = __ldg(p.loc + k);
      const auto vr = __ldg(p.var + k);
      pass = gate_chi2<T>(l0, l1, C00, C01, C11, lc.x, lc.y, vr.x, vr.y, chi2_max, c2);
    }
    const unsigned mask = __ballot_sync(0xffffffffu, pass);
    if (pass) {
      const int pos = count + __popc(mask & ((1u << lane) - 1u));
      if (pos < CAND) { cc[pos] = c2; ci[pos] = k; }
    }
    count += __popc(mask);
  }
  __syncwarp();
  int nsel;
  if (count <= CAND) {
    // fast path: rank the passers by (chi2, index)
    if (lane < count) {
      const T mc = cc[lane];
      const int mi = ci[lane];
      int rank = 0;
      for (int j = 0; j < count; ++j) rank += key_less<T>(cc[j], ci[j], mc, mi) ? 1 : 0;
      if (rank < K) { s.selchi2[rank * NT + slot] = mc; s.selidx[rank * NT + slot] = mi; }
    }
    nsel = count < K ? count : K;
  } else {
    // rare: more than CAND passers.  K rounds of "smallest key above the last one", recomputing chi2.
    T last_c = T(-1);
    int last_i = -1;
    for (int r = 0; r < K; ++r) {
      T bc = T(0);
      int bi = 0x7fffffff;
      for (int k = beg + lane; k < end; k += 32) {
        const auto lc = __ldg(p.loc + k);
        const auto vr = __ldg(p.var + k);
        T c2 = T(0);
        const bool ok = gate_chi2<T>(l0, l1, C00, C01, C11, lc.x, lc.y, vr.x, vr.y, chi2_max, c2);
        if (ok && key_less<T>(last_c, last_i, c2, k) && (bi == 0x7fffffff || key_less<T>(c2, k, bc, bi))) {
          bc = c2; bi = k;
        }
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        const T oc = __shfl_xor_sync(0xffffffffu, bc, o);
        const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
        if (oi != 0x7fffffff && (bi == 0x7fffffff || key_less<T>(oc, oi, bc, bi))) { bc = oc; bi = oi; }
      }
      if (lane == 0) { s.selchi2[r * NT + slot] = bc; s.selidx[r * NT + slot] = bi; }
      last_c = bc; last_i = bi;
    }
    nsel = K;
  }
  __syncwarp();
  return nsel;
}

template <typename T, int MINB>
__global__ void __launch_bounds__(NT, MINB) ckf_level_loop(const KParams<T> p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Smem<T> s;
  const int K = p.cfg.max_branches;
  s.carve(smem_raw, K);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int cap = p.cfg.max_cands;
  int2* Q0 = p.queue + (size_t)blockIdx.x * 2 * p.qcap;
  int2* Q1 = Q0 + p.qcap;
  if (tid < CNT_N) s.cnt[tid] = 0ull;
  if (tid == 0) { s.misc[M_NLIVE] = 0; }
  __syncthreads();
  const int fair = (p.n_seeds + gridDim.x - 1) / gridDim.x;
  unsigned long long my_trials = 0, my_accepted = 0, my_gate = 0, my_visits = 0, my_updates = 0;

  for (int iter = 0;; ++iter) {
    int2* Qin = (iter & 1) ? Q1 : Q0;
    int2* Qout = (iter & 1) ? Q0 : Q1;
    // ---------------- refill: pull seeds while the queue has room (continuous batching)
    if (tid == 0) {
      const int n_live = s.misc[M_NLIVE];
      int want = (NT - n_live) / 2;
      want = want > fair ? (fair > 0 ? fair : 1) : want;
      int base = 0, n = 0;
      if (want > 0 && *(volatile int32_t*)p.g_seed_cursor < p.n_seeds) {
        base = atomicAdd(p.g_seed_cursor, want);
        n = base < p.n_seeds ? min(want, p.n_seeds - base) : 0;
      }
      s.misc[M_PULL_BASE] = base;
      s.misc[M_PULL_N] = n;
    }
    __syncthreads();
    {
      const int n_live = s.misc[M_NLIVE], pn = s.misc[M_PULL_N], pb = s.misc[M_PULL_BASE];
      for (int i = tid; i < pn; i += NT) Qin[n_live + i] = make_int2(-(pb + i) - 1, pb + i);
      __syncthreads();
      if (tid == 0) { s.misc[M_NLIVE] = n_live + pn; s.misc[M_NOUT] = 0; }
      __syncthreads();
    }
    const int n_live = s.misc[M_NLIVE];
    if (n_live == 0) break;  // the pull returned nothing and nothing is alive: all seeds are taken

    // ---------------- passes of whole seeds, at most NT tips each
    for (int base = 0; base < n_live;) {
      if (tid == 0) s.misc[M_PASS_END] = base;
      __syncthreads();
      {
        const int pos = base + tid;
        if (pos < n_live) {
          const bool boundary = (pos + 1 == n_live) || (Qin[pos + 1].y != Qin[pos].y);
          if (boundary) atomicMax(&s.misc[M_PASS_END], pos + 1);
        }
      }
      __syncthreads();
      int n = s.misc[M_PASS_END] - base;  // >= 1 because max_candidates_per_seed <= NT
      if (n <= 0) n = min(NT, n_live - base);
      if (tid == 0) s.cnt[CNT_ITER] += 1ull;

      // ======== P1: thread per tip — load, navigate, propagate, predict (a3-a6)
      if (tid < n) {
        const int2 e = Qin[base + tid];
        const int seed = e.y;
        int link = e.x, stop = STOP_NONE, target = -1, counts = 0, lastmeas = -1;
        T c2s = T(0);
        if (link < 0) {
          // fresh seed: level 0 visits the seed's own module with identity transport (N6)
          link = -1;
          double x[6];
          bool ok = true;
#pragma unroll
          for (int i = 0; i < 6; ++i) { x[i] = (double)p.seed_x[(size_t)seed * 6 + i]; ok = ok && isfinite(x[i]); }
          ok = ok && (x[3] > 0.0 && x[3] < PI_D);
          target = p.seed_module[seed];
          if (!ok) stop = STOP_NUMERIC;
#pragma unroll
          for (int i = 0; i < 6; ++i) s.px[i * NT + tid] = x[i];
#pragma unroll
          for (int i = 0; i < 6; ++i)
#pragma unroll
            for (int j = i; j < 6; ++j) s.pC[tri(i, j) * NT + tid] = p.seed_C[(size_t)seed * 36 + i * 6 + j];
        } else {
          counts = p.lk_counts[link];
          lastmeas = p.lk_lastmeas[link];
          c2s = p.lk_chi2sum[link];
          const int level = (counts & 0xffff) + (counts >> 16);
          if (level >= p.cfg.max_levels) stop = STOP_LEVEL_LIMIT;
          else {
            double x[6], xp[6];
#pragma unroll
            for (int i = 0; i < 6; ++i) x[i] = p.lk_x[(size_t)i * p.max_links + link];
            const int from = p.lk_module[link];
            T J[5][5], qphi, qth;
            StepCtl sc;
            sc.n_trials = 0; sc.n_accepted = 0;
            stop = move_to_next_module<T>(p.geo, p.fld, p.cfg, from, x, target, xp, J, qphi, qth, sc);
            my_trials += sc.n_trials;
            my_accepted += sc.n_accepted;
            if (stop == STOP_NONE) {
              T C[21], Co[21];
#pragma unroll
              for (int i = 0; i < 21; ++i) C[i] = p.lk_C[(size_t)i * p.max_links + link];
              C[tri(2, 2)] += qphi;
              C[tri(3, 3)] += qth;
              transport_cov<T>(J, C, Co);
              bool fin = true;
#pragma unroll
              for (int i = 0; i < 21; ++i) { s.pC[i * NT + tid] = Co[i]; fin = fin && isfinite(Co[i]); }
#pragma unroll
              for (int i = 0; i < 6; ++i) s.px[i * NT + tid] = xp[i];
              if (!fin) stop = STOP_NUMERIC;
            }
          }
        }
        s.link[tid] = link; s.seed[tid] = seed; s.target[tid] = target; s.stop[tid] = stop;
        s.counts[tid] = counts; s.lastmeas[tid] = lastmeas; s.chi2sum[tid] = c2s;
      }
      __syncthreads();

      // ======== P2: warp per tip — chi2 gate over the module's CSR slice, k best (a7, a8)
      for (int i = warp; i < n; i += NW) {
        int nsel = 0, want = 0;
        if (s.stop[i] == STOP_NONE) {
          const int m = s.target[i];
          if (lane == 0) {
            my_gate += (unsigned long long)(__ldg(p.moff + m + 1) - __ldg(p.moff + m));
            my_visits += 1ull;
          }
          nsel = gate_tip<T>(p, s, i, warp, lane, K);
          if (lane == 0) {
            if (nsel == 0) {
              const int nh = (s.counts[i] >> 16) + 1;
              if (nh > p.cfg.max_holes) { s.stop[i] = STOP_HOLES; s.counts[i] += (1 << 16); }
              else want = 1;
            } else want = nsel;
          }
        }
        if (lane == 0) { s.nsel[i] = nsel; s.want[i] = want; }
      }
      __syncthreads();

      // ======== P3: per-seed cap R10 + prefix sums (a10)
      int my_want = 0, my_seed = -1, my_stop = 0, my_emit = 0, my_nm = 0;
      if (tid < n) {
        my_want = s.want[tid]; my_seed = s.seed[tid]; my_stop = s.stop[tid];
        my_nm = s.counts[tid] & 0xffff;
        my_emit = (my_stop != STOP_NONE && my_nm >= p.cfg.min_meas) ? 1 : 0;
      }
      const bool is_head = tid < n && (tid == 0 || s.seed[tid - 1] != my_seed);
      const bool is_tail = tid < n && (tid == n - 1 || s.seed[tid + 1] != my_seed);
      const int head = block_incl_max(is_head ? tid : 0, s.warp);
      int tot;
      const int e = my_want > 0 ? my_want - 1 : 0;
      const int Eex = block_excl_scan(e, s.warp, tot);
      s.Eex[tid] = Eex;
      const int Mex = block_excl_scan((my_emit << 16) | (my_emit ? my_nm : 0), s.warp, tot);
      s.Mex[tid] = Mex;
      if (tid == NT - 1) s.Mex[NT] = tot;
      int sd_extra = 0, sd_nemit = 0, sd_nent = 0;
      if (tid < n) { sd_extra = p.sd_extra[my_seed]; sd_nemit = p.sd_nemit[my_seed]; sd_nent = p.sd_nentries[my_seed]; }
      __syncthreads();
      int keep = 0;
      if (tid < n && my_want > 0) {
        const int Rm = cap - (1 + sd_extra);
        const int Pex = Eex - s.Eex[head];
        const int room = Rm - Pex;
        keep = 1 + min(e, room > 0 ? room : 0);
      }
      const int Kex = block_excl_scan(keep, s.warp, tot);
      s.Kex[tid] = Kex;
      if (tid == 0) {
        s.Kex[NT] = tot;
        int lb = 0, allowed = 0;
        if (tot > 0) {
          lb = atomicAdd(p.g_link_count, tot);
          allowed = p.max_links - lb;
          allowed = allowed < 0 ? 0 : (allowed > tot ? tot : allowed);
          if (allowed < tot) atomicOr(p.o_status, 4);
          const int room = p.qcap - s.misc[M_NOUT];
          if (allowed > room) { allowed = room; atomicOr(p.o_status, 4); }
        }
        s.misc[M_LINK_BASE] = lb;
        s.misc[M_ALLOWED] = allowed;
        s.cnt[CNT_TIPS] += (unsigned long long)n;
        s.cnt[CNT_LINKS] += (unsigned long long)allowed;
      }
      // emission records (a11) for tips that stopped at this level, in tip order within the seed
      if (tid < n) {
        if (keep > 1) atomicAdd(p.sd_extra + my_seed, keep - 1);
        if (my_emit) {
          const int hM = s.Mex[head];
          const int slot = sd_nemit + ((Mex >> 16) - (hM >> 16));
          const int eoff = sd_nent + ((Mex & 0xffff) - (hM & 0xffff));
          if (slot < cap) {
            const size_t li = (size_t)my_seed * cap + slot;
            p.leaf_link[li] = s.link[tid];
            p.leaf_meta[li] = my_stop | ((s.counts[tid] >> 16) << 8);
            p.leaf_entry[li] = eoff;
          }
        }
      }
      __syncthreads();
      if (is_tail) {
        const int incl = s.Mex[tid] + ((my_emit << 16) | (my_emit ? my_nm : 0));
        const int seg = incl - s.Mex[head];
        if (seg != 0) {
          p.sd_nemit[my_seed] = sd_nemit + (seg >> 16);
          p.sd_nentries[my_seed] = sd_nent + (seg & 0xffff);
        }
      }

      // ======== P4: thread per child — Kalman update or hole, link append, next queue (a9, a10)
      {
        const int allowed = s.misc[M_ALLOWED], lb = s.misc[M_LINK_BASE], n_out = s.misc[M_NOUT];
        for (int c = tid; c < allowed; c += NT) {
          // parent = last tip with Kex <= c
          int lo = 0, hi = n;  // invariant: Kex[lo] <= c < Kex[hi] (Kex[n] == total)
          while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            const int kv = (mid == n) ? s.Kex[NT] : s.Kex[mid];
            if (kv <= c) lo = mid; else hi = mid;
          }
          // tips with keep == 0 share Kex with their successor: walk to the one that owns c
          const int par = lo;
          const int j = c - s.Kex[par];
          const int link = lb + c;
          const int pc = s.counts[par];
          double x[6];
          T C[21];
#pragma unroll
          for (int i = 0; i < 6; ++i) x[i] = s.px[i * NT + par];
#pragma unroll
          for (int i = 0; i < 21; ++i) C[i] = s.pC[i * NT + par];
          int meas = -1, counts, lastmeas = s.lastmeas[par];
          T chi2 = T(0), c2s = s.chi2sum[par];
          if (s.nsel[par] == 0) {
            counts = pc + (1 << 16);
#pragma unroll
            for (int i = 0; i < 6; ++i) p.lk_x[(size_t)i * p.max_links + link] = x[i];
#pragma unroll
            for (int i = 0; i < 21; ++i) p.lk_C[(size_t)i * p.max_links + link] = C[i];
          } else {
            meas = s.selidx[j * NT + par];
            chi2 = s.selchi2[j * NT + par];
            const auto lc = __ldg(p.loc + meas);
            const auto vr = __ldg(p.var + meas);
            double xo[6];
            T Co[21];
            kalman_update<T>(x, C, lc.x, lc.y, vr.x, vr.y, xo, Co);
            counts = pc + 1;
            lastmeas = link;
            my_updates += 1ull;
            c2s += chi2;
#pragma unroll
            for (int i = 0; i < 6; ++i) p.lk_x[(size_t)i * p.max_links + link] = xo[i];
#pragma unroll
            for (int i = 0; i < 21; ++i) p.lk_C[(size_t)i * p.max_links + link] = Co[i];
          }
          p.lk_module[link] = s.target[par];
          p.lk_parent[link] = s.link[par];
          p.lk_meas[link] = meas;
          p.lk_chi2[link] = chi2;
          p.lk_chi2sum[link] = c2s;
          p.lk_counts[link] = counts;
          p.lk_lastmeas[link] = lastmeas;
          Qout[n_out + c] = make_int2(link, s.seed[par]);
        }
      }
      __syncthreads();
      if (tid == 0) s.misc[M_NOUT] += s.misc[M_ALLOWED];
      base += n;
      __syncthreads();
    }
    if (tid == 0) s.misc[M_NLIVE] = s.misc[M_NOUT];
    __syncthreads();
  }

  // ---------------- work counters
  for (int o = 16; o > 0; o >>= 1) {
    my_trials += __shfl_xor_sync(0xffffffffu, my_trials, o);
    my_accepted += __shfl_xor_sync(0xffffffffu, my_accepted, o);
    my_gate += __shfl_xor_sync(0xffffffffu, my_gate, o);
    my_visits += __shfl_xor_sync(0xffffffffu, my_visits, o);
    my_updates += __shfl_xor_sync(0xffffffffu, my_updates, o);
  }
  if (lane == 0) {
    atomicAdd(&s.cnt[CNT_TRIALS], my_trials);
    atomicAdd(&s.cnt[CNT_ACCEPTED], my_accepted);
    atomicAdd(&s.cnt[CNT_GATE], my_gate);
    atomicAdd(&s.cnt[CNT_VISITS], my_visits);
    atomicAdd(&s.cnt[CNT_UPDATES], my_updates);
  }
  __syncthreads();
  if (tid < CNT_N && s.cnt[tid] != 0ull) atomicAdd(p.counters + tid, s.cnt[tid]);
}

}  // namespace ckf
