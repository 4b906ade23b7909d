// ckf_branch.cuh — branching of a level (a9-a11): per-seed cap + emission records, child offsets, and the
// children themselves (Kalman update or hole, link append, departure state of the next level).
#pragma once
#include "ckf_kernels.cuh"

namespace ckf {

// a10 (R10) + a11: the thread of a seed's FIRST tip of the level walks the seed's tips in order, so the greedy
// cap and the emission slots are the sequential rule itself and only one thread touches the seed's counters.
// Seeds hold a few tips on average (at most max_candidates_per_seed), so the walk is short.
template <typename T>
__global__ void __launch_bounds__(SCAN_NT) ckf_cap(const KParams<T> p, int level) {
  const int n = p.g[G_NTIPS0 + (level & 1)];
  if (n == 0) return;
  const size_t TC = (size_t)p.tcap;
  const int32_t* tlink = p.tip_link + (size_t)(level & 1) * TC;
  const int32_t* tseed = p.tip_seed + (size_t)(level & 1) * TC;
  const int cap = p.cfg.max_cands;
  for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < n; t += gridDim.x * blockDim.x) {
    const int seed = tseed[t];
    if (t > 0 && tseed[t - 1] == seed) continue;  // not the seed's first tip
    const int extra0 = p.sd_extra[seed];
    const int Rm = cap - (1 + extra0);
    int P = 0, KM = 0, nemit = p.sd_nemit[seed], nent = p.sd_nentries[seed];
    for (int j = t; j < n && tseed[j] == seed; ++j) {
      const int want = p.t_want[j];
      const int e = want > 0 ? want - 1 : 0;
      int keep = 0;
      if (want > 0) {
        const int room = Rm - P;
        keep = 1 + min(e, room > 0 ? room : 0);
      }
      P += e;
      KM += keep > 1 ? keep - 1 : 0;
      p.t_keep[j] = keep;
      // emission record of a tip that stopped at this level, in tip order within the seed
      const int stop = p.mv_stop[j], counts = p.t_counts[j], nm = counts & 0xffff;
      if (stop != STOP_NONE && nm >= p.cfg.min_meas) {
        if (nemit < cap) {
          const size_t li = (size_t)seed * cap + nemit;
          p.leaf_link[li] = tlink[j];
          p.leaf_meta[li] = stop | ((counts >> 16) << 8);
          p.leaf_entry[li] = nent;
        }
        nemit += 1;
        nent += nm;
      }
    }
    if (KM) p.sd_extra[seed] = extra0 + KM;
    p.sd_nemit[seed] = nemit;
    p.sd_nentries[seed] = nent;
  }
}

// Exclusive scan of t_keep over the level's tips: per-tile prefix (t_kex) + per-tile sums; the last tile to
// finish turns the sums into offsets, reserves the level's links (contiguous, so link ids are deterministic)
// and publishes the next level's size.
template <typename T>
__global__ void __launch_bounds__(SCAN_NT) ckf_scan(const KParams<T> p, int level) {
  const int n = p.g[G_NTIPS0 + (level & 1)];
  const int nb = n > 0 ? (n + SCAN_NT - 1) / SCAN_NT : 1;
  if ((int)blockIdx.x >= nb) return;
  __shared__ int s_w[SCAN_NT / 32];
  __shared__ int s_last;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  {
    const int t = blockIdx.x * SCAN_NT + tid;
    const int v = t < n ? p.t_keep[t] : 0;
    const int inc = warp_incl_scan(v, lane);
    if (lane == 31) s_w[w] = inc;
    __syncthreads();
    int base = 0, tot = 0;
#pragma unroll
    for (int i = 0; i < SCAN_NT / 32; ++i) {
      const int x = s_w[i];
      if (i < w) base += x;
      tot += x;
    }
    if (t < n) p.t_kex[t] = base + inc - v;
    if (tid == 0) p.blk_sum[blockIdx.x] = tot;
  }
  __threadfence();
  __syncthreads();
  if (tid == 0) s_last = (atomicAdd(p.g + G_SCAN_TICKET, 1) == nb - 1) ? 1 : 0;
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  // exclusive scan of the tile sums, SCAN_NT at a time with a running carry
  int carry = 0;
  for (int b0 = 0; b0 < nb; b0 += SCAN_NT) {
    const int b = b0 + tid;
    const int v = b < nb ? ((volatile int32_t*)p.blk_sum)[b] : 0;
    const int inc = warp_incl_scan(v, lane);
    __syncthreads();
    if (lane == 31) s_w[w] = inc;
    __syncthreads();
    int base = 0, tot = 0;
#pragma unroll
    for (int i = 0; i < SCAN_NT / 32; ++i) {
      const int x = s_w[i];
      if (i < w) base += x;
      tot += x;
    }
    if (b < nb) p.blk_sum[b] = carry + base + inc - v;
    carry += tot;
  }
  if (tid == 0) {
    const int tot = carry;
    const int lbase = p.g[G_LINK_COUNT];
    int allowed = p.max_links - lbase;
    allowed = allowed < 0 ? 0 : (allowed > tot ? tot : allowed);
    if (allowed > p.tcap) allowed = p.tcap;
    if (allowed < tot) atomicOr(p.o_status, 4);
    p.g[G_LBASE] = lbase;
    p.g[G_LINK_COUNT] = lbase + allowed;
    p.g[G_NTIPS0 + ((level + 1) & 1)] = allowed;
    p.g[G_STEP_CURSOR] = 0;
    p.g[G_SCAN_TICKET] = 0;
    p.blk_sum[nb] = tot;
    atomicAdd(p.counters + CNT_TIPS, (unsigned long long)n);
    atomicAdd(p.counters + CNT_LINKS, (unsigned long long)allowed);
    atomicAdd(p.counters + CNT_ITER, 1ull);
  }
}

// a9 + a10: thread per child, in child order (parent tip order, then (chi2, index) rank): Kalman update or hole
// copy, link append, and the departure state (J1, V5) of the child as a tip of the next level.
template <typename T>
__global__ void __launch_bounds__(SCAN_NT) ckf_update(const KParams<T> p, int level) {
  const int n = p.g[G_NTIPS0 + (level & 1)];
  const int nc = p.g[G_NTIPS0 + ((level + 1) & 1)];
  if (n == 0 || nc == 0) return;
  const size_t TC = (size_t)p.tcap;
  const int32_t* tlink = p.tip_link + (size_t)(level & 1) * TC;
  const int32_t* tseed = p.tip_seed + (size_t)(level & 1) * TC;
  int32_t* nlink = p.tip_link + (size_t)((level + 1) & 1) * TC;
  int32_t* nseed = p.tip_seed + (size_t)((level + 1) & 1) * TC;
  const int nb = (n + SCAN_NT - 1) / SCAN_NT;
  const int lbase = p.g[G_LBASE];
  unsigned long long my_updates = 0;
  for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < nc; c += gridDim.x * blockDim.x) {
    // parent = last tip whose exclusive prefix is <= c (tips that keep nothing share it with their successor)
    int lo = 0, hi = nb;  // invariant: blk_sum[lo] <= c < blk_sum[hi]  (blk_sum[nb] = total)
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (p.blk_sum[mid] <= c) lo = mid; else hi = mid;
    }
    const int boff = p.blk_sum[lo];
    int a = lo * SCAN_NT, b = min(n, a + SCAN_NT);  // invariant: kex[a] <= c - boff < kex[b] (virtual kex[b] = inf)
    while (b - a > 1) {
      const int mid = (a + b) >> 1;
      if (boff + p.t_kex[mid] <= c) a = mid; else b = mid;
    }
    const int par = a;
    const int j = c - (boff + p.t_kex[par]);
    const int nl = lbase + c;
    const int plink = tlink[par], seed = tseed[par];
    const int pc = p.t_counts[par];
    const int target = p.mv_tgt[par];
    double x[6], xo[6];
    T C[21];
#pragma unroll
    for (int i = 0; i < 6; ++i) x[i] = p.pd_x[i * TC + par];
#pragma unroll
    for (int i = 0; i < 21; ++i) C[i] = p.pd_C[i * TC + par];
    int meas = -1, ncounts, nlast = plink >= 0 ? p.lk_lastmeas[plink] : -1;
    T chi2 = T(0), nc2s = plink >= 0 ? p.lk_chi2sum[plink] : T(0);
    if (p.t_nsel[par] == 0) {
      ncounts = pc + (1 << 16);
#pragma unroll
      for (int i = 0; i < 6; ++i) { xo[i] = x[i]; p.lk_x[(size_t)i * p.max_links + nl] = x[i]; }
#pragma unroll
      for (int i = 0; i < 21; ++i) p.lk_C[(size_t)i * p.max_links + nl] = C[i];
    } else {
      meas = p.sel_idx[j * TC + par];
      chi2 = p.sel_chi2[j * TC + par];
      const auto lc = __ldg(p.loc + meas);
      const auto vr = __ldg(p.var + meas);
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
    p.lk_module[nl] = target;
    p.lk_parent[nl] = plink;
    p.lk_meas[nl] = meas;
    p.lk_chi2[nl] = chi2;
    p.lk_chi2sum[nl] = nc2s;
    p.lk_counts[nl] = ncounts;
    p.lk_lastmeas[nl] = nlast;
    // the child as a tip of the next level
    nlink[c] = nl;
    nseed[c] = seed;
    p.mv_from[c] = target;
    int stop = STOP_NONE;
    if ((ncounts & 0xffff) + (ncounts >> 16) >= p.cfg.max_levels) stop = STOP_LEVEL_LIMIT;
    else {
      Traj y;
      T dep[5];
      stop = departure_state<T>(p.geo, p.cfg, target, xo, y, dep);
      if (stop == STOP_NONE) {
#pragma unroll
        for (int i = 0; i < 3; ++i) { p.mv_y[i * TC + c] = y.r[i]; p.mv_y[(3 + i) * TC + c] = y.d[i]; }
        p.mv_y[6 * TC + c] = y.t;
        p.mv_y[7 * TC + c] = y.qop;
#pragma unroll
        for (int i = 0; i < 5; ++i) p.mv_dep[i * TC + c] = dep[i];
      }
    }
    p.mv_stop[c] = stop;
  }
  flush_counter(p.counters + CNT_UPDATES, my_updates);
}

}  // namespace ckf
