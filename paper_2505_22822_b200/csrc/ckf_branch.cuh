// ckf_branch.cuh — branching of a level (a9-a11): per-seed cap + emission records, child offsets, and the
// children themselves (Kalman update or hole, link append, departure state of the next level).
#pragma once
#include "ckf_kernels.cuh"

namespace ckf {

// a10 (R10) + a11 + child offsets, one kernel.
//  1. Thread per tip: the tip looks BACK over the earlier tips of its seed at this level (a few on average, at
//     most max_candidates_per_seed) and so evaluates the sequential rules in closed form, independently of
//     every other thread: kept children (R10: exclusive prefix of the extra wants), emission slot and entry
//     offset (exclusive prefix of the emitting tips).  The seed's LAST tip also sees the seed's totals; it
//     parks them in t_fin* for ckf_update to apply to the per-seed counters (no thread reads a counter that
//     another thread of this launch writes).
//  2. Exclusive scan of the kept children: per-tile prefix (t_kex) + per-tile sums; the last block to finish
//     turns the sums into offsets, reserves the level's links (contiguous, so link ids are deterministic) and
//     publishes the next level's size.
template <typename T>
__global__ void __launch_bounds__(SCAN_NT) ckf_scan(const KParams<T> p, int level) {
  chain_enter();
  const int n = p.g[G_NTIPS0 + (level & 1)];
  if (n == 0) {
    if (blockIdx.x == 0 && threadIdx.x == 0) p.g[G_NTIPS0 + ((level + 1) & 1)] = 0;  // the slot held level - 1
    return;
  }
  const int nb = (n + SCAN_NT - 1) / SCAN_NT;
  __shared__ int s_w[SCAN_NT / 32];
  __shared__ int s_last;
  const size_t TC = (size_t)p.tcap;
  const int32_t* tlink = p.tip_link + (size_t)(level & 1) * TC;
  const int32_t* tseed = p.tip_seed + (size_t)(level & 1) * TC;
  const int cap = p.cfg.max_cands, min_meas = p.cfg.min_meas;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  for (int b = blockIdx.x; b < nb; b += gridDim.x) {
    const int t = b * SCAN_NT + tid;
    int keep = 0;
    if (t < n) {
      const int seed = tseed[t];
      const int want = p.t_want[t];
      const int e = want > 0 ? want - 1 : 0;
      const int stop = p.mv_stop[t], counts = p.t_counts[t], nm = counts & 0xffff;
      const bool emit = stop != STOP_NONE && nm >= min_meas;
      // look back over the seed's earlier tips of this level
      int P = 0, nemit_before = 0, nent_before = 0;
      for (int j = t - 1; j >= 0 && tseed[j] == seed; --j) {
        const int wj = p.t_want[j];
        P += wj > 0 ? wj - 1 : 0;
        const int cj = p.t_counts[j], nmj = cj & 0xffff;
        if (p.mv_stop[j] != STOP_NONE && nmj >= min_meas) { nemit_before += 1; nent_before += nmj; }
      }
      const int extra0 = p.sd_extra[seed];
      if (want > 0) {
        const int room = cap - (1 + extra0) - P;
        keep = 1 + min(e, room > 0 ? room : 0);
      }
      p.t_keep[t] = keep;
      const int nemit0 = p.sd_nemit[seed], nent0 = p.sd_nentries[seed];
      if (emit) {
        const int slot = nemit0 + nemit_before;
        if (slot < cap) {
          const size_t li = (size_t)seed * cap + slot;
          p.leaf_link[li] = tlink[t];
          p.leaf_meta[li] = stop | ((counts >> 16) << 8);
          p.leaf_entry[li] = nent0 + nent_before;
        }
      }
      const bool tail = (t + 1 == n) || (tseed[t + 1] != seed);
      if (tail) {
        // totals of the seed at this level: kept extras need every tip's keep, recomputed from the prefixes
        int KM = 0, Pj = 0;
        const int Rm = cap - (1 + extra0);
        int j0 = t;
        while (j0 > 0 && tseed[j0 - 1] == seed) --j0;
        for (int j = j0; j <= t; ++j) {
          const int wj = p.t_want[j];
          const int ej = wj > 0 ? wj - 1 : 0;
          if (wj > 0) { const int room = Rm - Pj; KM += min(ej, room > 0 ? room : 0); }
          Pj += ej;
        }
        p.t_fin[t] = seed;
        p.t_fin[TC + t] = extra0 + KM;
        p.t_fin[2 * TC + t] = nemit0 + nemit_before + (emit ? 1 : 0);
        p.t_fin[3 * TC + t] = nent0 + nent_before + (emit ? nm : 0);
      } else {
        p.t_fin[t] = -1;
      }
    }
    const int inc = warp_incl_scan(keep, lane);
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
    if (t < n) p.t_kex[t] = base + inc - keep;
    if (tid == 0) p.blk_sum[b] = tot;
  }
  __threadfence();
  __syncthreads();
  const int nblocks = min((int)gridDim.x, nb);
  if ((int)blockIdx.x >= nb) return;
  if (tid == 0) s_last = (atomicAdd(p.g + G_SCAN_TICKET, 1) == nblocks - 1) ? 1 : 0;
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
    for (int b = 0; b < NBIN; ++b) p.g[G_BIN0 + b] = 0;  // ckf_update of this level refills the step schedule
    p.blk_sum[nb] = tot;
    atomicAdd(p.counters + CNT_TIPS, (unsigned long long)n);
    atomicAdd(p.counters + CNT_LINKS, (unsigned long long)allowed);
    atomicAdd(p.counters + CNT_ITER, 1ull);
  }
}

// Parent tip of child c: the last tip whose global exclusive prefix (tile offset + in-tile prefix) is <= c; tips
// that keep nothing share their prefix with their successor, so "last" skips them.
template <typename T>
__device__ __forceinline__ int find_parent(const KParams<T>& p, int n, int nb, int c) {
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
  return a;
}

// Cost class of the move a live child is about to make = its predicted number of RKN4 trials (DESIGN.md §6,
// "step schedule").  A scheduling hint only: ckf_step processes the classes in descending order so that the
// lanes of a warp run moves of similar length and the launch ends on the short ones; results do not depend on
// it.  trials ~ 0.26 (gap / sin theta)^0.71 (0.6 |q/p| / sin theta)^0.27, fitted on configs[3] (r = 0.95).
__device__ __forceinline__ int step_cost_bin(const GeoDev& g, int module, const Traj& y, int overlap) {
  if (overlap >= 0) return 0;  // same-layer neighbour: one or two short trials
  const int L = g.mod[module].layer;
  const LayerRec LR = g.layer[L];
  const float st = sqrtf((float)(y.d[0] * y.d[0] + y.d[1] * y.d[1]));
  float path;  // rough length of the move: to the next cylinder, or from a disc to the next disc of its side
  if (LR.kind == 0) {
    if (L + 1 >= g.n_barrel) return 0;  // leaves the barrel at once
    path = (float)(g.layer[L + 1].r - LR.r) / st;
  } else {
    if (LR.next_disc < 0) return 0;
    path = fabsf((float)(g.layer[LR.next_disc].half_z - LR.half_z)) / fmaxf(fabsf((float)y.d[2]), 0.05f);
  }
  const float pred = 0.2565f * __powf(path, 0.713f) * __powf(0.6f * fabsf((float)y.qop) / st, 0.266f);
  const int b = (int)(pred * ((float)NBIN / 16.0f));  // NBIN / 16 classes per predicted trial
  return b < 1 ? 1 : (b > NBIN - 1 ? NBIN - 1 : b);
}

// a9 + a10: thread per child, in child order (parent tip order, then (chi2, index) rank): Kalman update or hole
// copy, link append, and the departure state (J1, V5) of the child as a tip of the next level.  Also applies the
// per-seed totals parked by ckf_scan.  The child -> parent search is staged: two threads bracket the block's
// 256 children in the global prefix, the bracket is copied to shared memory, every thread searches there.
constexpr int UPD_WIN = 1024;
// The same search by one WARP: every round probes 32 evenly spaced keys at once and keeps the sub-range that brackets c,
// so a range of n keys costs ceil(log32 n) dependent loads instead of log2 n.  key(i) must be non-decreasing and
// key(lo) <= c; returns the last i in [lo, hi) with key(i) <= c.
template <typename F>
__device__ __forceinline__ int warp_last_le(F key, int lo, int hi, int c, int lane) {
  while (hi - lo > 1) {
    const int step = (hi - lo + 31) / 32;
    const int idx = lo + (lane + 1) * step;
    const bool le = idx < hi && key(idx) <= c;
    const int m = __popc(__ballot_sync(0xffffffffu, le));  // the probes that are <= c form a prefix
    const int nlo = lo + m * step;
    hi = min(hi, nlo + step);
    lo = nlo;
  }
  return lo;
}
template <typename T>
__device__ __forceinline__ int find_parent_warp(const KParams<T>& p, int n, int nb, int c, int lane) {
  const int tile = warp_last_le([&](int i) { return p.blk_sum[i]; }, 0, nb, c, lane);
  const int boff = p.blk_sum[tile];
  const int a = tile * SCAN_NT, b = min(n, a + SCAN_NT);
  return warp_last_le([&](int i) { return boff + p.t_kex[i]; }, a, b, c, lane);
}
template <typename T>
#ifndef CKF_UPDATE_MINB
#define CKF_UPDATE_MINB 2
#endif
__global__ void __launch_bounds__(SCAN_NT, CKF_UPDATE_MINB) ckf_update(const KParams<T> p, int level) {
  chain_enter();
  const int n = p.g[G_NTIPS0 + (level & 1)];
  if (n == 0) return;
  const int nc = p.g[G_NTIPS0 + ((level + 1) & 1)];
  const size_t TC = (size_t)p.tcap;
  for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < n; t += gridDim.x * blockDim.x) {
    const int seed = p.t_fin[t];
    if (seed >= 0) {
      p.sd_extra[seed] = p.t_fin[TC + t];
      p.sd_nemit[seed] = p.t_fin[2 * TC + t];
      p.sd_nentries[seed] = p.t_fin[3 * TC + t];
    }
  }
  if (nc == 0) return;
  __shared__ int s_gk[UPD_WIN + 1];
  __shared__ int s_p[2];
  const int32_t* tlink = p.tip_link + (size_t)(level & 1) * TC;
  const int32_t* tseed = p.tip_seed + (size_t)(level & 1) * TC;
  int32_t* nlink = p.tip_link + (size_t)((level + 1) & 1) * TC;
  int32_t* nseed = p.tip_seed + (size_t)((level + 1) & 1) * TC;
  const int nb = (n + SCAN_NT - 1) / SCAN_NT;
  const int lbase = p.g[G_LBASE];
  unsigned long long my_updates = 0;
  for (int c0 = blockIdx.x * SCAN_NT; c0 < nc; c0 += gridDim.x * SCAN_NT) {
    const int c = c0 + threadIdx.x;
    __syncthreads();
    if (threadIdx.x < 64) {  // warp 0 brackets the block's first child, warp 1 its last
      const int w = threadIdx.x >> 5;
      const int r = find_parent_warp<T>(p, n, nb, w == 0 ? c0 : min(c0 + SCAN_NT, nc) - 1, threadIdx.x & 31);
      if ((threadIdx.x & 31) == 0) s_p[w] = r;
    }
    __syncthreads();
    const int p0 = s_p[0], win = s_p[1] - p0 + 1;
    int par;
    if (win <= UPD_WIN) {
      for (int i = threadIdx.x; i < win; i += SCAN_NT) s_gk[i] = p.blk_sum[(p0 + i) / SCAN_NT] + p.t_kex[p0 + i];
      __syncthreads();
      int a = 0, b = win;  // invariant: gk[a] <= c < gk[b] (virtual gk[win] = inf)
      if (c < nc) {
        while (b - a > 1) {
          const int mid = (a + b) >> 1;
          if (s_gk[mid] <= c) a = mid; else b = mid;
        }
      }
      par = p0 + a;
    } else {
      par = c < nc ? find_parent<T>(p, n, nb, c) : 0;
    }
    int bin = -1;
    if (c < nc) {
    const int j = c - (p.blk_sum[par / SCAN_NT] + p.t_kex[par]);
    const int nl = lbase + c;
    const int plink = tlink[par], seed = tseed[par];
    const int pc = p.t_counts[par];
    const int target = p.mv_tgt[par];
    double x[6], xo[6];
    double C[21];
#pragma unroll
    for (int i = 0; i < 6; ++i) x[i] = p.pd_x[i * TC + par];
#pragma unroll
    for (int i = 0; i < 21; ++i) C[i] = p.pd_C[i * TC + par];
    int meas = -1, ncounts, nlast = plink >= 0 ? p.lk_lastmeas[plink] : -1;
    T chi2 = T(0);
    double nc2s = plink >= 0 ? p.lk_chi2sum[plink] : 0.0;
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
      double Co[21];
      kalman_update(x, C, lc.x, lc.y, vr.x, vr.y, xo, Co);
      ncounts = pc + 1;
      nlast = nl;
      my_updates += 1ull;
      nc2s += (double)chi2;
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
      double dep[NDEP];
      stop = departure_state(p.geo, p.cfg, target, xo, y, dep);
      if (stop == STOP_NONE) {
        store_traj(p.mv_y, (size_t)c, y);
#pragma unroll
        for (int i = 0; i < NDEP; ++i) p.mv_dep[i * TC + c] = dep[i];
        // N2 here, at full lanes, instead of inside the RKN4 kernel: the overlap neighbour of the child's departure
        const int ov = overlap_neighbour(p.geo, target, y.r, y.d);
        p.mv_tgt[TC + c] = ov;
        bin = step_cost_bin(p.geo, target, y, ov);
      }
    }
    p.mv_stop[c] = stop;
    }
    // step schedule: append the live child to its cost class (one atomic per class present in the warp)
    const unsigned live = __ballot_sync(0xffffffffu, bin >= 0);
    if (bin >= 0) {
      const int lane = threadIdx.x & 31;
      const unsigned peers = __match_any_sync(live, bin);
      const int leader = __ffs(peers) - 1;
      int base = 0;
      if (lane == leader) base = atomicAdd(p.g + G_BIN0 + bin, __popc(peers));
      base = __shfl_sync(peers, base, leader);
      p.mv_order[(size_t)bin * TC + base + __popc(peers & ((1u << lane) - 1u))] = c;
    }
  }
  flush_counter(p.counters + CNT_UPDATES, my_updates);
}

}  // namespace ckf
