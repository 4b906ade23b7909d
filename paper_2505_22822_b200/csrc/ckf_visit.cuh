// ckf_visit.cuh — arrival on the module and the visit (a6-a8): one warp per 32 consecutive tips of the level.
//   lane per tip : arrival Jacobian (J4, J5), C' = J (C + Q) J^T, predicted (x, C) -> shared + global
//   whole warp   : chi2 gate over the loc0 windows of the sorted slices, as flattened (tip, measurement) pairs
//   lane per tip : k best by (chi2, index), hole rule (V4)
#pragma once
#include "ckf_kernels.cuh"

namespace ckf {

// Shared memory of ONE warp (sizes depend on max_branches K).  Arrays are [..][32], tip (lane) index fastest.
template <typename T>
struct VSmem {
  double* px;       // [6][32] predicted bound parameters
  double* pC;       // [21][32] predicted packed covariance
  T* selchi2;       // [K][32]
  int32_t* selidx;  // [K][32]
  T* candchi2;      // [CAND][32]
  int32_t* candidx; // [CAND][32]
  int32_t *target, *lo, *cnt;  // [32] each
  int32_t* off;     // [33]
  __host__ __device__ static size_t bytes(int K) {
    size_t b = sizeof(double) * 6 * 32 + sizeof(double) * 21 * 32 + (sizeof(T) + 4) * (size_t)K * 32 +
               (sizeof(T) + 4) * (size_t)CAND * 32 + 4 * 3 * 32 + 4 * 33;
    return (b + 15) & ~(size_t)15;
  }
  __device__ void carve(unsigned char* raw, int K) {
    unsigned char* p = raw;
    px = (double*)p; p += sizeof(double) * 6 * 32;
    pC = (double*)p; p += sizeof(double) * 21 * 32;
    selchi2 = (T*)p; p += sizeof(T) * (size_t)K * 32;
    candchi2 = (T*)p; p += sizeof(T) * (size_t)CAND * 32;
    selidx = (int32_t*)p; p += 4 * (size_t)K * 32;
    candidx = (int32_t*)p; p += 4 * (size_t)CAND * 32;
    target = (int32_t*)p; p += 4 * 32;
    lo = (int32_t*)p; p += 4 * 32;
    cnt = (int32_t*)p; p += 4 * 32;
    off = (int32_t*)p; p += 4 * 33;
  }
};

// a7, a8: gate of the <= 32 tips of a warp.  Lane = tip for the window search and the ranking; the chi2 tests
// run over the FLATTENED (tip, measurement) pairs of all windows, 32 pairs per round, so the lanes stay full
// whatever the individual window lengths are.  Passers of a tip are collected in any order (shared-memory
// counter) and then ranked by (chi2, index), which makes the result order-independent.
// Returns the number of selected measurements of this lane's tip, written in rank order to sel*[rank][lane].
template <typename T>
__device__ __forceinline__ int gate_chunk(const KParams<T>& p, const VSmem<T>& s, int lane, bool visit, int K,
                                          unsigned long long& n_exec) {
  const double chi2_max = p.cfg.chi2_max;
  int lo = 0, len = 0;
  if (visit) {
    const int m = s.target[lane];
    int beg, end;
    slice_of<T>(p, m, beg, end);
    int hi = end;
    lo = beg;
    if (end > beg) {
      const T v0max = p.s_v0max[m];
      const double C00 = s.pC[tri(0, 0) * 32 + lane], C01 = s.pC[tri(0, 1) * 32 + lane], C11 = s.pC[tri(1, 1) * 32 + lane];
      if (v0max >= T(0) && C00 > 0.0 && C11 > 0.0 && C00 * C11 - C01 * C01 > 0.0) {
        // chi2 >= r0^2 / S00 and S00 <= C00 + v0max: nothing outside |loc0 - l0| <= w can pass
        const double w = sqrt(p.cfg.chi2_max * (C00 + (double)v0max)) * (1.0 + 1e-6) + 1e-9;
        if (isfinite(w)) {
          const double l0 = s.px[0 * 32 + lane];
          const double a = l0 - w, b = l0 + w;
          // both ends of the window at once: the two chains of dependent loads overlap
          int x0 = beg, x1 = end;  // first k with loc0[k] >= a
          int y0 = beg, y1 = end;  // first k with loc0[k] > b
          while (x0 < x1 || y0 < y1) {
            const int mx = (x0 + x1) >> 1, my = (y0 + y1) >> 1;
            const double vx = x0 < x1 ? (double)p.s_loc[mx].x : 0.0;
            const double vy = y0 < y1 ? (double)p.s_loc[my].x : 0.0;
            if (x0 < x1) { if (vx < a) x0 = mx + 1; else x1 = mx; }
            if (y0 < y1) { if (vy <= b) y0 = my + 1; else y1 = my; }
          }
          lo = x0;
          hi = y0;
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
      const int oi = p.s_idx[k];  // loaded with the rest (coalesced), not after the test by the few lanes that pass
      double c2 = 0.0;
      const bool pass = gate_chi2<T>(s.px[0 * 32 + t], s.px[1 * 32 + t], s.pC[tri(0, 0) * 32 + t],
                                     s.pC[tri(0, 1) * 32 + t], s.pC[tri(1, 1) * 32 + t], lc.x, lc.y, vr.x, vr.y,
                                     chi2_max, c2);
      if (pass) {
        const int pos = atomicAdd(&s.cnt[t], 1);
        if (pos < CAND) { s.candchi2[pos * 32 + t] = (T)c2; s.candidx[pos * 32 + t] = oi; }
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
      const double C00 = s.pC[tri(0, 0) * 32 + lane], C01 = s.pC[tri(0, 1) * 32 + lane], C11 = s.pC[tri(1, 1) * 32 + lane];
      T last_c = T(-1);
      int last_i = -1;
      nsel = count < K ? count : K;
      for (int r = 0; r < nsel; ++r) {
        T bc = T(0);
        int bi = 0x7fffffff;
        for (int k = lo; k < lo + len; ++k) {
          const auto lc = p.s_loc[k];
          const auto vr = p.s_var[k];
          double c2d = 0.0;
          const bool ok = gate_chi2<T>(l0, l1, C00, C01, C11, lc.x, lc.y, vr.x, vr.y, chi2_max, c2d);
          const T c2 = (T)c2d;
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

template <typename T, int MINB, bool GRAD = false>
__global__ void __launch_bounds__(VISIT_NT, MINB) ckf_visit(const KParams<T> p, int level) {
  chain_enter();
  const int n = p.g[G_NTIPS0 + (level & 1)];
  if (n == 0) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int K = p.cfg.max_branches;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  VSmem<T> s;
  s.carve(smem_raw + (size_t)wib * VSmem<T>::bytes(K), K);
  const size_t TC = (size_t)p.tcap;
  const int32_t* tlink = p.tip_link + (size_t)(level & 1) * TC;
  const int32_t* tseed = p.tip_seed + (size_t)(level & 1) * TC;
  const int gw = blockIdx.x * (VISIT_NT / 32) + wib, nw = gridDim.x * (VISIT_NT / 32);
  unsigned long long my_gate = 0, my_visits = 0, w_exec = 0;

  for (int t0 = gw * 32; t0 < n; t0 += nw * 32) {
    const int t = t0 + lane;
    const bool act = t < n;
    int stop = STOP_NONE, target = -1, counts = 0;
    if (act) {
      const int link = tlink[t];
      if (link < 0) {
        // fresh seed: level 0 visits the seed's own module with identity transport (N6)
        const int seed = tseed[t];
        bool ok = true;
#pragma unroll
        for (int i = 0; i < 6; ++i) {
          const double v = (double)p.seed_x[(size_t)seed * 6 + i];
          ok = ok && isfinite(v);
          if (i == 3) ok = ok && (v > 0.0 && v < PI_D);
          s.px[i * 32 + lane] = v;
          p.pd_x[i * TC + t] = v;
        }
#pragma unroll
        for (int i = 0; i < 6; ++i)
#pragma unroll
          for (int j = i; j < 6; ++j) {
            const double c = (double)p.seed_C[(size_t)seed * 36 + i * 6 + j];
            s.pC[tri(i, j) * 32 + lane] = c;
            p.pd_C[tri(i, j) * TC + t] = c;
          }
        const int eoff = p.sd_eoff[seed];
        if (eoff < 0) ok = false;     // seed module out of range (flagged by ckf_init_event): never used as an index
        target = ok ? p.seed_module[seed] - eoff : -1;
        p.mv_tgt[t] = target;
        if (!ok) stop = STOP_NUMERIC;
      } else {
        counts = p.lk_counts[link];
        stop = p.mv_stop[t];
        if (stop == STOP_NONE) {
          // arrival (J4, J5) and covariance transport
          Move<T> m;
          load_traj(p.mv_y, (size_t)t, m.y);
          load_jac(p.mv_D, (size_t)t, m.D);
          m.from = p.mv_from[t];
          m.tgt = p.mv_tgt[t];
          double dep[NDEP];
#pragma unroll
          for (int i = 0; i < NDEP; ++i) dep[i] = p.mv_dep[i * TC + t];
          double xp[6];
          double J[5][5];
          if constexpr (GRAD) {
            JacR<T> R;
            load_jacr(p.mv_Dr, (size_t)t, R);
            stop = move_arrive<T>(m, dep, p.geo, p.fld, p.cfg, xp, J, &R);
          } else {
            stop = move_arrive<T>(m, dep, p.geo, p.fld, p.cfg, xp, J);
          }
          if (stop == STOP_NONE) {
            target = m.tgt;
            double C[21], Co[21];
#pragma unroll
            for (int i = 0; i < 21; ++i) C[i] = p.lk_C[(size_t)i * p.max_links + link];
            leave_module_cov(C, dep);
            transport_cov<double>(J, C, Co);
            bool fin = true;
#pragma unroll
            for (int i = 0; i < 21; ++i) { s.pC[i * 32 + lane] = Co[i]; p.pd_C[i * TC + t] = Co[i]; fin = fin && isfinite(Co[i]); }
#pragma unroll
            for (int i = 0; i < 6; ++i) { s.px[i * 32 + lane] = xp[i]; p.pd_x[i * TC + t] = xp[i]; }
            if (!fin) stop = STOP_NUMERIC;
          }
        }
      }
    }
    const int vtarget = (act && target >= 0) ? target + p.sd_eoff[tseed[t]] : target;  // slice of the tip's own event
    s.target[lane] = vtarget;
    __syncwarp();
    const bool visit = act && stop == STOP_NONE;
    if (visit) {
      int sb, se;
      slice_of<T>(p, vtarget, sb, se);
      my_gate += (unsigned long long)(se - sb);
      my_visits += 1ull;
    }
    const int nsel = gate_chunk<T>(p, s, lane, visit, K, w_exec);
    int want = 0;
    if (visit) {
      if (nsel == 0) {
        const int nh = (counts >> 16) + 1;
        if (nh > p.cfg.max_holes) { stop = STOP_HOLES; counts += (1 << 16); }  // V4: the fatal hole is counted
        else want = 1;
      } else want = nsel;
      for (int r = 0; r < nsel; ++r) {
        p.sel_chi2[r * TC + t] = s.selchi2[r * 32 + lane];
        p.sel_idx[r * TC + t] = s.selidx[r * 32 + lane];
      }
    }
    if (act) {
      p.t_nsel[t] = nsel;
      p.t_want[t] = want;
      p.t_counts[t] = counts;
      p.mv_stop[t] = stop;
    }
    __syncwarp();
  }
  flush_counter(p.counters + CNT_GATE, my_gate);
  flush_counter(p.counters + CNT_VISITS, my_visits);
  flush_counter(p.counters + CNT_GATE_EXEC, w_exec);
}

}  // namespace ckf
