// ckf_sort.cuh — per-event gate index (a7): every module's CSR slice re-ordered by loc0.
//
// chi2 = r^T S^-1 r >= r0^2 / S00 for a positive-definite 2x2 S, so a measurement can only pass the gate
// chi2 < chi2_max if |loc0 - l0| < sqrt(chi2_max (C00 + var0)).  With the slice sorted by loc0 and the
// slice's largest var0 known, the gate of a tip is a binary search for that window plus chi2 on the few
// entries inside it, instead of chi2 on the whole slice (inner-layer modules of configs[3] hold ~500
// measurements, a tip's window ~1-30).  The passer set, hence every result, is unchanged.
#pragma once
#include <climits>
#include "ckf_kernels.cuh"

namespace ckf {

// Slices of at most 32 measurements (most modules) are rank-sorted by ONE warp with shuffles, four modules per
// block at a time; slices of up to SORT_WARP_MAX by one warp through shared memory; longer slices by the whole block
// with a bitonic sort in shared memory.  Slices longer than
// SORT_CAP, or holding a variance that is not a positive finite number, are copied through unsorted and flagged
// (s_v0max < 0): their tips gate the whole slice.
template <typename T>
__device__ __forceinline__ void sort_slice_warp(const KParams<T>& p, int m, int beg, int n, int lane) {
  if (n <= 0) {
    if (lane == 0) p.s_v0max[m] = T(0);
    return;
  }
  T key = (T)INFINITY, vmax = T(0);
  int id = INT_MAX;
  bool bad = false;
  typename Vec2<T>::type lc, vr;
  if (lane < n) {
    id = beg + lane;
    lc = p.loc[id];
    vr = p.var[id];
    key = lc.x;
    if (!(key == key)) key = (T)INFINITY;  // NaN sorts last; it can never pass the gate
    bad = !(vr.x > T(0)) || !(vr.y > T(0)) || !isfinite(vr.x) || !isfinite(vr.y);
    vmax = vr.x;
  }
  const bool any_bad = __any_sync(0xffffffffu, bad);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const T ov = __shfl_xor_sync(0xffffffffu, vmax, o);
    vmax = ov > vmax ? ov : vmax;
  }
  int rank = 0;
  for (int j = 0; j < n; ++j) {
    const T kj = __shfl_sync(0xffffffffu, key, j);
    const int ij = __shfl_sync(0xffffffffu, id, j);
    rank += key_less<T>(kj, ij, key, id) ? 1 : 0;
  }
  if (any_bad) rank = lane;
  if (lane < n) {
    p.s_loc[beg + rank] = lc;
    p.s_var[beg + rank] = vr;
    p.s_idx[beg + rank] = id;
  }
  if (lane == 0) p.s_v0max[m] = any_bad ? T(-1) : vmax;
}

// Slices of 33 .. SORT_WARP_MAX measurements: still one warp, keys staged in the warp's own shared-memory strip, every
// lane ranks its (up to SORT_WARP_MAX / 32) keys against all of them (broadcast reads).  Same order as the other paths:
// ascending (loc0, index), NaN last.
constexpr int SORT_WARP_MAX = 128;
template <typename T>
__device__ __forceinline__ void sort_slice_warp_mid(const KParams<T>& p, int m, int beg, int n, int lane, T* wkey) {
  constexpr int PER = SORT_WARP_MAX / 32;
  typename Vec2<T>::type lc[PER], vr[PER];
  T vmax = T(0);
  bool bad = false;
#pragma unroll
  for (int k = 0; k < PER; ++k) {
    const int i = lane + 32 * k;
    if (i < n) {
      lc[k] = p.loc[beg + i];
      vr[k] = p.var[beg + i];
      T key = lc[k].x;
      if (!(key == key)) key = (T)INFINITY;
      wkey[i] = key;
      bad = bad || !(vr[k].x > T(0)) || !(vr[k].y > T(0)) || !isfinite(vr[k].x) || !isfinite(vr[k].y);
      vmax = vr[k].x > vmax ? vr[k].x : vmax;
    }
  }
  __syncwarp();
  const bool any_bad = __any_sync(0xffffffffu, bad);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const T ov = __shfl_xor_sync(0xffffffffu, vmax, o);
    vmax = ov > vmax ? ov : vmax;
  }
  int rank[PER];
#pragma unroll
  for (int k = 0; k < PER; ++k) rank[k] = 0;
  if (!any_bad) {
    T key[PER];
#pragma unroll
    for (int k = 0; k < PER; ++k) key[k] = (lane + 32 * k < n) ? wkey[lane + 32 * k] : (T)INFINITY;
    for (int j = 0; j < n; ++j) {
      const T kj = wkey[j];
#pragma unroll
      for (int k = 0; k < PER; ++k) rank[k] += key_less<T>(kj, j, key[k], lane + 32 * k) ? 1 : 0;
    }
  }
#pragma unroll
  for (int k = 0; k < PER; ++k) {
    const int i = lane + 32 * k;
    if (i < n) {
      const int r = any_bad ? i : rank[k];
      p.s_loc[beg + r] = lc[k];
      p.s_var[beg + r] = vr[k];
      p.s_idx[beg + r] = beg + i;
    }
  }
  if (lane == 0) p.s_v0max[m] = any_bad ? T(-1) : vmax;
  __syncwarp();  // the strip is reused by the warp's next module
}

// Module m of (round r, block b, warp w) is r * G * MPB + w * G + b (G = gridDim.x): consecutive modules -- the crowded
// inner-layer ones have consecutive ids -- land on different blocks.  A warp sorts its module if the slice holds at
// most SORT_WARP_MAX measurements; the longer ones of a round are then sorted by the whole block, one after the other.
template <typename T>
__global__ void __launch_bounds__(SORT_NT) ckf_sort_slices(const KParams<T> p) {
  chain_enter();
  __shared__ T s_key[SORT_CAP];
  __shared__ int32_t s_id[SORT_CAP];
  __shared__ T s_red[SORT_NT / 32];
  __shared__ int s_bad;
  constexpr int MPB = SORT_NT / 32;  // modules taken per block and round, one per warp
  __shared__ T s_wkey[MPB][SORT_WARP_MAX];
  __shared__ int s_long[MPB];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int G = gridDim.x;
  for (int m0 = 0; m0 < p.n_vmod; m0 += G * MPB) {   // same trip count for every thread of the block
    const int mw = m0 + warp * G + (int)blockIdx.x;
    int is_long = -1;
    if (mw < p.n_vmod) {
      int begw, endw;
      slice_of<T>(p, mw, begw, endw);
      const int nw = endw - begw;
      if (lane == 0) {  // malformed CSR: flagged, and every reader clamps the slice the same way
        const int rb = __ldg(p.moff + mw), re = __ldg(p.moff + mw + 1);
        if (rb != begw || re != endw) atomicOr(p.g + G_BAD_INPUT, 1);
      }
      if (nw <= 32) sort_slice_warp<T>(p, mw, begw, nw, lane);
      else if (nw <= SORT_WARP_MAX) sort_slice_warp_mid<T>(p, mw, begw, nw, lane, s_wkey[warp]);
      else is_long = mw;
    }
    if (lane == 0) s_long[warp] = is_long;
    __syncthreads();
    for (int q = 0; q < MPB; ++q) {
      const int m = s_long[q];
      if (m < 0) continue;
      int beg, end;
      slice_of<T>(p, m, beg, end);
      const int n = end - beg;
      __syncthreads();
      if (tid == 0) s_bad = 0;
      __syncthreads();
      // largest var0 and validity of the slice's variances
      T vmax = T(0);
      bool bad = false;
      for (int i = tid; i < n; i += SORT_NT) {
        const auto vr = p.var[beg + i];
        bad = bad || !(vr.x > T(0)) || !(vr.y > T(0)) || !isfinite(vr.x) || !isfinite(vr.y);
        vmax = vr.x > vmax ? vr.x : vmax;
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        const T ov = __shfl_xor_sync(0xffffffffu, vmax, o);
        vmax = ov > vmax ? ov : vmax;
      }
      if (lane == 0) s_red[warp] = vmax;
      if (bad) s_bad = 1;
      __syncthreads();
      const bool unsorted = (s_bad != 0) || n > SORT_CAP;
      if (unsorted) {
        for (int i = tid; i < n; i += SORT_NT) {
          p.s_loc[beg + i] = p.loc[beg + i];
          p.s_var[beg + i] = p.var[beg + i];
          p.s_idx[beg + i] = beg + i;
        }
        if (tid == 0) p.s_v0max[m] = T(-1);
        continue;
      }
      int P = 64;
      while (P < n) P <<= 1;
      for (int i = tid; i < P; i += SORT_NT) {
        T key = (T)INFINITY;
        int id = INT_MAX;
        if (i < n) {
          key = p.loc[beg + i].x;
          if (!(key == key)) key = (T)INFINITY;  // NaN sorts last; it can never pass the gate
          id = beg + i;
        }
        s_key[i] = key;
        s_id[i] = id;
      }
      __syncthreads();
      // bitonic sort, ascending by (loc0, index)
      for (int kk = 2; kk <= P; kk <<= 1) {
        for (int j = kk >> 1; j > 0; j >>= 1) {
          for (int i = tid; i < P; i += SORT_NT) {
            const int ixj = i ^ j;
            if (ixj > i) {
              const T ka = s_key[i], kb = s_key[ixj];
              const int ia = s_id[i], ib = s_id[ixj];
              const bool up = (i & kk) == 0;
              const bool a_gt_b = key_less<T>(kb, ib, ka, ia);
              if (a_gt_b == up) { s_key[i] = kb; s_key[ixj] = ka; s_id[i] = ib; s_id[ixj] = ia; }
            }
          }
          __syncthreads();
        }
      }
      for (int i = tid; i < n; i += SORT_NT) {
        const int id = s_id[i];
        p.s_loc[beg + i] = p.loc[id];
        p.s_var[beg + i] = p.var[id];
        p.s_idx[beg + i] = id;
      }
      if (tid == 0) {
        T v = s_red[0];
#pragma unroll
        for (int w = 1; w < SORT_NT / 32; ++w) v = s_red[w] > v ? s_red[w] : v;
        p.s_v0max[m] = v;
      }
    }
    __syncthreads();  // s_long is rewritten by the next round
  }
}

}  // namespace ckf
