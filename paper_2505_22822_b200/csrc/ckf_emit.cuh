// ckf_emit.cuh — per-event init and the emission kernels (a11): leaves -> CSR track list.
#pragma once
#include <climits>
#include "ckf_kernels.cuh"

namespace ckf {

// Resets every per-event device counter and lays down level 0: one tip per seed, standing on no link.
// (No allocation, no memset calls in ckf_find.)
template <typename T>
__global__ void ckf_init_event(const KParams<T> p) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < p.n_seeds) {
    p.sd_extra[i] = 0; p.sd_nemit[i] = 0; p.sd_nentries[i] = 0;
    if (i < p.tcap) { p.tip_link[i] = -1; p.tip_seed[i] = i; p.mv_stop[i] = STOP_NONE; }
  }
  if (i == 0) {
    for (int k = 0; k < G_N; ++k) p.g[k] = 0;
    p.g[G_FIRST_BAD] = INT_MAX;
    p.g[G_NTIPS0] = p.n_seeds < p.tcap ? p.n_seeds : p.tcap;
    *p.o_status = p.n_seeds > p.tcap ? 4 : 0;
    *p.o_ntracks = 0;
  }
  if (i < CNT_N) p.counters[i] = 0ull;
}

// Exclusive scan over seeds of (emitted candidates, their entries) -> per-seed bases.  One block: the array is
// tens of thousands of ints, a few microseconds.  Order by seed id is what makes the output deterministic.
template <typename T>
__global__ void __launch_bounds__(1024) ckf_scan_seeds(const KParams<T> p) {
  __shared__ int s_a[1024], s_b[1024];
  const int tid = threadIdx.x, S = p.n_seeds;
  const int per = (S + 1023) / 1024;
  const int lo = min(S, tid * per), hi = min(S, lo + per);
  int a = 0, b = 0;
  for (int i = lo; i < hi; ++i) { a += p.sd_nemit[i]; b += p.sd_nentries[i]; }
  s_a[tid] = a; s_b[tid] = b;
  __syncthreads();
  // Hillis-Steele inclusive scan over the 1024 partials
  for (int o = 1; o < 1024; o <<= 1) {
    int va = 0, vb = 0;
    if (tid >= o) { va = s_a[tid - o]; vb = s_b[tid - o]; }
    __syncthreads();
    s_a[tid] += va; s_b[tid] += vb;
    __syncthreads();
  }
  int ra = s_a[tid] - a, rb = s_b[tid] - b;
  for (int i = lo; i < hi; ++i) {
    p.sd_track_base[i] = ra; p.sd_entry_base[i] = rb;
    ra += p.sd_nemit[i]; rb += p.sd_nentries[i];
  }
  if (tid == 1023) {
    p.sd_track_base[S] = s_a[1023]; p.sd_entry_base[S] = s_b[1023];
    p.g[G_TOTAL_TRACKS] = s_a[1023]; p.g[G_TOTAL_ENTRIES] = s_b[1023];
  }
}

// Thread per candidate: backtrace the links into the index list, copy the state at the last measurement.
template <typename T>
__global__ void __launch_bounds__(256) ckf_emit_tracks(const KParams<T> p) {
  const int total = p.g[G_TOTAL_TRACKS];
  const int cap = p.cfg.max_cands;
  for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < total; t += gridDim.x * blockDim.x) {
    // seed = last s with track_base[s] <= t
    int lo = 0, hi = p.n_seeds;
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (p.sd_track_base[mid] <= t) lo = mid; else hi = mid;
    }
    const int seed = lo, j = t - p.sd_track_base[seed];
    const size_t li = (size_t)seed * cap + j;
    const int leaf = p.leaf_link[li], meta = p.leaf_meta[li];
    const int off = p.sd_entry_base[seed] + p.leaf_entry[li];
    const int nm = p.lk_counts[leaf] & 0xffff;
    if (t >= p.max_tracks || off + nm > p.max_entries) {
      atomicMin(p.g + G_FIRST_BAD, t);
      atomicOr(p.o_status, t >= p.max_tracks ? 1 : 2);
      continue;
    }
    p.o_offsets[t] = off;
    p.o_offsets[t + 1] = off + nm;
    int pos = off + nm - 1;
    for (int l = leaf; l >= 0; l = p.lk_parent[l]) {
      const int m = p.lk_meas[l];
      if (m >= 0) { p.o_meas[pos] = m; p.o_entrychi2[pos] = p.lk_chi2[l]; --pos; }
    }
    const int ls = p.lk_lastmeas[leaf];
    p.o_seed[t] = seed;
    p.o_nholes[t] = meta >> 8;
    p.o_stop[t] = meta & 0xff;
    p.o_lastmod[t] = p.lk_module[ls];
    p.o_chi2sum[t] = p.lk_chi2sum[leaf];
#pragma unroll
    for (int i = 0; i < 6; ++i) p.o_params[(size_t)t * 6 + i] = (T)p.lk_x[(size_t)i * p.max_links + ls];
#pragma unroll
    for (int i = 0; i < 6; ++i)
#pragma unroll
      for (int k = 0; k < 6; ++k) p.o_cov[(size_t)t * 36 + i * 6 + k] = p.lk_C[(size_t)tri(i, k) * p.max_links + ls];
  }
}

template <typename T>
__global__ void ckf_finalize(const KParams<T> p) {
  const int total = p.g[G_TOTAL_TRACKS], bad = p.g[G_FIRST_BAD];
  const int n = total < bad ? total : bad;
  *p.o_ntracks = n;
  if (n == 0) p.o_offsets[0] = 0;
}

}  // namespace ckf
