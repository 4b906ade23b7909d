// ckf_emit.cuh — per-event init and the emission kernels (a11): leaves -> CSR track list.
#pragma once
#include <climits>
#include "ckf_kernels.cuh"

namespace ckf {

// Resets every per-event device counter and lays down level 0: one tip per seed, standing on no link.
// (No allocation, no memset calls in ckf_find.)
template <typename T>
__global__ void ckf_init_event(const KParams<T> p) {
  chain_enter();
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < p.n_seeds) {
    p.sd_extra[i] = 0; p.sd_nemit[i] = 0; p.sd_nentries[i] = 0;
    // a seed whose (virtual) module id is out of range is malformed input: it is flagged (sd_eoff < 0), stops NUMERIC
    // at level 0 and sets CKF_STATUS_BAD_INPUT; nothing is ever indexed with its module id
    const int sm = p.seed_module[i];
    const bool bad = sm < 0 || sm >= p.n_vmod;
    p.sd_eoff[i] = bad ? -1 : (sm / p.geo.n_modules) * p.geo.n_modules;
    if (bad) atomicOr(p.g + G_BAD_INPUT, 1);
    if (i < p.tcap) { p.tip_link[i] = -1; p.tip_seed[i] = i; p.mv_stop[i] = STOP_NONE; }
  }
  if (i == 0) {
    for (int k = 0; k < G_N; ++k)
      if (k != G_BAD_INPUT) p.g[k] = 0;   // G_BAD_INPUT is cleared by ckf_finalize (other threads of this launch set it)
    p.g[G_FIRST_BAD] = INT_MAX;
    p.g[G_NTIPS0] = p.n_seeds < p.tcap ? p.n_seeds : p.tcap;
    *p.o_status = p.n_seeds > p.tcap ? 4 : 0;
    *p.o_ntracks = 0;
  }
  if (i < CNT_N) p.counters[i] = 0ull;
}

// Exclusive scan over seeds of (emitted candidates, their entries) -> per-seed bases.  Order by seed id is what
// makes the output deterministic.  One block per tile of 1024 seeds writes the in-tile prefixes; the last block
// to finish scans the tile totals (seed_tile[2][tiles + 1]).  Global base of seed s = tile offset + prefix.
constexpr int SEED_TILE = 1024;
template <typename T>
__global__ void __launch_bounds__(SEED_TILE) ckf_scan_seeds(const KParams<T> p) {
  chain_enter();
  __shared__ unsigned long long s_w[32];
  __shared__ int s_last;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5, S = p.n_seeds;
  const int ntiles = S > 0 ? (S + SEED_TILE - 1) / SEED_TILE : 1;
  if ((int)blockIdx.x >= ntiles) return;
  int32_t* tile_trk = p.seed_tile;
  int32_t* tile_ent = p.seed_tile + (p.seed_tiles_cap + 1);
  {
    const int i = blockIdx.x * SEED_TILE + tid;
    unsigned long long v = 0ull;  // (tracks << 32) | entries: both stay below 2^31
    if (i < S) v = ((unsigned long long)(unsigned)p.sd_nemit[i] << 32) | (unsigned long long)(unsigned)p.sd_nentries[i];
    unsigned long long inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned long long n = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += n;
    }
    if (lane == 31) s_w[w] = inc;
    __syncthreads();
    unsigned long long base = 0ull, tot = 0ull;
#pragma unroll
    for (int k = 0; k < 32; ++k) {
      const unsigned long long x = s_w[k];
      if (k < w) base += x;
      tot += x;
    }
    const unsigned long long ex = base + inc - v;
    if (i < S) { p.sd_track_base[i] = (int)(ex >> 32); p.sd_entry_base[i] = (int)(ex & 0xffffffffull); }
    if (tid == 0) { tile_trk[blockIdx.x] = (int)(tot >> 32); tile_ent[blockIdx.x] = (int)(tot & 0xffffffffull); }
  }
  __threadfence();
  __syncthreads();
  if (tid == 0) s_last = (atomicAdd(p.g + G_SEED_TICKET, 1) == ntiles - 1) ? 1 : 0;
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  if (tid == 0) {
    int a = 0, b = 0;
    for (int k = 0; k < ntiles; ++k) {
      const int ta = ((volatile int32_t*)tile_trk)[k], tb = ((volatile int32_t*)tile_ent)[k];
      tile_trk[k] = a; tile_ent[k] = b;
      a += ta; b += tb;
    }
    tile_trk[ntiles] = a; tile_ent[ntiles] = b;
    p.g[G_TOTAL_TRACKS] = a; p.g[G_TOTAL_ENTRIES] = b;
    p.g[G_SEED_TICKET] = 0;
  }
}

// Thread per candidate: backtrace the links into the index list, copy the state at the last measurement.  The 6 + 36
// numbers per candidate are transposed through a shared-memory tile of the warp, so that the 32 candidates of a warp
// (consecutive in the output) are written as contiguous runs instead of 42 stores of stride 24 / 144 bytes per lane.
constexpr int EMIT_NT = 128;
template <typename T>
__global__ void __launch_bounds__(EMIT_NT) ckf_emit_tracks(const KParams<T> p) {
  chain_enter();
  __shared__ T s_tile[EMIT_NT / 32][32 * 37];
  const int lane = threadIdx.x & 31;
  T* tile = s_tile[threadIdx.x >> 5];
  const int total = p.g[G_TOTAL_TRACKS];
  const int cap = p.cfg.max_cands;
  const int ntiles = p.n_seeds > 0 ? (p.n_seeds + SEED_TILE - 1) / SEED_TILE : 1;
  const int32_t* tile_trk = p.seed_tile;
  const int32_t* tile_ent = p.seed_tile + (p.seed_tiles_cap + 1);
  const int stride = gridDim.x * blockDim.x;
  for (int t0 = (blockIdx.x * blockDim.x + threadIdx.x) - lane; t0 < total; t0 += stride) {   // warp-uniform
    const int t = t0 + lane;
    bool ok = t < total;
    int ls = 0;
    if (ok) {
      // seed = last s with (tile offset + in-tile prefix) <= t: tile first, then inside the tile
      int lo = 0, hi = ntiles;
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (tile_trk[mid] <= t) lo = mid; else hi = mid;
      }
      const int toff = tile_trk[lo], eoff = tile_ent[lo];
      int a = lo * SEED_TILE, b = min(p.n_seeds, a + SEED_TILE);
      while (b - a > 1) {
        const int mid = (a + b) >> 1;
        if (toff + p.sd_track_base[mid] <= t) a = mid; else b = mid;
      }
      const int seed = a, j = t - (toff + p.sd_track_base[seed]);
      const size_t li = (size_t)seed * cap + j;
      const int leaf = p.leaf_link[li], meta = p.leaf_meta[li];
      const int off = eoff + p.sd_entry_base[seed] + p.leaf_entry[li];
      const int nm = p.lk_counts[leaf] & 0xffff;
      if (t >= p.max_tracks || off + nm > p.max_entries) {
        atomicMin(p.g + G_FIRST_BAD, t);
        atomicOr(p.o_status, t >= p.max_tracks ? 1 : 2);
        ok = false;
      } else {
        p.o_offsets[t] = off;
        p.o_offsets[t + 1] = off + nm;
        int pos = off + nm - 1;
        for (int l = leaf; l >= 0; l = p.lk_parent[l]) {
          const int m = p.lk_meas[l];
          if (m >= 0) { p.o_meas[pos] = m; p.o_entrychi2[pos] = p.lk_chi2[l]; --pos; }
        }
        ls = p.lk_lastmeas[leaf];
        p.o_seed[t] = seed;
        p.o_nholes[t] = meta >> 8;
        p.o_stop[t] = meta & 0xff;
        p.o_lastmod[t] = p.lk_module[ls];
        p.o_chi2sum[t] = (T)p.lk_chi2sum[leaf];
      }
    }
    const unsigned okm = __ballot_sync(0xffffffffu, ok);
    if (okm == 0u) continue;
    // covariance: lane's row of the tile (row stride 37: conflict-free), then the tile row-major to the output
    if (ok) {
#pragma unroll
      for (int i = 0; i < 6; ++i)
#pragma unroll
        for (int k = 0; k < 6; ++k) tile[lane * 37 + i * 6 + k] = (T)p.lk_C[(size_t)tri(i, k) * p.max_links + ls];
    }
    __syncwarp();
    {
      int row = 0, col = lane;   // element lane + 32 * n of the 32 x 36 block
      T* dst = p.o_cov + (size_t)t0 * 36;
      for (int i = lane; i < 32 * 36; i += 32) {
        if ((okm >> row) & 1u) dst[i] = tile[row * 37 + col];
        col += 32;
        if (col >= 36) { col -= 36; ++row; }
      }
    }
    __syncwarp();
    if (ok) {
#pragma unroll
      for (int i = 0; i < 6; ++i) tile[lane * 7 + i] = (T)p.lk_x[(size_t)i * p.max_links + ls];
    }
    __syncwarp();
    {
      T* dst = p.o_params + (size_t)t0 * 6;
#pragma unroll
      for (int n = 0; n < 6; ++n) {
        const int i = lane + 32 * n, row = i / 6, col = i - row * 6;
        if ((okm >> row) & 1u) dst[i] = tile[row * 7 + col];
      }
    }
    __syncwarp();
  }
}

template <typename T>
__global__ void ckf_finalize(const KParams<T> p) {
  chain_enter();
  const int total = p.g[G_TOTAL_TRACKS], bad = p.g[G_FIRST_BAD];
  const int n = total < bad ? total : bad;
  *p.o_ntracks = n;
  if (n == 0) p.o_offsets[0] = 0;
  if (p.g[G_BAD_INPUT]) { atomicOr(p.o_status, 8); p.g[G_BAD_INPUT] = 0; }
  // what ckf_find_host needs to size its copies: candidates, status, entries
  if (p.o_summary) { p.o_summary[0] = n; p.o_summary[1] = *p.o_status; p.o_summary[2] = n > 0 ? p.o_offsets[n] : 0; }
}

}  // namespace ckf
