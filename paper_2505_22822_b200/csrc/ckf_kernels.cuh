// ckf_kernels.cuh — the CKF level loop as ONE persistent kernel per event, plus the emission kernels.
//
// Design: seeds never interact (the only cross-branch rule, the per-seed cap R10, is per
// seed), so a thread block owns whole seeds from pull to emission and the entire level loop
//   propagate (thread per tip) -> gate (warp per tip over the module's CSR slice) -> cap + prefix sums ->
//   update + link append (thread per child) -> emission records
// runs inside the block with __syncthreads only: no host round trip for "n_active == 0", no per-level
// launches, no device-wide scan.  Blocks pull seeds from a global cursor whenever their tip queue has room
// (continuous batching), so lanes stay filled while branches die at different levels.  Results are placed by
// seed id and in-seed order, so the output is deterministic no matter which block took which seed.
#pragma once
#include <cuda_runtime.h>
#include "ckf_nav.cuh"

namespace ckf {

constexpr int NT = 256;       // threads per block of the level loop
constexpr int NW = NT / 32;
constexpr int CAND = 32;      // per-warp passer buffer of the gate fast path

template <typename T> struct Vec2;
template <> struct Vec2<float> { using type = float2; };
template <> struct Vec2<double> { using type = double2; };

enum CounterId { CNT_TIPS = 0, CNT_VISITS, CNT_TRIALS, CNT_ACCEPTED, CNT_GATE, CNT_UPDATES, CNT_LINKS, CNT_ITER, CNT_N };

template <typename T>
struct KParams {
  GeoDev geo;
  FieldDev fld;
  CfgDev cfg;
  // event (caller's device buffers)
  int32_t n_meas, n_seeds;
  const int32_t* moff;
  const typename Vec2<T>::type* loc;
  const typename Vec2<T>::type* var;
  const int32_t* seed_module;
  const T* seed_x;   // [n][6]
  const T* seed_C;   // [n][36]
  // candidate-link buffer (a10): SoA, one entry per child ever made
  int32_t max_links;
  double* lk_x;        // [6][max_links]   bound parameters after the visit
  T* lk_C;             // [21][max_links]  packed covariance after the visit
  int32_t* lk_module;  // module visited
  int32_t* lk_parent;  // previous link of the branch, -1 = seed
  int32_t* lk_meas;    // measurement index, -1 = hole
  T* lk_chi2;          // predicted chi2 of that measurement
  T* lk_chi2sum;
  int32_t* lk_counts;  // n_meas | n_holes << 16
  int32_t* lk_lastmeas;  // link of the branch's last measurement (state reported on emission)
  // per seed
  int32_t* sd_extra;     // leaves - 1 (R10)
  int32_t* sd_nemit;     // emitted candidates so far
  int32_t* sd_nentries;  // their measurement entries so far
  int32_t* leaf_link;    // [n_seeds * cap]
  int32_t* leaf_meta;    // stop reason | n_holes << 8
  int32_t* leaf_entry;   // entry offset inside the seed
  int32_t* sd_track_base;  // [n_seeds + 1] (emission scan)
  int32_t* sd_entry_base;  // [n_seeds + 1]
  // per block tip queues, double buffered: int2 (link or -(seed+1), seed)
  int2* queue;
  int32_t qcap;
  // globals
  int32_t* g_seed_cursor;
  int32_t* g_link_count;
  int32_t* g_first_bad;
  int32_t* g_total;  // [2] total tracks, total entries
  unsigned long long* counters;
  // output
  int32_t max_tracks, max_entries;
  int32_t* o_ntracks; int32_t* o_status; int32_t* o_offsets; int32_t* o_meas; int32_t* o_seed; int32_t* o_nholes;
  int32_t* o_lastmod; int32_t* o_stop;
  T* o_params; T* o_cov; T* o_chi2sum; T* o_entrychi2;
};

// ------------------------------------------------------------------------------------------ block primitives
__device__ __forceinline__ int warp_incl_scan(int v, int lane) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int n = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v += n;
  }
  return v;
}
__device__ __forceinline__ int warp_incl_max(int v, int lane) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int n = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v = max(v, n);
  }
  return v;
}
// Exclusive block scan (sum).  All NT threads call; s_w holds NW ints.  Returns exclusive prefix; total out.
__device__ __forceinline__ int block_excl_scan(int v, int* s_w, int& total) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int inc = warp_incl_scan(v, lane);
  __syncthreads();
  if (lane == 31) s_w[w] = inc;
  __syncthreads();
  int base = 0, tot = 0;
#pragma unroll
  for (int i = 0; i < NW; ++i) {
    const int x = s_w[i];
    if (i < w) base += x;
    tot += x;
  }
  total = tot;
  return base + inc - v;
}
__device__ __forceinline__ int block_incl_max(int v, int* s_w) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int inc = warp_incl_max(v, lane);
  __syncthreads();
  if (lane == 31) s_w[w] = inc;
  __syncthreads();
  int r = inc;
#pragma unroll
  for (int i = 0; i < NW; ++i)
    if (i < w) r = max(r, s_w[i]);
  return r;
}

template <typename T>
__device__ __forceinline__ bool key_less(T c1, int i1, T c2, int i2) {
  return c1 < c2 || (c1 == c2 && i1 < i2);
}

// Shared-memory carve-up of the level loop (sizes depend on max_branches K).
template <typename T>
struct Smem {
  double* px;      // [6][NT] predicted bound parameters
  T* pC;           // [21][NT] predicted packed covariance
  T* selchi2;      // [K][NT]
  int32_t* selidx; // [K][NT]
  T* chi2sum;      // [NT]
  T* candchi2;     // [NW][CAND]
  int32_t* candidx;
  int32_t *link, *seed, *target, *stop, *counts, *lastmeas, *want, *nsel, *head;
  int32_t *Eex, *Kex, *Mex;  // [NT + 1] scans
  int32_t* warp;   // [NW]
  int32_t* misc;   // [16]
  unsigned long long* cnt;  // [CNT_N]
  __host__ __device__ static size_t bytes(int K) {
    size_t b = 0;
    b += sizeof(double) * 6 * NT;
    b += sizeof(T) * 21 * NT;
    b += (sizeof(T) + 4) * (size_t)K * NT;
    b += sizeof(T) * NT;
    b += (sizeof(T) + 4) * NW * CAND;
    b += 4 * 9 * NT;
    b += 4 * 3 * (NT + 1);
    b += 4 * NW + 4 * 16 + 8 * CNT_N;
    return b + 64;
  }
  __device__ void carve(unsigned char* raw, int K) {
    unsigned char* p = raw;
    cnt = (unsigned long long*)p; p += 8 * CNT_N;
    px = (double*)p; p += sizeof(double) * 6 * NT;
    pC = (T*)p; p += sizeof(T) * 21 * NT;
    selchi2 = (T*)p; p += sizeof(T) * (size_t)K * NT;
    chi2sum = (T*)p; p += sizeof(T) * NT;
    candchi2 = (T*)p; p += sizeof(T) * NW * CAND;
    selidx = (int32_t*)p; p += 4 * (size_t)K * NT;
    candidx = (int32_t*)p; p += 4 * NW * CAND;
    link = (int32_t*)p; p += 4 * NT;
    seed = (int32_t*)p; p += 4 * NT;
    target = (int32_t*)p; p += 4 * NT;
    stop = (int32_t*)p; p += 4 * NT;
    counts = (int32_t*)p; p += 4 * NT;
    lastmeas = (int32_t*)p; p += 4 * NT;
    want = (int32_t*)p; p += 4 * NT;
    nsel = (int32_t*)p; p += 4 * NT;
    head = (int32_t*)p; p += 4 * NT;
    Eex = (int32_t*)p; p += 4 * (NT + 1);
    Kex = (int32_t*)p; p += 4 * (NT + 1);
    Mex = (int32_t*)p; p += 4 * (NT + 1);
    warp = (int32_t*)p; p += 4 * NW;
    misc = (int32_t*)p; p += 4 * 16;
  }
};

enum Misc { M_NLIVE = 0, M_NOUT, M_PASS_END, M_PULL_BASE, M_PULL_N, M_LINK_BASE, M_ALLOWED };

}  // namespace ckf
