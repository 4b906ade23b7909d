// ckf_kernels.cuh — the CKF level loop as ONE persistent kernel per event whose worker is the WARP, plus the
// slice-sort and emission kernels.
//
// Design: seeds never interact (the only cross-branch rule, the per-seed cap R10, is per
// seed), so a warp owns whole seeds from pull to emission and runs the entire level loop
//   propagate (lane per tip, lockstep RKN4) -> gate (lanes over the flattened (tip, measurement) pairs of the
//   loc0 windows) -> cap + warp prefix sums -> update + link append (lane per child) -> emission records
// with __syncwarp only: no block barrier (a slow RKN4 loop delays 31 neighbours, not 255), no host round trip
// for "n_active == 0", no per-level launches, no device-wide scan.  Warps pull seeds from a global cursor
// whenever their last chunk of tips has free lanes (continuous batching).  Results are placed by seed id and
// in-seed order, so the output is deterministic no matter which warp took which seed.
#pragma once
#include <cuda_runtime.h>
#include "ckf_nav.cuh"

namespace ckf {

constexpr int WPB = 4;            // warps per block of the level loop (blocks exist only to carve shared memory)
constexpr int NT = 32 * WPB;      // threads per block
constexpr int CAND = 16;          // per-tip passer buffer of the gate fast path
constexpr int MAX_LIVE_SEEDS = 48;  // seeds a warp may hold at once (bounds its tip queue)
constexpr int SUBW = 128;          // tips of a warp's wave propagated together (persistent lanes); multiple of 32
#ifndef CKF_SERVICE_MIN
#define CKF_SERVICE_MIN 12
#endif
constexpr int SERVICE_MIN = CKF_SERVICE_MIN;    // lanes that must be waiting before a P1 service point is run early
constexpr int SORT_NT = 128;      // threads per block of the slice sort
constexpr int SORT_CAP = 2048;    // largest module slice sorted in shared memory; larger ones stay unsorted

template <typename T> struct Vec2;
template <> struct Vec2<float> { using type = float2; };
template <> struct Vec2<double> { using type = double2; };

enum CounterId { CNT_TIPS = 0, CNT_VISITS, CNT_TRIALS, CNT_ACCEPTED, CNT_GATE, CNT_UPDATES, CNT_LINKS, CNT_ITER,
                 CNT_GATE_EXEC, CNT_N };

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
  // a7 gate index, rebuilt per event by ckf_sort_slices: every module slice re-ordered by loc0
  typename Vec2<T>::type* s_loc;   // [n_meas]
  typename Vec2<T>::type* s_var;   // [n_meas]
  int32_t* s_idx;                  // [n_meas] position in the caller's arrays (what meas_idx reports)
  T* s_v0max;                      // [n_modules] largest var0 of the slice; < 0 = slice left unsorted
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
  // per warp tip queues, double buffered: int2 (link or -(seed+1), seed)
  int2* queue;
  int32_t qcap;
  // per warp predictions of one sub-wave (P1 -> P2-P4)
  double* pred_x;    // [n_warps][6][SUBW]
  T* pred_C;         // [n_warps][21][SUBW]
  int32_t* pred_ts;  // [n_warps][2][SUBW] target, stop
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

// ------------------------------------------------------------------------------------------ warp primitives
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

template <typename T>
__device__ __forceinline__ bool key_less(T c1, int i1, T c2, int i2) {
  return c1 < c2 || (c1 == c2 && i1 < i2);
}

// Shared memory of ONE warp of the level loop (sizes depend on max_branches K).  Arrays are [..][32] with the
// tip (lane) index fastest, so lane-per-tip accesses are conflict-free.
template <typename T>
struct WSmem {
  double* px;       // [6][32] predicted bound parameters
  T* pC;            // [21][32] predicted packed covariance
  T* selchi2;       // [K][32]
  int32_t* selidx;  // [K][32]
  T* candchi2;      // [CAND][32]
  int32_t* candidx; // [CAND][32]
  T* chi2sum;       // [32]
  int32_t *link, *seed, *target, *counts, *lastmeas, *nsel, *lo, *cnt;  // [32] each
  int32_t *off, *Kex;  // [33]
  __host__ __device__ static size_t bytes(int K) {
    size_t b = 0;
    b += sizeof(double) * 6 * 32;
    b += sizeof(T) * 21 * 32;
    b += (sizeof(T) + 4) * (size_t)K * 32;
    b += (sizeof(T) + 4) * (size_t)CAND * 32;
    b += sizeof(T) * 32;
    b += 4 * 8 * 32;
    b += 4 * 2 * 33;
    const size_t p1 = 8 * 9 * 32 + 8 * 6 * 32 + 4 * 9 * 32 + 4 * 5 * 32;  // P1Smem::bytes(), aliased
    b = b > p1 ? b : p1;
    return (b + 15) & ~(size_t)15;
  }
  __device__ void carve(unsigned char* raw, int K) {
    unsigned char* p = raw;
    px = (double*)p; p += sizeof(double) * 6 * 32;
    pC = (T*)p; p += sizeof(T) * 21 * 32;
    selchi2 = (T*)p; p += sizeof(T) * (size_t)K * 32;
    candchi2 = (T*)p; p += sizeof(T) * (size_t)CAND * 32;
    chi2sum = (T*)p; p += sizeof(T) * 32;
    selidx = (int32_t*)p; p += 4 * (size_t)K * 32;
    candidx = (int32_t*)p; p += 4 * (size_t)CAND * 32;
    link = (int32_t*)p; p += 4 * 32;
    seed = (int32_t*)p; p += 4 * 32;
    target = (int32_t*)p; p += 4 * 32;
    counts = (int32_t*)p; p += 4 * 32;
    lastmeas = (int32_t*)p; p += 4 * 32;
    nsel = (int32_t*)p; p += 4 * 32;
    lo = (int32_t*)p; p += 4 * 32;
    cnt = (int32_t*)p; p += 4 * 32;
    off = (int32_t*)p; p += 4 * 33;
    Kex = (int32_t*)p; p += 4 * 33;
  }
};

}  // namespace ckf
