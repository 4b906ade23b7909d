// ckf_kernels.cuh — shared declarations of the CKF kernels (a3-a11).
//
// Design: the level loop is LEVEL-SYNCHRONOUS over the whole event and PHASE-SEPARATED into
// small kernels, four per level:
//   ckf_step    persistent lanes pull tips of the level from a global cursor and run the navigation +
//               adaptive RKN4 state machine (ckf_nav.cuh) until the tip stands on its next module
//   ckf_visit   arrival Jacobian + covariance transport (lane per tip), then the chi2 gate over the loc0
//               windows of the sorted slices (flattened (tip, measurement) pairs) and the k best
//   ckf_scan    per-seed cap R10 + emission records (every tip looks back over its seed's earlier tips), then
//               the exclusive scan of the kept children -> child offsets, link allocation, next level's size
//   ckf_update  thread per child: Kalman update or hole, link append, departure state of the next level
// Why not one persistent kernel: measured on B200 (profiles/r01b), the monolithic level loop is ~100 KB of
// SASS; with the warps of an SM in different phases the SM instruction cache misses 31 % of its requests and
// the GPC-level instruction cache saturates (77 % of peak), which bounds the kernel regardless of occupancy.
// Each kernel here keeps its hot loop within the SM's instruction cache and gets its own register budget.
// Everything is placed by prefix sums in tip order (seed, then lineage), so the output is deterministic.
#pragma once
#include <cuda_runtime.h>
#include "ckf_nav.cuh"

namespace ckf {

constexpr int CAND = 16;          // per-tip passer buffer of the gate fast path
constexpr int STEP_NT = 128;      // threads per block of ckf_step
constexpr int VISIT_NT = 128;     // threads per block of ckf_visit (4 warps, 32 tips each)
constexpr int SCAN_NT = 256;      // threads per block of ckf_scan / ckf_update; tile of the scan
constexpr int SORT_NT = 512;      // threads per block of the slice sort
constexpr int SORT_CAP = 2048;    // largest module slice sorted in shared memory; larger ones stay unsorted
#ifndef CKF_FETCH_MIN
#define CKF_FETCH_MIN 32
#endif
#ifndef CKF_PICK_MIN
#define CKF_PICK_MIN 32
#endif
constexpr int FETCH_MIN = CKF_FETCH_MIN;  // finished / tip-less lanes that must wait before write-back + fetch run early
constexpr int PICK_MIN = CKF_PICK_MIN;    // lanes on a portal that must wait before the module choice runs early

template <typename T> struct Vec2;
template <> struct Vec2<float> { using type = float2; };
template <> struct Vec2<double> { using type = double2; };

enum CounterId { CNT_TIPS = 0, CNT_VISITS, CNT_TRIALS, CNT_ACCEPTED, CNT_GATE, CNT_UPDATES, CNT_LINKS, CNT_ITER,
                 CNT_GATE_EXEC, CNT_N };

// per-event device globals (int32 each)
#ifndef CKF_NBIN
#define CKF_NBIN 8
#endif
enum GlobalId { G_LINK_COUNT = 0, G_FIRST_BAD, G_TOTAL_TRACKS, G_TOTAL_ENTRIES, G_NTIPS0, G_NTIPS1, G_STEP_CURSOR,
                G_SCAN_TICKET, G_LBASE, G_SEED_TICKET, G_BAD_INPUT, G_BIN0, G_N = G_BIN0 + CKF_NBIN };
constexpr int NBIN = CKF_NBIN;    // cost classes of the step schedule (G_BIN0 .. G_BIN0 + NBIN - 1 hold their sizes)
constexpr int GBLK = 64;          // ints reserved for one block of globals

template <typename T>
struct KParams {
  GeoDev geo;
  FieldDev fld;
  CfgDev cfg;
  // event (caller's device buffers)
  int32_t n_meas, n_seeds;
  const int32_t* moff;             // [n_vmod + 1]
  int32_t n_vmod;                  // n_events * n_modules: a batch of events is ONE find over replicas of the detector
                                   // (virtual module id = event * n_modules + module; only the CSR of measurements and
                                   // the seeds' module ids use virtual ids, geometry and navigation use real ones)
  const typename Vec2<T>::type* loc;
  const typename Vec2<T>::type* var;
  const int32_t* seed_module;
  const T* seed_x;   // [n][6]
  const T* seed_C;   // [n][36]
  // a7 gate index, rebuilt per event by ckf_sort_slices: every module slice re-ordered by loc0
  typename Vec2<T>::type* s_loc;   // [n_meas]
  typename Vec2<T>::type* s_var;   // [n_meas]
  int32_t* s_idx;                  // [n_meas] position in the caller's arrays (what meas_idx reports)
  T* s_v0max;                      // [n_vmod] largest var0 of the slice; < 0 = slice left unsorted
  // candidate-link buffer (a10): SoA, one entry per child ever made; a level's links are contiguous
  int32_t max_links;
  double* lk_x;        // [6][max_links]   bound parameters after the visit
  double* lk_C;        // [21][max_links]  packed covariance after the visit (float64 in both modes)
  int32_t* lk_module;  // module visited
  int32_t* lk_parent;  // previous link of the branch, -1 = seed
  int32_t* lk_meas;    // measurement index, -1 = hole
  T* lk_chi2;          // predicted chi2 of that measurement
  double* lk_chi2sum;
  int32_t* lk_counts;  // n_meas | n_holes << 16
  int32_t* lk_lastmeas;  // link of the branch's last measurement (state reported on emission)
  // per seed
  int32_t* sd_eoff;      // event * n_modules of the seed's event: real module id + sd_eoff = virtual module id
  int32_t* sd_extra;     // leaves - 1 (R10)
  int32_t* sd_nemit;     // emitted candidates so far
  int32_t* sd_nentries;  // their measurement entries so far
  int32_t* leaf_link;    // [n_seeds * cap]
  int32_t* leaf_meta;    // stop reason | n_holes << 8
  int32_t* leaf_entry;   // entry offset inside the seed
  int32_t* sd_track_base;  // [n_seeds + 1] (emission scan) prefix inside the seed's tile of 1024
  int32_t* sd_entry_base;  // [n_seeds + 1]
  int32_t* seed_tile;      // [2][seed_tiles_cap + 1] tile offsets (tracks, entries)
  int32_t seed_tiles_cap;
  // ---- tips of a level, ordered by seed then lineage; arrays [..][tcap], tip index fastest
  int32_t tcap;
  int32_t* tip_link;   // [2][tcap] (ping-pong by level parity) link the tip stands on, -1 = fresh seed
  int32_t* tip_seed;   // [2][tcap]
  // departure / arrival state of the move (ckf_update -> ckf_step -> ckf_visit)
  double* mv_y;        // [tcap][8] r, d, t, q/p (move records, see below)
  T* mv_D;             // [tcap][MVD] transport Jacobian (ckf_step -> ckf_visit)
  T* mv_Dr;            // [tcap][12] position columns of D (J2', config.field_gradient; null otherwise)
  double* mv_dep;      // [NDEP][tcap] direction on departure, Highland q_phi, q_theta, energy-loss factor g
  int32_t* mv_from;    // [tcap] module the tip stands on
  int32_t* mv_tgt;     // [2][tcap] module reached; overlap neighbour at departure (N2, by ckf_update), -1 none
  int32_t* mv_stop;    // [tcap] stop reason so far
  int32_t* mv_order;   // [NBIN][tcap] live tips of the level grouped by predicted RKN4 trial count (step schedule)
  // prediction + selection (ckf_visit -> ckf_cap, ckf_update)
  double* pd_x;        // [6][tcap]
  double* pd_C;        // [21][tcap]
  T* sel_chi2;         // [K][tcap]
  int32_t* sel_idx;    // [K][tcap]
  int32_t* t_nsel;     // [tcap]
  int32_t* t_want;     // [tcap]
  int32_t* t_counts;   // [tcap] n_meas | n_holes << 16 of the tip (fatal hole included)
  int32_t* t_keep;     // [tcap] children kept after R10
  int32_t* t_kex;      // [tcap] exclusive prefix of t_keep inside the tip's scan tile
  int32_t* blk_sum;    // [tcap / SCAN_NT + 2] kept children per scan tile, then exclusive offsets
  int32_t* t_fin;      // [4][tcap] per-seed totals parked by the seed's last tip: seed (-1 none), extra, nemit, nentries
  // globals
  int32_t* g;          // [G_N]
  unsigned long long* counters;
  // output
  int32_t max_tracks, max_entries;
  int32_t* o_ntracks; int32_t* o_status; int32_t* o_offsets; int32_t* o_meas; int32_t* o_seed; int32_t* o_nholes;
  int32_t* o_lastmod; int32_t* o_stop;
  T* o_params; T* o_cov; T* o_chi2sum; T* o_entrychi2;
  int32_t* o_summary;  // [3] or null (ckf_find_host): n_tracks, status, entries, written last by ckf_finalize
};

// CSR slice of (virtual) module m, clamped into [0, n_meas]: a malformed module_offsets array (not monotonic, or an
// offset beyond n) shortens slices, it never reads outside loc / var (ckf_sort_slices flags it CKF_STATUS_BAD_INPUT).
template <typename T>
__device__ __forceinline__ void slice_of(const KParams<T>& p, int m, int& beg, int& end) {
  int b = __ldg(p.moff + m), e = __ldg(p.moff + m + 1);
  b = b < 0 ? 0 : (b > p.n_meas ? p.n_meas : b);
  e = e < b ? b : (e > p.n_meas ? p.n_meas : e);
  beg = b; end = e;
}

// ------------------------------------------------------------------------------------------ move records
// The state of a move is kept per tip as two contiguous records (AoS), not [component][tip]: ckf_step reaches its tips
// through the step schedule, i.e. in scattered order, and a contiguous record costs whole sectors whatever the order
// (the [component][tip] form cost 33 partial-sector accesses per tip there); the lane-per-tip readers (ckf_visit,
// ckf_update, ckf_fit_level) read the same bytes either way.
//   mv_y[t * 8 ..)    r[3], d[3], t, q/p   float64 (one 64-byte record)
//   mv_D[t * MVD ..)  Rd[9], Dd[9], rq[3], dq[3], tq, padding   T (one 128- / 256-byte record)
constexpr int MVD = 32;
// 256-bit accesses (sm_100a: LDG.E.256 / STG.E.256): a record is read or written by ONE lane, the lanes of a warp touch
// unrelated records, and what the L1 data pipe then counts is instructions x lanes -- half as many with 32-byte pieces.
__device__ __forceinline__ void ld256(const void* p, double& a, double& b, double& c, double& d) {
  asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p) : "memory");
}
__device__ __forceinline__ void st256(void* p, double a, double b, double c, double d) {
  asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}
__device__ __forceinline__ double pack2(float lo, float hi) {
  return __longlong_as_double(((long long)__float_as_uint(hi) << 32) | (long long)__float_as_uint(lo));
}
__device__ __forceinline__ void unpack2(double v, float& lo, float& hi) {
  const long long b = __double_as_longlong(v);
  lo = __uint_as_float((unsigned)b);
  hi = __uint_as_float((unsigned)(b >> 32));
}
__device__ __forceinline__ void store_traj(double* mv_y, size_t t, const Traj& y) {
  double* q = mv_y + t * 8;
  st256(q, y.r[0], y.r[1], y.r[2], y.d[0]);
  st256(q + 4, y.d[1], y.d[2], y.t, y.qop);
}
__device__ __forceinline__ void load_traj(const double* mv_y, size_t t, Traj& y) {
  const double* q = mv_y + t * 8;
  ld256(q, y.r[0], y.r[1], y.r[2], y.d[0]);
  ld256(q + 4, y.d[1], y.d[2], y.t, y.qop);
}
__device__ __forceinline__ void store_jac(float* mv_D, size_t t, const Jac<float>& D) {
  float* q = mv_D + t * MVD;
  const float v[32] = {D.Rd[0][0], D.Rd[0][1], D.Rd[0][2], D.Rd[1][0], D.Rd[1][1], D.Rd[1][2], D.Rd[2][0], D.Rd[2][1],
                       D.Rd[2][2], D.Dd[0][0], D.Dd[0][1], D.Dd[0][2], D.Dd[1][0], D.Dd[1][1], D.Dd[1][2], D.Dd[2][0],
                       D.Dd[2][1], D.Dd[2][2], D.rq[0], D.rq[1], D.rq[2], D.dq[0], D.dq[1], D.dq[2], D.tq, 0.f, 0.f, 0.f,
                       0.f, 0.f, 0.f, 0.f};
#pragma unroll
  for (int i = 0; i < 4; ++i)
    st256(q + 8 * i, pack2(v[8 * i], v[8 * i + 1]), pack2(v[8 * i + 2], v[8 * i + 3]), pack2(v[8 * i + 4], v[8 * i + 5]),
          pack2(v[8 * i + 6], v[8 * i + 7]));
}
__device__ __forceinline__ void load_jac(const float* mv_D, size_t t, Jac<float>& D) {
  const float* q = mv_D + t * MVD;
  float v[32];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    double a, b, c, d;
    ld256(q + 8 * i, a, b, c, d);
    unpack2(a, v[8 * i], v[8 * i + 1]); unpack2(b, v[8 * i + 2], v[8 * i + 3]);
    unpack2(c, v[8 * i + 4], v[8 * i + 5]); unpack2(d, v[8 * i + 6], v[8 * i + 7]);
  }
#pragma unroll
  for (int i = 0; i < 3; ++i) {
#pragma unroll
    for (int j = 0; j < 3; ++j) { D.Rd[i][j] = v[i * 3 + j]; D.Dd[i][j] = v[9 + i * 3 + j]; }
    D.rq[i] = v[18 + i];
    D.dq[i] = v[21 + i];
  }
  D.tq = v[24];
}
__device__ __forceinline__ void store_jac(double* mv_D, size_t t, const Jac<double>& D) {
  double* q = mv_D + t * MVD;
  const double v[28] = {D.Rd[0][0], D.Rd[0][1], D.Rd[0][2], D.Rd[1][0], D.Rd[1][1], D.Rd[1][2], D.Rd[2][0], D.Rd[2][1],
                        D.Rd[2][2], D.Dd[0][0], D.Dd[0][1], D.Dd[0][2], D.Dd[1][0], D.Dd[1][1], D.Dd[1][2], D.Dd[2][0],
                        D.Dd[2][1], D.Dd[2][2], D.rq[0], D.rq[1], D.rq[2], D.dq[0], D.dq[1], D.dq[2], D.tq, 0.0, 0.0, 0.0};
#pragma unroll
  for (int i = 0; i < 7; ++i) st256(q + 4 * i, v[4 * i], v[4 * i + 1], v[4 * i + 2], v[4 * i + 3]);
}
__device__ __forceinline__ void load_jac(const double* mv_D, size_t t, Jac<double>& D) {
  const double* q = mv_D + t * MVD;
  double v[28];
#pragma unroll
  for (int i = 0; i < 7; ++i) ld256(q + 4 * i, v[4 * i], v[4 * i + 1], v[4 * i + 2], v[4 * i + 3]);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
#pragma unroll
    for (int j = 0; j < 3; ++j) { D.Rd[i][j] = v[i * 3 + j]; D.Dd[i][j] = v[9 + i * 3 + j]; }
    D.rq[i] = v[18 + i];
    D.dq[i] = v[21 + i];
  }
  D.tq = v[24];
}

// position columns (J2'): Ru, Du, Rv, Dv, 12 T per tip
template <typename T>
__device__ __forceinline__ void store_jacr(T* mv_Dr, size_t t, const JacR<T>& R) {
  T* q = mv_Dr + t * 12;
#pragma unroll
  for (int i = 0; i < 3; ++i) { q[i] = R.Ru[i]; q[3 + i] = R.Du[i]; q[6 + i] = R.Rv[i]; q[9 + i] = R.Dv[i]; }
}
template <typename T>
__device__ __forceinline__ void load_jacr(const T* mv_Dr, size_t t, JacR<T>& R) {
  const T* q = mv_Dr + t * 12;
#pragma unroll
  for (int i = 0; i < 3; ++i) { R.Ru[i] = q[i]; R.Du[i] = q[3 + i]; R.Rv[i] = q[6 + i]; R.Dv[i] = q[9 + i]; }
}

// ------------------------------------------------------------------------------------------ launch chain
// Every kernel of a find is launched with programmatic stream serialisation (ckf.cu, launch_chain): its blocks may become
// resident while the previous kernel of the stream drains, and they wait HERE until that kernel has completed and its
// writes are visible.  Nothing is read or written before this call.  Under a plain launch both instructions are no-ops.
__device__ __forceinline__ void chain_enter() {
  asm volatile("griddepcontrol.launch_dependents;");
  asm volatile("griddepcontrol.wait;" ::: "memory");
}

// ------------------------------------------------------------------------------------------ warp primitives
__device__ __forceinline__ int warp_incl_scan(int v, int lane) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int n = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v += n;
  }
  return v;
}

template <typename T>
__device__ __forceinline__ bool key_less(T c1, int i1, T c2, int i2) {
  return c1 < c2 || (c1 == c2 && i1 < i2);
}

__device__ __forceinline__ void flush_counter(unsigned long long* dst, unsigned long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0 && v) atomicAdd(dst, v);
}

}  // namespace ckf
