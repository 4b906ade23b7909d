// ckf_step.cuh — navigation + adaptive RKN4 of every tip of a level (a4, a5): the hot kernel.
//
// Persistent lanes: every lane owns one Move (ckf_nav.cuh) at a time and pulls the next tip of the level
// from a global cursor when its move is done, so lanes do not idle while a neighbour needs more RKN4 trials
// (the imbalance the paper names).  The code that is not the trial — write-back + fetch,
// module choice — runs at SERVICE points: lanes that finished, lanes without a tip and lanes that need a
// module choice wait until FETCH_MIN / PICK_MIN of them have gathered (or no lane can step), then are served together.
// The module choice spreads its nine straight-line tests per tip over all 32 lanes.
#pragma once
#include <type_traits>
#include "ckf_kernels.cuh"

namespace ckf {

// scratch of one warp for the module choice
struct PickSmem {
  double* hit;     // [32][9] path length of each (requester rank, neighbour) test; NaN = no hit
  double* rd;      // [6][32] position and direction of the requesting tips
  int32_t* hid;    // [32][9] module id of each test
  int32_t *rl, *ri, *rj, *rx, *list;  // [32] request: layer, iphi, iz, exclude | s_min sign; compacted lanes
  int32_t *rnp, *rnz, *rof;           // [32] the layer's n_phi, n_z, module offset (read once by the requesting lane)
  static constexpr size_t BYTES = 8 * 9 * 32 + 8 * 6 * 32 + 4 * 9 * 32 + 4 * 8 * 32;
  __host__ __device__ static constexpr size_t bytes() { return BYTES; }
  __device__ void carve(unsigned char* raw) {
    unsigned char* p = raw;
    hit = (double*)p; p += 8 * 9 * 32;
    rd = (double*)p; p += 8 * 6 * 32;
    hid = (int32_t*)p; p += 4 * 9 * 32;
    rl = (int32_t*)p; p += 4 * 32;
    ri = (int32_t*)p; p += 4 * 32;
    rj = (int32_t*)p; p += 4 * 32;
    rx = (int32_t*)p; p += 4 * 32;
    list = (int32_t*)p; p += 4 * 32;
    rnp = (int32_t*)p; p += 4 * 32;
    rnz = (int32_t*)p; p += 4 * 32;
    rof = (int32_t*)p; p += 4 * 32;
  }
};

// a4: module choice for all lanes in PH_START / PH_LANDED at once (N2, N4).  The nine tests of each requesting
// tip are flattened into (tip, neighbour) pairs over the 32 lanes; the owning lane then scans its nine
// results in the order of the sequential rule (nearest first, tie -> lower id).
template <typename T>
__device__ __forceinline__ void pick_warp(const GeoDev& geo, const PickSmem& ps, Move<T>& m, int lane) {
  const bool need = m.phase == PH_START || m.phase == PH_LANDED;
  PickRequest q;
  int what = PICK_SKIP;
  if (need) what = move_pick_request(m, geo, q);
  const bool ok = what == PICK_TEST;
  const unsigned breq = __ballot_sync(0xffffffffu, ok);
  if (ok) {
    ps.rl[lane] = q.layer; ps.ri[lane] = q.iphi; ps.rj[lane] = q.iz;
    { const LayerRec* LR = geo.layer + q.layer; ps.rnp[lane] = LR->n_phi; ps.rnz[lane] = LR->n_z; ps.rof[lane] = LR->offset; }
    ps.rx[lane] = (q.exclude < 0 ? 0 : q.exclude + 1) * 2 + (q.s_min > 0.0 ? 1 : 0);
#pragma unroll
    for (int i = 0; i < 3; ++i) { ps.rd[i * 32 + lane] = m.y.r[i]; ps.rd[(3 + i) * 32 + lane] = m.y.d[i]; }
    ps.list[__popc(breq & ((1u << lane) - 1u))] = lane;
  }
  __syncwarp();
  const int total = 9 * __popc(breq);
  for (int q0 = 0; q0 < total; q0 += 32) {
    const int pr = q0 + lane;
    if (pr < total) {
      const int t = ps.list[pr / 9], nb = pr % 9;
      const int Ln_phi = ps.rnp[t], Ln_z = ps.rnz[t], Loffset = ps.rof[t];
      int ii = ps.ri[t] + (nb / 3 - 1);
      ii = ii < 0 ? ii + Ln_phi : (ii >= Ln_phi ? ii - Ln_phi : ii);
      const int jj = ps.rj[t] + (nb % 3 - 1);
      const int rx = ps.rx[t];
      double sres = __longlong_as_double(0x7ff8000000000000LL);
      int id = -1;
      if (jj >= 0 && jj < Ln_z) {
        id = Loffset + ii * Ln_z + jj;
        if (id != (rx >> 1) - 1) {
          const double r[3] = {ps.rd[0 * 32 + t], ps.rd[1 * 32 + t], ps.rd[2 * 32 + t]};
          const double d[3] = {ps.rd[3 * 32 + t], ps.rd[4 * 32 + t], ps.rd[5 * 32 + t]};
          // no early exits: the four groups of fields of the module record are loaded at once instead of one L2 round
          // trip per passed test (that chain was a quarter of this kernel's stall samples)
          // the record as four 256-bit loads (c, u, v, n, half_u, half_v = its first 112 bytes): what the L1 data pipe of
          // this kernel counts is load instructions x scattered lanes, and the module tests were half of them
          double rec[16];
          ld_module_rec(geo.mod + id, rec);
          sres = line_test_rec(rec, r, d, (rx & 1) ? 1e-3 : -1e-3, geo.bidir);
        }
      }
      ps.hit[pr] = sres;   // [requester rank][neighbour]: consecutive lanes, consecutive words (no bank conflicts)
      ps.hid[pr] = id;
    }
  }
  __syncwarp();
  if (need) {
    int best = -1;
    double best_s = 0.0;
    if (ok) {
      const int rank9 = 9 * __popc(breq & ((1u << lane) - 1u));
#pragma unroll 1
      for (int nb = 0; nb < 9; ++nb) {
        const double sv = ps.hit[rank9 + nb];
        const int id = ps.hid[rank9 + nb];
        if (sv == sv && (best < 0 || sv < best_s || (sv == best_s && id < best))) { best = id; best_s = sv; }
      }
    }
    move_pick_apply(m, geo, best);
  }
  __syncwarp();
}

template <typename T, int MINB, bool GRAD = false>
__global__ void __launch_bounds__(STEP_NT, MINB) ckf_step(const KParams<T> p, int level) {
  chain_enter();
  if (p.g[G_NTIPS0 + (level & 1)] == 0 || level == 0) return;  // level 0: the seed's own module, identity transport (N6)
  __shared__ __align__(16) unsigned char smem_raw[(STEP_NT / 32) * PickSmem::bytes()];
  // step schedule: the live tips of the level, grouped by predicted trial count (ckf_update), longest first
  __shared__ int s_binend[NBIN];
  if (threadIdx.x == 0) {
    int acc = 0;
    for (int k = 0; k < NBIN; ++k) { acc += p.g[G_BIN0 + NBIN - 1 - k]; s_binend[k] = acc; }
  }
  __syncthreads();
  const int n = s_binend[NBIN - 1];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  PickSmem ps;
  ps.carve(smem_raw + (size_t)wib * PickSmem::bytes());
  const size_t TC = (size_t)p.tcap;

  typename std::conditional<GRAD, MoveG<T>, Move<T>>::type m;
  if constexpr (GRAD) jacr_begin(m.Dr, p.geo.mod[0].u, p.geo.mod[0].v);
  m.phase = PH_IDLE; m.stop = STOP_NONE; m.from = 0; m.tgt = -1; m.lp = 0; m.lb = -1; m.ld = -1; m.n_steps = 0; m.targeted = false; m.inward = false;
  m.B1[0] = m.B1[1] = m.B1[2] = 0.0;
  m.h = 0.0; m.h_ctrl = 0.0; m.R = 0.0; m.y.qop = 0.0; m.ib = 0.0; m.dib = 0.0;
  int tip = -1, nt = 0, na = 0;
  bool more = true;  // the level's cursor is not exhausted (warp-uniform)
  for (;;) {
    const unsigned bI = __ballot_sync(0xffffffffu, m.phase == PH_IDLE);
    const unsigned bP = __ballot_sync(0xffffffffu, m.phase == PH_START || m.phase == PH_LANDED);
    const unsigned bS = __ballot_sync(0xffffffffu, is_stepping(m.phase));
    const unsigned bF = __ballot_sync(0xffffffffu, m.phase == PH_FIN);
    if (!bP && !bS && !bF && !more) break;
    const int waiting = __popc(bF) + (more ? __popc(bI) : 0);
    if (bS == 0u || waiting >= FETCH_MIN || __popc(bP) >= PICK_MIN) {
      // ---- write-back of finished moves
      if (m.phase == PH_FIN) {
        if (m.stop == STOP_NONE) {
          store_traj(p.mv_y, (size_t)tip, m.y);
          store_jac(p.mv_D, (size_t)tip, m.D);
          if constexpr (GRAD) store_jacr(p.mv_Dr, (size_t)tip, m.Dr);
          p.mv_tgt[tip] = m.tgt;
        }
        p.mv_stop[tip] = m.stop;
        m.phase = PH_IDLE;
      }
      // ---- fetch: idle lanes take the next tips of the level, in order
      const unsigned idle = __ballot_sync(0xffffffffu, m.phase == PH_IDLE);
      if (idle && more) {
        int base = 0;
        if (lane == 0) base = atomicAdd(p.g + G_STEP_CURSOR, __popc(idle));
        base = __shfl_sync(0xffffffffu, base, 0);
        if (base + __popc(idle) >= n) more = false;
        const int q = base + __popc(idle & ((1u << lane) - 1u));
        int t = -1;
        if (m.phase == PH_IDLE && q < n) {
          int k = 0;
          while (q >= s_binend[k]) ++k;
          t = p.mv_order[(size_t)(NBIN - 1 - k) * TC + (q - (k ? s_binend[k - 1] : 0))];
        }
        if (t >= 0) {  // every tip of the schedule is live (ckf_update / ckf_fit_level only append live ones)
          tip = t;
          load_traj(p.mv_y, (size_t)t, m.y);
          if constexpr (GRAD) move_begin(m, p.geo, p.cfg, p.mv_from[t]);
          else move_begin<T>(m, p.cfg, p.mv_from[t]);
          move_pick_apply<T>(m, p.geo, p.mv_tgt[TC + t]);  // N2 was decided by ckf_update
        }
      }
      // ---- module choice at the portal (N3, N4) once enough lanes need one
      {
        const unsigned need = __ballot_sync(0xffffffffu, m.phase == PH_START || m.phase == PH_LANDED);
        const unsigned step = __ballot_sync(0xffffffffu, is_stepping(m.phase));
        if (need && (step == 0u || __popc(need) >= PICK_MIN)) pick_warp<T>(p.geo, ps, m, lane);
      }
    }
    // ---- one step: targeting + landing, else one RKN4 trial
    if (is_stepping(m.phase)) move_step<T>(m, p.fld, p.cfg, nt, na);
    __syncwarp();
  }
  flush_counter(p.counters + CNT_TRIALS, (unsigned long long)nt);
  flush_counter(p.counters + CNT_ACCEPTED, (unsigned long long)na);
}

}  // namespace ckf
