// ckf_fit.cuh — Kalman-filter track fit + RTS smoother over the candidates ckf_find reported.
//
// the CKF's parameters are best at the LAST measurement; "a Kalman Filter-based fitting, which runs
// a smoothing algorithm called the Rauch-Tung-Striebel (RTS) smoother, is applied additionally to the tracks to
// make all track parameters consider all measurements".  Rules K1-K5 of DESIGN.md §3:
//   forward filter   level-synchronous like the CKF, one tip per track, the branch choice replaced by the candidate's
//                    list: the moves of a level run on the CKF's own ckf_step kernel (navigation, RKN4 + Jacobian),
//                    ckf_fit_level does the rest of the state with the CKF's per-tip code (arrival, covariance
//                    transport, Highland, gain-form update: ckf_nav.cuh / ckf_math.cuh); every visited module is a
//                    STATE whose predicted / filtered parameters, covariances and Jacobian go to the state store
//   ckf_fit_smooth   thread per track: RTS backward recursion over the stored states, float64 arithmetic in
//                    both modes (the gain needs the inverse of a predicted covariance whose entries span ten
//                    orders of magnitude; PAPER.md:61, :100 report the float32 smoother as unstable)
// State store: [state][component][track], track fastest, so the lanes of a warp (consecutive tracks) coalesce.
#pragma once
#include "ckf_branch.cuh"
#include "ckf_step.cuh"

namespace ckf {

constexpr int FIT_NT = 128;
constexpr int FIT_CHUNK = 262144;   // tracks per pass: bounds the state store (ckf.cu loops over the chunks)
// float64 per state: xp[6], xf[6], Cp[21], Cf[21] (packed upper triangles), the V5 variances (phi, theta) added on
// leaving the previous state -- the covariance algebra is float64 in both modes
// (FS_Q: q_phi, q_theta, and the energy-loss factor g of rule E, the q/p row of the full Jacobian being g e_4)
constexpr int FS_XP = 0, FS_XF = 6, FS_CP = 12, FS_CF = 33, FS_Q = 54, FS_X = 57;
constexpr int FS_T = 25;            // T per state: J (5x5 block, row-major), built from the T-typed transport Jacobian

template <typename T>
struct FitParams {
  GeoDev geo;
  FieldDev fld;
  CfgDev cfg;
  // event
  const int32_t* moff;
  const typename Vec2<T>::type* loc;
  const typename Vec2<T>::type* var;
  const int32_t* seed_module;
  const T* seed_x;
  const T* seed_C;
  // candidates, as ckf_find wrote them (device)
  const int32_t* n_tracks;
  const int32_t* offsets;
  const int32_t* meas;
  const int32_t* seed;
  int32_t max_tracks;   // capacity of the caller's per-track arrays
  int32_t first;        // first track of this pass
  int32_t chunk;        // tracks of this pass = stride of the state store
  int32_t max_states;
  double* fs_x;         // [max_states][FS_X][chunk]
  T* fs_t;              // [max_states][FS_T][chunk]
  int32_t* fs_meas;     // [max_states][chunk] measurement used by the state, -1 = module passed without one
  int32_t* fs_next;     // [chunk] list entries the track has consumed so far (level-synchronous forward filter)
  // output (device, caller-owned)
  int32_t* o_status; int32_t* o_nstates;
  T* o_chi2; T* o_lastx; T* o_lastC; T* o_firstC; T* o_entryx;
  unsigned long long* o_work;  // [4] or null: RKN4 trials, accepted steps, moves, updates are ADDED here
};

// ---- level-synchronous forward filter: the moves of a level run on the CKF's own ckf_step (persistent lanes,
// step schedule), one tip per track; this kernel is the rest of a level, thread per track: arrival (J4, J5),
// covariance transport, the listed measurement (or none), state store, departure + N2 + cost class of the next move.
// kp carries only what ckf_step needs (level arrays with tcap = chunk, globals, counters), all owned by the fit store.
constexpr int FIT_RUNNING = -1;

// The step schedule is double-buffered by level parity (two blocks of globals, G_N ints apart): kp.g is the block
// this level appends to for the next level's ckf_step; `g_done` is the block the ckf_step before this kernel
// consumed, which thread 0 clears for the level after next.
template <typename T, bool GRAD = false>
__global__ void __launch_bounds__(FIT_NT) ckf_fit_level(const KParams<T> kp, const FitParams<T> p, int level, int32_t* g_done) {
  chain_enter();
  if (blockIdx.x == 0 && threadIdx.x < G_N - G_STEP_CURSOR) g_done[G_STEP_CURSOR + threadIdx.x] = 0;
  const int nt = min(*p.n_tracks, p.max_tracks);
  const size_t CH = (size_t)p.chunk;
  const int s = blockIdx.x * FIT_NT + threadIdx.x;
  const int tr = p.first + s;
  unsigned long long w_moves = 0, w_upd = 0;
  int bin = -1;
  if (s < p.chunk && tr < nt && (level == 0 || p.o_status[tr] == FIT_RUNNING)) {
    const int e0 = p.offsets[tr], n = p.offsets[tr + 1] - e0;
    const int sd0 = p.seed[tr];
    const int eoff = (p.seed_module[sd0] / p.geo.n_modules) * p.geo.n_modules;  // batch of events: see KParams::n_vmod
    double xp[6], xf[6];
    double Cp[21], Cf[21], J[5][5];
    int status = STOP_NONE, module = 0, next = 0, stored = level;
    bool done = false;
    T c2sum = T(0);
    double q_in[3] = {0.0, 0.0, 1.0};
#pragma unroll
    for (int i = 0; i < 6; ++i) xf[i] = 0.0;
#pragma unroll
    for (int i = 0; i < 21; ++i) Cf[i] = 0.0;
    if (level == 0) {  // N6: the seed's own module, identity transport
      const int sd = sd0;
      bool ok = true;
#pragma unroll
      for (int i = 0; i < 6; ++i) { xp[i] = (double)p.seed_x[(size_t)sd * 6 + i]; ok = ok && isfinite(xp[i]); }
      ok = ok && (xp[3] > 0.0 && xp[3] < PI_D);
#pragma unroll
      for (int i = 0; i < 6; ++i)
#pragma unroll
        for (int j = i; j < 6; ++j) Cp[tri(i, j)] = (double)p.seed_C[(size_t)sd * 36 + i * 6 + j];
#pragma unroll
      for (int a = 0; a < 5; ++a)
#pragma unroll
        for (int b = 0; b < 5; ++b) J[a][b] = (a == b && a < 4) ? 1.0 : 0.0;
      module = p.seed_module[sd] - eoff;
      if (n < 1) done = true;
      else if (!ok) status = STOP_NUMERIC;
    } else {
      next = p.fs_next[s];
      c2sum = p.o_chi2[tr];
      w_moves += 1;
      status = kp.mv_stop[s];
      if (status == STOP_NONE) {
        Move<T> m;
        load_traj(kp.mv_y, (size_t)s, m.y);
        load_jac(kp.mv_D, (size_t)s, m.D);
        m.from = kp.mv_from[s];
        m.tgt = kp.mv_tgt[s];
        double dep[NDEP];
#pragma unroll
        for (int i = 0; i < NDEP; ++i) dep[i] = kp.mv_dep[i * CH + s];
        if constexpr (GRAD) {
          JacR<T> R;
          load_jacr(kp.mv_Dr, (size_t)s, R);
          status = move_arrive<T>(m, dep, p.geo, p.fld, p.cfg, xp, J, &R);
        } else {
          status = move_arrive<T>(m, dep, p.geo, p.fld, p.cfg, xp, J);
        }
        if (status == STOP_NONE) {
          double C[21];
          const double* pt = p.fs_x + (size_t)(level - 1) * FS_X * CH + s;  // filtered covariance of the previous state
#pragma unroll
          for (int i = 0; i < 21; ++i) C[i] = pt[(FS_CF + i) * CH];
          leave_module_cov(C, dep);  // V5 and rule E on leaving
          q_in[0] = dep[3]; q_in[1] = dep[4]; q_in[2] = dep[5];
          transport_cov<double>(J, C, Cp);
          bool fin = true;
#pragma unroll
          for (int i = 0; i < 21; ++i) fin = fin && isfinite(Cp[i]);
          if (!fin) status = STOP_NUMERIC;
          module = m.tgt;
        }
      }
    }
    if (status == STOP_NONE && !done) {
      const int k = p.meas[e0 + next];
      int used = -1;
      if (k >= p.moff[eoff + module] && k < p.moff[eoff + module + 1]) {
        const typename Vec2<T>::type mm = p.loc[k], vv = p.var[k];
        const double c2 = predicted_chi2<double>(xp[0], xp[1], Cp[tri(0, 0)], Cp[tri(0, 1)], Cp[tri(1, 1)], (double)mm.x,
                                                 (double)mm.y, (double)vv.x, (double)vv.y);
        c2sum += (T)c2;
        kalman_update(xp, Cp, mm.x, mm.y, vv.x, vv.y, xf, Cf);
        used = k;
        ++next;
        w_upd += 1;
      } else {
#pragma unroll
        for (int i = 0; i < 6; ++i) xf[i] = xp[i];
#pragma unroll
        for (int i = 0; i < 21; ++i) Cf[i] = Cp[i];
      }
      double* fx = p.fs_x + (size_t)level * FS_X * CH + s;
      T* ft = p.fs_t + (size_t)level * FS_T * CH + s;
#pragma unroll
      for (int i = 0; i < 6; ++i) { fx[(FS_XP + i) * CH] = xp[i]; fx[(FS_XF + i) * CH] = xf[i]; }
#pragma unroll
      for (int i = 0; i < 21; ++i) { fx[(FS_CP + i) * CH] = Cp[i]; fx[(FS_CF + i) * CH] = Cf[i]; }
#pragma unroll
      for (int a = 0; a < 5; ++a)
#pragma unroll
        for (int b = 0; b < 5; ++b) ft[(a * 5 + b) * CH] = (T)J[a][b];
      fx[(FS_Q + 0) * CH] = q_in[0];
      fx[(FS_Q + 1) * CH] = q_in[1];
      fx[(FS_Q + 2) * CH] = q_in[2];
      p.fs_meas[(size_t)level * CH + s] = used;
      stored = level + 1;
      if (next == n) done = true;
      else if (stored >= p.cfg.max_levels || stored >= p.max_states) status = STOP_LEVEL_LIMIT;
      else {
        Traj y;
        double dep[NDEP];
        status = departure_state(p.geo, p.cfg, module, xf, y, dep);
        if (status == STOP_NONE) {  // the track as a tip of the next level's ckf_step
          store_traj(kp.mv_y, (size_t)s, y);
#pragma unroll
          for (int i = 0; i < NDEP; ++i) kp.mv_dep[i * CH + s] = dep[i];
          kp.mv_from[s] = module;
          const int ov = overlap_neighbour(p.geo, module, y.r, y.d);  // N2
          kp.mv_tgt[CH + s] = ov;
          kp.mv_stop[s] = STOP_NONE;
          bin = step_cost_bin(p.geo, module, y, ov);
          p.fs_next[s] = next;
          p.o_chi2[tr] = c2sum;
          p.o_status[tr] = FIT_RUNNING;
          p.o_nstates[tr] = stored;
        }
      }
    }
    if (done || status != STOP_NONE) {  // the forward pass of this track ends here
      const bool good = status == STOP_NONE && stored > 0;
      p.o_status[tr] = status;
      p.o_nstates[tr] = stored;
      p.o_chi2[tr] = good ? c2sum : T(0);
#pragma unroll
      for (int i = 0; i < 6; ++i) p.o_lastx[(size_t)tr * 6 + i] = good ? (T)xf[i] : T(0);
#pragma unroll
      for (int i = 0; i < 6; ++i)
#pragma unroll
        for (int j = 0; j < 6; ++j) p.o_lastC[(size_t)tr * 36 + i * 6 + j] = good ? (T)Cf[tri(i, j)] : T(0);
    }
  }
  // step schedule of the next level: append the running track to its cost class (as ckf_update does)
  const unsigned live = __ballot_sync(0xffffffffu, bin >= 0);
  if (bin >= 0) {
    const int lane = threadIdx.x & 31;
    const unsigned peers = __match_any_sync(live, bin);
    const int leader = __ffs(peers) - 1;
    int base = 0;
    if (lane == leader) base = atomicAdd(kp.g + G_BIN0 + bin, __popc(peers));
    base = __shfl_sync(peers, base, leader);
    kp.mv_order[(size_t)bin * CH + base + __popc(peers & ((1u << lane) - 1u))] = s;
  }
  if (p.o_work) {
    flush_counter(p.o_work + 2, w_moves);
    flush_counter(p.o_work + 3, w_upd);
  }
}

// adds the RKN4 counters ckf_step accumulated for this pass to the caller's work counters
__global__ void ckf_fit_flush_work(const unsigned long long* counters, unsigned long long* o_work) {
  if (o_work && threadIdx.x == 0 && blockIdx.x == 0) {
    o_work[0] += counters[CNT_TRIALS];
    o_work[1] += counters[CNT_ACCEPTED];
  }
}

// ---- RTS smoother (K4).  Register-resident: the symmetric matrices stay packed (21 numbers), the gain is solved
// column by column in place, every loop is unrolled with constant indices (no local memory).
template <typename A>
__device__ __forceinline__ A wrap_pi(A a) {
  while (a > (A)PI_D) a -= (A)(2.0 * PI_D);
  while (a <= -(A)PI_D) a += (A)(2.0 * PI_D);
  return a;
}

// Cholesky of G scaled to unit diagonal: G' = S G S = L L^T, S = diag(1 / sqrt(G_ii)).  L is packed by rows
// (L[i][j], j <= i, at tri(j, i)).  false when G is not positive definite.
template <typename A>
__device__ __forceinline__ bool chol6_scaled(const A G[21], A s[6], A L[21]) {
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    if (!(G[tri(i, i)] > A(0))) return false;
    s[i] = A(1) / sqrt(G[tri(i, i)]);
  }
#pragma unroll
  for (int j = 0; j < 6; ++j) {
    A d = G[tri(j, j)] * s[j] * s[j];
#pragma unroll
    for (int k = 0; k < j; ++k) d -= L[tri(k, j)] * L[tri(k, j)];
    if (!(d > A(0))) return false;
    L[tri(j, j)] = sqrt(d);
#pragma unroll
    for (int i = j + 1; i < 6; ++i) {
      A v = G[tri(i, j)] * s[i] * s[j];
#pragma unroll
      for (int k = 0; k < j; ++k) v -= L[tri(k, i)] * L[tri(k, j)];
      L[tri(j, i)] = v / L[tri(j, j)];
    }
  }
  return true;
}

// one column: b <- G^-1 b with the factor above (L z = S b, L^T w = z, x = S w)
template <typename A>
__device__ __forceinline__ void chol6_solve(const A s[6], const A L[21], A b[6]) {
  A z[6];
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    A v = b[i] * s[i];
#pragma unroll
    for (int k = 0; k < i; ++k) v -= L[tri(k, i)] * z[k];
    z[i] = v / L[tri(i, i)];
  }
#pragma unroll
  for (int i = 5; i >= 0; --i) {
    A v = z[i];
#pragma unroll
    for (int k = i + 1; k < 6; ++k) v -= L[tri(i, k)] * b[k];
    b[i] = v / L[tri(i, i)];   // b[i..5] now hold w[i..5]
  }
#pragma unroll
  for (int i = 0; i < 6; ++i) b[i] *= s[i];
}

// A = arithmetic type of the recursion: double (the product's choice, K5), or float for the study of the float32
// smoother's instability that PAPER.md:61, :100 report (fp32 mode only).
#ifndef CKF_SMOOTH_MINB
#define CKF_SMOOTH_MINB 2
#endif
template <typename T, typename A>
__global__ void __launch_bounds__(FIT_NT, CKF_SMOOTH_MINB) ckf_fit_smooth(const FitParams<T> p) {
  const int nt = min(*p.n_tracks, p.max_tracks);
  const size_t CH = (size_t)p.chunk;
  for (int s = blockIdx.x * FIT_NT + threadIdx.x; s < p.chunk; s += gridDim.x * FIT_NT) {
    const int tr = p.first + s;
    if (tr >= nt) return;
    const int e0 = p.offsets[tr], n = p.offsets[tr + 1] - e0;
    const int ns = p.o_nstates[tr];
    bool good = p.o_status[tr] == STOP_NONE && ns > 0;
    A xs[6], Cs[21];
    int e = n - 1;  // entries are filled from the back: the forward pass ends on the last measurement
    if (good) {
      const double* fx = p.fs_x + (size_t)(ns - 1) * FS_X * CH + s;
      const T* ft = p.fs_t + (size_t)(ns - 1) * FS_T * CH + s;
#pragma unroll
      for (int i = 0; i < 6; ++i) xs[i] = (A)fx[(FS_XF + i) * CH];
#pragma unroll
      for (int i = 0; i < 21; ++i) Cs[i] = (A)fx[(size_t)(FS_CF + i) * CH];
      for (int k = ns - 1;; --k) {
        if (p.fs_meas[(size_t)k * CH + s] >= 0) {
#pragma unroll
          for (int i = 0; i < 6; ++i) p.o_entryx[(size_t)(e0 + e) * 6 + i] = (T)xs[i];
          if (e == 0) {  // first measurement of the track: the state PAPER.md:35 wants improved
#pragma unroll
            for (int i = 0; i < 6; ++i)
#pragma unroll
              for (int j = 0; j < 6; ++j) p.o_firstC[(size_t)tr * 36 + i * 6 + j] = (T)Cs[tri(i, j)];
          }
          --e;
        }
        if (k == 0 || e < 0) break;  // states before the first measurement are not reported
        // ---- one RTS step: state k -> k - 1.  b = state k (xp, Cp, J), a = state k - 1 (xf, Cf)
        const double* bx = p.fs_x + (size_t)k * FS_X * CH + s;
        const T* bt = p.fs_t + (size_t)k * FS_T * CH + s;
        const double* ax = p.fs_x + (size_t)(k - 1) * FS_X * CH + s;
        const T* at = p.fs_t + (size_t)(k - 1) * FS_T * CH + s;
        A sc[6], L[21], dC[21], Cf[21];
        {
          A G[21];
#pragma unroll
          for (int i = 0; i < 21; ++i) { G[i] = (A)bx[(size_t)(FS_CP + i) * CH]; dC[i] = Cs[i] - G[i]; }
          if (!chol6_scaled<A>(G, sc, L)) { good = false; break; }
        }
#pragma unroll
        for (int i = 0; i < 21; ++i) Cf[i] = (A)ax[(size_t)(FS_CF + i) * CH];
        // X = Cp^-1 (Jf Cf) = A_k^T, column by column.  Jf rows 0..3 = J[0..3] over columns 0..4, row 4 = e_4,
        // row 5 = J[4] plus 1 at column 5
        A X[6][6];
        {
          A Jb[5][5];
#pragma unroll
          for (int r = 0; r < 5; ++r)
#pragma unroll
            for (int l = 0; l < 5; ++l) Jb[r][l] = (A)bt[(size_t)(r * 5 + l) * CH];
          // rule E: the full Jacobian is J_arrival J_E, J_E = diag(1,1,1,1,g,1): column q/p times g, row q/p = g e_4
          const A gE = (A)bx[(size_t)(FS_Q + 2) * CH];
#pragma unroll
          for (int r = 0; r < 5; ++r) Jb[r][4] *= gE;
#pragma unroll
          for (int c = 0; c < 6; ++c) {
            A col[6];
#pragma unroll
            for (int i = 0; i < 6; ++i) {
              if (i == 4) col[i] = gE * Cf[tri(4, c)];
              else {
                const int r = (i == 5) ? 4 : i;
                A v = (i == 5) ? Cf[tri(5, c)] : A(0);
#pragma unroll
                for (int l = 0; l < 5; ++l) v += Jb[r][l] * Cf[tri(l, c)];
                col[i] = v;
              }
            }
            chol6_solve<A>(sc, L, col);
#pragma unroll
            for (int i = 0; i < 6; ++i) X[i][c] = col[i];
          }
        }
        A dx[6];
#pragma unroll
        for (int i = 0; i < 6; ++i) dx[i] = xs[i] - (A)bx[(FS_XP + i) * CH];
        dx[2] = wrap_pi<A>(dx[2]);
#pragma unroll
        for (int i = 0; i < 6; ++i) {
          A v = A(0);
#pragma unroll
          for (int j = 0; j < 6; ++j) v += X[j][i] * dx[j];
          xs[i] = (A)ax[(FS_XF + i) * CH] + v;
        }
        xs[2] = wrap_pi<A>(xs[2]);
        // Cs <- sym(Cf + X^T (dC X)), one column of dC X at a time
        A R[6][6];
#pragma unroll
        for (int j = 0; j < 6; ++j) {
          A t[6];
#pragma unroll
          for (int i = 0; i < 6; ++i) {
            A v = A(0);
#pragma unroll
            for (int l = 0; l < 6; ++l) v += dC[tri(i, l)] * X[l][j];
            t[i] = v;
          }
#pragma unroll
          for (int i = 0; i < 6; ++i) {
            A v = A(0);
#pragma unroll
            for (int l = 0; l < 6; ++l) v += X[l][i] * t[l];
            R[i][j] = Cf[tri(i, j)] + v;
          }
        }
#pragma unroll
        for (int i = 0; i < 6; ++i)
#pragma unroll
          for (int j = i; j < 6; ++j) Cs[tri(i, j)] = A(0.5) * (R[i][j] + R[j][i]);
      }
    }
    if (!good) {
      if (p.o_status[tr] == STOP_NONE && ns > 0) p.o_status[tr] = STOP_NUMERIC;  // a predicted covariance was not positive definite
      p.o_chi2[tr] = T(0);
      for (int i = 0; i < 6; ++i) p.o_lastx[(size_t)tr * 6 + i] = T(0);
      for (int i = 0; i < 36; ++i) { p.o_lastC[(size_t)tr * 36 + i] = T(0); p.o_firstC[(size_t)tr * 36 + i] = T(0); }
      for (int i = 0; i < 6 * n; ++i) p.o_entryx[(size_t)e0 * 6 + i] = T(0);
    }
  }
}

// ---- two-filter ("optimal") smoother K4' (the variant the paper names as more stable than RTS).
// The smoothed state = forward-filtered state combined with the information (Y, y) a BACKWARD filter has gathered from
// the later measurements, on the same linearised model as the RTS recursion (stored J, xp, xf, Cf, V5 noise), in
// deviations from xf[k].  No difference of nearly equal covariances appears:
//   Cf = B B^T (scaled Cholesky), A = I + B^T Y B = La La^T, U = La^-1 B^T:  Cs = U^T U,  xs = xf + U^T La^-1 B^T y.
// plain Cholesky of a packed symmetric 6x6 (lower factor packed by rows, L[i][j] at tri(j, i)); false if not p.d.
template <typename A>
__device__ __forceinline__ bool chol6(const A G[21], A L[21]) {
#pragma unroll
  for (int j = 0; j < 6; ++j) {
    A d = G[tri(j, j)];
#pragma unroll
    for (int k = 0; k < j; ++k) d -= L[tri(k, j)] * L[tri(k, j)];
    if (!(d > A(0))) return false;
    L[tri(j, j)] = sqrt(d);
#pragma unroll
    for (int i = j + 1; i < 6; ++i) {
      A v = G[tri(i, j)];
#pragma unroll
      for (int k = 0; k < j; ++k) v -= L[tri(k, i)] * L[tri(k, j)];
      L[tri(j, i)] = v / L[tri(j, j)];
    }
  }
  return true;
}

template <typename T, typename A>
__global__ void __launch_bounds__(FIT_NT, CKF_SMOOTH_MINB) ckf_fit_smooth_tf(const FitParams<T> p) {
  const int nt = min(*p.n_tracks, p.max_tracks);
  const size_t CH = (size_t)p.chunk;
  for (int s = blockIdx.x * FIT_NT + threadIdx.x; s < p.chunk; s += gridDim.x * FIT_NT) {
    const int tr = p.first + s;
    if (tr >= nt) return;
    const int e0 = p.offsets[tr], n = p.offsets[tr + 1] - e0;
    const int ns = p.o_nstates[tr];
    bool good = p.o_status[tr] == STOP_NONE && ns > 0;
    int e = n - 1;
    if (good) {
      A Y[21], y[6];  // backward information about the deviation of state k, from the measurements after k
#pragma unroll
      for (int i = 0; i < 21; ++i) Y[i] = A(0);
#pragma unroll
      for (int i = 0; i < 6; ++i) y[i] = A(0);
      for (int k = ns - 1;; --k) {
        const double* fx = p.fs_x + (size_t)k * FS_X * CH + s;
        const T* ft = p.fs_t + (size_t)k * FS_T * CH + s;
        const int used = p.fs_meas[(size_t)k * CH + s];
        if (used >= 0) {  // a reported state: combine
          A B[21];  // Cf = B B^T, B lower triangular, packed like a Cholesky factor
          {
            A Cf[21], sc[6], L[21];
#pragma unroll
            for (int i = 0; i < 21; ++i) Cf[i] = (A)fx[(size_t)(FS_CF + i) * CH];
            if (!chol6_scaled<A>(Cf, sc, L)) { good = false; break; }
#pragma unroll
            for (int i = 0; i < 6; ++i)
#pragma unroll
              for (int j = 0; j <= i; ++j) B[tri(j, i)] = L[tri(j, i)] / sc[i];
          }
          A Am[21], t[6];
          {
            A YB[6][6];  // Y B
#pragma unroll
            for (int i = 0; i < 6; ++i)
#pragma unroll
              for (int j = 0; j < 6; ++j) {
                A v = A(0);
#pragma unroll
                for (int l = j; l < 6; ++l) v += Y[tri(i, l)] * B[tri(j, l)];  // B[l][j], l >= j
                YB[i][j] = v;
              }
#pragma unroll
            for (int i = 0; i < 6; ++i) {
#pragma unroll
              for (int j = i; j < 6; ++j) {
                A v = (i == j) ? A(1) : A(0);
#pragma unroll
                for (int l = i; l < 6; ++l) v += B[tri(i, l)] * YB[l][j];  // B^T[i][l] = B[l][i], l >= i
                Am[tri(i, j)] = v;
              }
              A v = A(0);
#pragma unroll
              for (int l = i; l < 6; ++l) v += B[tri(i, l)] * y[l];
              t[i] = v;
            }
          }
          A La[21];
          if (!chol6<A>(Am, La)) { good = false; break; }
          // U = La^-1 B^T (forward substitution, column j of B^T = row j of B), w = La^-1 t
          A U[6][6], w[6];
#pragma unroll
          for (int i = 0; i < 6; ++i) {
#pragma unroll
            for (int j = 0; j < 6; ++j) {
              A v = (i <= j) ? B[tri(i, j)] : A(0);  // B^T[i][j] = B[j][i], non-zero for i <= j
#pragma unroll
              for (int l = 0; l < i; ++l) v -= La[tri(l, i)] * U[l][j];
              U[i][j] = v / La[tri(i, i)];
            }
            A v = t[i];
#pragma unroll
            for (int l = 0; l < i; ++l) v -= La[tri(l, i)] * w[l];
            w[i] = v / La[tri(i, i)];
          }
          A xs[6];
#pragma unroll
          for (int i = 0; i < 6; ++i) {
            A v = A(0);
#pragma unroll
            for (int l = 0; l < 6; ++l) v += U[l][i] * w[l];
            xs[i] = (A)fx[(FS_XF + i) * CH] + v;
          }
          xs[2] = wrap_pi<A>(xs[2]);
#pragma unroll
          for (int i = 0; i < 6; ++i) p.o_entryx[(size_t)(e0 + e) * 6 + i] = (T)xs[i];
          if (e == 0) {
#pragma unroll
            for (int i = 0; i < 6; ++i)
#pragma unroll
              for (int j = i; j < 6; ++j) {
                A v = A(0);
#pragma unroll
                for (int l = 0; l < 6; ++l) v += U[l][i] * U[l][j];
                p.o_firstC[(size_t)tr * 36 + i * 6 + j] = (T)v;
                p.o_firstC[(size_t)tr * 36 + j * 6 + i] = (T)v;
              }
          }
          --e;
        }
        if (k == 0 || e < 0) break;
        // ---- backward step k -> k - 1: measurement of state k, then back through d_k = c + Jf (d_{k-1} + u)
        if (used >= 0) {
          const typename Vec2<T>::type mm = p.loc[used], vv = p.var[used];
          Y[tri(0, 0)] += A(1) / (A)vv.x;
          Y[tri(1, 1)] += A(1) / (A)vv.y;
          y[0] += (A)((double)mm.x - fx[(FS_XF + 0) * CH]) / (A)vv.x;
          y[1] += (A)((double)mm.y - fx[(FS_XF + 1) * CH]) / (A)vv.y;
        }
        A yc[6];
        {
          A c6[6];
#pragma unroll
          for (int i = 0; i < 6; ++i) c6[i] = (A)(fx[(FS_XP + i) * CH] - fx[(FS_XF + i) * CH]);
          c6[2] = wrap_pi<A>(c6[2]);
#pragma unroll
          for (int i = 0; i < 6; ++i) {
            A v = y[i];
#pragma unroll
            for (int l = 0; l < 6; ++l) v -= Y[tri(i, l)] * c6[l];
            yc[i] = v;
          }
        }
        // Jf: rows 0..3 = J[0..3] over columns 0..4, row 4 = e_4, row 5 = J[4] plus 1 at column 5
        const A gE = (A)fx[(size_t)(FS_Q + 2) * CH];
        A Jf[6][6];
#pragma unroll
        for (int i = 0; i < 6; ++i)
#pragma unroll
          for (int j = 0; j < 6; ++j) {
            if (i == 4) Jf[i][j] = (j == 4) ? gE : A(0);     // rule E: J_arrival J_E
            else if (j == 5) Jf[i][j] = (i == 5) ? A(1) : A(0);
            else Jf[i][j] = (A)ft[(size_t)(((i == 5) ? 4 : i) * 5 + j) * CH] * ((j == 4) ? gE : A(1));
          }
        A Yz[21], yz[6];
        {
          A YJ[6][6];
#pragma unroll
          for (int i = 0; i < 6; ++i)
#pragma unroll
            for (int j = 0; j < 6; ++j) {
              A v = A(0);
#pragma unroll
              for (int l = 0; l < 6; ++l) v += Y[tri(i, l)] * Jf[l][j];
              YJ[i][j] = v;
            }
#pragma unroll
          for (int i = 0; i < 6; ++i) {
#pragma unroll
            for (int j = i; j < 6; ++j) {
              A v = A(0), u = A(0);
#pragma unroll
              for (int l = 0; l < 6; ++l) { v += Jf[l][i] * YJ[l][j]; u += Jf[l][j] * YJ[l][i]; }
              Yz[tri(i, j)] = A(0.5) * (v + u);
            }
            A v = A(0);
#pragma unroll
            for (int l = 0; l < 6; ++l) v += Jf[l][i] * yc[l];
            yz[i] = v;
          }
        }
        const A qp = (A)fx[(FS_Q + 0) * CH], qt = (A)fx[(FS_Q + 1) * CH];
        if (qp > A(0) && qt > A(0)) {  // marginalise the scattering angles u ~ N(0, diag(qp, qt)) on (phi, theta)
          const A s00 = A(1) / qp + Yz[tri(2, 2)], s01 = Yz[tri(2, 3)], s11 = A(1) / qt + Yz[tri(3, 3)];
          const A det = s00 * s11 - s01 * s01;
          if (!(det > A(0))) { good = false; break; }
          const A i00 = s11 / det, i01 = -s01 / det, i11 = s00 / det;
          A K2[6], K3[6];
#pragma unroll
          for (int i = 0; i < 6; ++i) {
            K2[i] = Yz[tri(i, 2)] * i00 + Yz[tri(i, 3)] * i01;
            K3[i] = Yz[tri(i, 2)] * i01 + Yz[tri(i, 3)] * i11;
          }
#pragma unroll
          for (int i = 0; i < 6; ++i) {
#pragma unroll
            for (int j = i; j < 6; ++j) {
              const A a = Yz[tri(i, j)] - (K2[i] * Yz[tri(2, j)] + K3[i] * Yz[tri(3, j)]);
              const A b = Yz[tri(i, j)] - (K2[j] * Yz[tri(2, i)] + K3[j] * Yz[tri(3, i)]);
              Y[tri(i, j)] = A(0.5) * (a + b);
            }
            y[i] = yz[i] - (K2[i] * yz[2] + K3[i] * yz[3]);
          }
        } else {
#pragma unroll
          for (int i = 0; i < 21; ++i) Y[i] = Yz[i];
#pragma unroll
          for (int i = 0; i < 6; ++i) y[i] = yz[i];
        }
      }
    }
    if (!good) {
      if (p.o_status[tr] == STOP_NONE && ns > 0) p.o_status[tr] = STOP_NUMERIC;
      p.o_chi2[tr] = T(0);
      for (int i = 0; i < 6; ++i) p.o_lastx[(size_t)tr * 6 + i] = T(0);
      for (int i = 0; i < 36; ++i) { p.o_lastC[(size_t)tr * 36 + i] = T(0); p.o_firstC[(size_t)tr * 36 + i] = T(0); }
      for (int i = 0; i < 6 * n; ++i) p.o_entryx[(size_t)e0 * 6 + i] = T(0);
    }
  }
}

}  // namespace ckf
