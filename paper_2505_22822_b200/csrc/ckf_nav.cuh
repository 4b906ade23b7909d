// ckf_nav.cuh — navigation (N2-N5), arrival Jacobian (J4, J5), covariance transport, material (V5),
// chi2 (V1) and Kalman update (V3) of the CKF hot path.  See ckf_math.cuh for the conventions.
#pragma once
#include "ckf_math.cuh"

namespace ckf {

struct GeoDev {
  const ModuleRec* mod;
  const LayerRec* layer;
  int32_t n_layers, n_modules;
  int32_t n_barrel;        // barrel layers come first, by increasing radius; disc layers follow
  int32_t first_disc[2];   // innermost disc of the +z side, of the -z side (-1 = none)
  int32_t bidir;           // config.bidirectional: inward-moving tips are navigated, modules may be crossed against n
};

constexpr int NDEP = 6;  // numbers of a departure record (departure_state): direction[3], q_phi, q_theta, g

// Packed upper triangle of a symmetric 6x6: index of (i, j), i <= j.
CKF_HD constexpr int tri(int i, int j) { return i <= j ? i * 6 - (i * (i - 1)) / 2 + (j - i) : j * 6 - (j * (j - 1)) / 2 + (i - j); }

// N2 / N4: straight-line test of one module from (r, d).
CKF_HD bool line_hits_module(const ModuleRec& k, const double r[3], const double d[3], double s_min, double& s_out,
                             int bidir = 0) {
  const double dn = dot3(d, k.n);
  if (bidir ? fabs(dn) <= 1e-6 : dn <= 1e-6) return false;
  const double rel[3] = {k.c[0] - r[0], k.c[1] - r[1], k.c[2] - r[2]};
  const double s = dot3(rel, k.n) / dn;
  const double q[3] = {r[0] + s * d[0] - k.c[0], r[1] + s * d[1] - k.c[1], r[2] + s * d[2] - k.c[2]};
  if (!(fabs(dot3(q, k.u)) <= k.half_u)) return false;
  if (!(fabs(dot3(q, k.v)) <= k.half_v)) return false;
  if (!(s > s_min)) return false;
  s_out = s;
  return true;
}

// The same test without early exits: path length, or NaN for "no hit".  Nine of these in a row have no control
// dependence between them, so the loads of the nine module records overlap (thread-per-tip callers: ckf_update's N2,
// ckf_fit_level; a chain of nine dependent L2 round trips was 25 % of ckf_update's stall samples).
CKF_HD double line_test_module(const ModuleRec& k, const double r[3], const double d[3], double s_min, int bidir = 0) {
  const double dn = dot3(d, k.n);
  const double rel[3] = {k.c[0] - r[0], k.c[1] - r[1], k.c[2] - r[2]};
  const double s = dot3(rel, k.n) / dn;
  const double q[3] = {r[0] + s * d[0] - k.c[0], r[1] + s * d[1] - k.c[1], r[2] + s * d[2] - k.c[2]};
  const bool ok = (bidir ? fabs(dn) > 1e-6 : dn > 1e-6) && fabs(dot3(q, k.u)) <= k.half_u && fabs(dot3(q, k.v)) <= k.half_v && s > s_min;
#if defined(__CUDA_ARCH__)
  return ok ? s : __longlong_as_double(0x7ff8000000000000LL);
#else
  return ok ? s : NAN;
#endif
}

// The same test on a record held as 16 doubles in ModuleRec order (c, u, v, n, half_u, half_v, ..), and the loader that
// fills it with four 256-bit loads on the device.
CKF_HD void ld_module_rec(const ModuleRec* k, double rec[16]) {
#if defined(__CUDA_ARCH__)
#pragma unroll
  for (int i = 0; i < 4; ++i)
    asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];"
        : "=d"(rec[4 * i]), "=d"(rec[4 * i + 1]), "=d"(rec[4 * i + 2]), "=d"(rec[4 * i + 3])
        : "l"((const double*)k + 4 * i));
#else
  const double* q = (const double*)k;
  for (int i = 0; i < 16; ++i) rec[i] = q[i];
#endif
}
// A module record in registers: the fields the per-tip code uses, filled by four 256-bit loads.
struct ModuleLite {
  double c[3], u[3], v[3], n[3], half_u, half_v, xx0;
};
CKF_HD void load_module(const ModuleRec* k, ModuleLite& o) {
  double rec[16];
  ld_module_rec(k, rec);
#pragma unroll
  for (int i = 0; i < 3; ++i) { o.c[i] = rec[i]; o.u[i] = rec[3 + i]; o.v[i] = rec[6 + i]; o.n[i] = rec[9 + i]; }
  o.half_u = rec[12]; o.half_v = rec[13]; o.xx0 = rec[14];
}
CKF_HD double line_test_rec(const double rec[16], const double r[3], const double d[3], double s_min, int bidir = 0) {
  const double *c = rec, *u = rec + 3, *v = rec + 6, *n = rec + 9;
  const double half_u = rec[12], half_v = rec[13];
  const double dn = dot3(d, n);
  const double rel[3] = {c[0] - r[0], c[1] - r[1], c[2] - r[2]};
  const double s = dot3(rel, n) / dn;
  const double q[3] = {r[0] + s * d[0] - c[0], r[1] + s * d[1] - c[1], r[2] + s * d[2] - c[2]};
  const bool ok = (bidir ? fabs(dn) > 1e-6 : dn > 1e-6) && fabs(dot3(q, u)) <= half_u && fabs(dot3(q, v)) <= half_v && s > s_min;
#if defined(__CUDA_ARCH__)
  return ok ? s : __longlong_as_double(0x7ff8000000000000LL);
#else
  return ok ? s : NAN;
#endif
}

// Nearest in-bounds module of the 3x3 neighbourhood (phi wraps, z clamps) of (iphi, iz) on `layer`, one tip per
// thread.  ckf_step evaluates the same nine tests cooperatively over a warp, see pick_warp.
CKF_HD int pick_in_neighbourhood(const GeoDev& g, int layer, int iphi, int iz, int exclude, const double r[3],
                                 const double d[3], double s_min) {
  const LayerRec L = g.layer[layer];
  double sv[9];
  int idv[9];
#pragma unroll
  for (int nb = 0; nb < 9; ++nb) {
    int ii = iphi + (nb / 3 - 1);
    ii = ii < 0 ? ii + L.n_phi : (ii >= L.n_phi ? ii - L.n_phi : ii);
    const int jj = iz + (nb % 3 - 1);
    const int id = L.offset + ii * L.n_z + jj;
    const bool test = jj >= 0 && jj < L.n_z && id != exclude;   // a predicate, not a branch around the loads
    double rec[16];   // the record as four 256-bit loads (see pick_warp); an untested neighbour reads a valid record
    ld_module_rec(g.mod + (test ? id : L.offset), rec);
    sv[nb] = test ? line_test_rec(rec, r, d, s_min, g.bidir) : 0.0;
    idv[nb] = test ? id : -1;
  }
  int best = -1;
  double best_s = 0.0;
#pragma unroll
  for (int nb = 0; nb < 9; ++nb) {   // the sequential rule's order: nearest first, tie -> lower id
    const double s = sv[nb];
    const int id = idv[nb];
    if (id >= 0 && s == s && (best < 0 || s < best_s || (s == best_s && id < best))) { best = id; best_s = s; }
  }
  return best;
}

// V5: Highland theta0^2 for a tip leaving module m with direction d (unit) and q/p.
CKF_HD double highland_theta0_sq(double xx0, double cosi, double qop, double mass) {
  const double p = 1.0 / fabs(qop);
  const double beta = p / sqrt(p * p + mass * mass);
  const double X = xx0 / cosi;
  const double th0 = 0.0136 / (beta * p) * sqrt(X) * (1.0 + 0.038 * log(X / (beta * beta)));
  return th0 * th0;
}

// E: mean energy loss of the muon hypothesis in a silicon module (rule E).  Mean stopping power
// of a heavy singly charged particle (Bethe, PDG review "Passage of particles through matter"), density correction
// neglected, in GeV cm^2 / g:  K (Z/A) / beta^2 [ 1/2 ln(2 me (beta gamma)^2 Wmax / I^2) - beta^2 ],
// Wmax = 2 me (beta gamma)^2 / (1 + 2 gamma me/M + (me/M)^2);  silicon: Z/A 0.49848, I 173 eV, X0 21.82 g/cm^2.
CKF_HD double mean_dedx_silicon(double p, double M) {
  const double me = 0.51099895e-3, I = 173.0e-9, KZA = 0.307075e-3 * 0.49848;
  const double E = sqrt(p * p + M * M);
  const double bg2 = (p * p) / (M * M), beta2 = (p * p) / (E * E), rm = me / M;
  const double wmax = 2.0 * me * bg2 / (1.0 + 2.0 * (E / M) * rm + rm * rm);
  return KZA / beta2 * (0.5 * log(2.0 * me * bg2 * wmax / (I * I)) - beta2);
}

// J4 + J5: the non-trivial 5x5 block of the bound->bound Jacobian.  Rows (l0, l1, phi, theta, t), columns
// (l0, l1, phi, theta, q/p); the full 6x6 has row q/p = e_4, column t = e_5.
//   dep_u, dep_v : axes of the departure module;  dep_d : direction at departure (gives d d/d phi, d d/d theta)
//   arr          : arrival module;  y : state on its plane;  B : field there
// T = arithmetic type of the bound->bound block (float64 in the product), TD = type the running
// transport Jacobian D was accumulated in (float32 in fp32 mode).
template <typename T, typename TD, typename MOD>
CKF_HD void arrival_jacobian(const Jac<TD>& D, const double dep_u[3], const double dep_v[3], const T dep_d[3],
                             const MOD& arr, const Traj& y, const double Bd[3], double mass, T J[5][5],
                             const JacR<TD>* R = nullptr) {
  const double lam = KAPPA * y.qop;
  double kd[3];
  cross3(y.d, Bd, kd);
  T k[3], n[3], u0[3], v0[3], dT[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    k[i] = (T)(lam * kd[i]);
    n[i] = (T)arr.n[i];
    u0[i] = R ? (T)R->Ru[i] : (T)dep_u[i];   // dr/dl0, dr/dl1: the departure axes unless J2' transported them
    v0[i] = R ? (T)R->Rv[i] : (T)dep_v[i];
    dT[i] = (T)y.d[i];
  }
  const T nd = dot3(n, dT);
  const T ib = (T)inv_beta(y.qop, mass);
  // departure: d d/d phi = (-dy, dx, 0);  d d/d theta = (dz dx / st, dz dy / st, -st)
  const T st0 = sqrt(dep_d[0] * dep_d[0] + dep_d[1] * dep_d[1]);
  const T gphi[3] = {-dep_d[1], dep_d[0], T(0)};
  const T gth[3] = {dep_d[2] * dep_d[0] / st0, dep_d[2] * dep_d[1] / st0, -st0};
  // arrival: d phi/d d = (-dy, dx, 0) / st^2;  d theta/d d = (dz dx / st, dz dy / st, -st)
  const T st2 = dT[0] * dT[0] + dT[1] * dT[1];
  const T st = sqrt(st2);
  const T fphi[3] = {-dT[1] / st2, dT[0] / st2, T(0)};
  const T fth[3] = {dT[2] * dT[0] / st, dT[2] * dT[1] / st, -st};
  // n^T Rd, n.rq, n.u0, n.v0
  T nR[3];
#pragma unroll
  for (int j = 0; j < 3; ++j) nR[j] = n[0] * D.Rd[0][j] + n[1] * D.Rd[1][j] + n[2] * D.Rd[2][j];
  const T nrq = (T)dot3(n, D.rq), nu0 = dot3(n, u0), nv0 = dot3(n, v0);
  const T nRgphi = dot3(nR, gphi), nRgth = dot3(nR, gth);
  // rows l0, l1
#pragma unroll
  for (int a = 0; a < 2; ++a) {
    T w[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) w[i] = (T)(a == 0 ? arr.u[i] : arr.v[i]);
    const T f = dot3(w, dT) / nd;
    T wp[3], wR[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) wp[i] = w[i] - f * n[i];
#pragma unroll
    for (int j = 0; j < 3; ++j) wR[j] = wp[0] * D.Rd[0][j] + wp[1] * D.Rd[1][j] + wp[2] * D.Rd[2][j];
    J[a][0] = dot3(wp, u0);
    J[a][1] = dot3(wp, v0);
    J[a][2] = dot3(wR, gphi);
    J[a][3] = dot3(wR, gth);
    J[a][4] = (T)dot3(wp, D.rq);
  }
  // rows phi, theta
#pragma unroll
  for (int a = 0; a < 2; ++a) {
    T f[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) f[i] = (a == 0 ? fphi[i] : fth[i]);
    const T fk = dot3(f, k) / nd;
    T row[3];
#pragma unroll
    for (int j = 0; j < 3; ++j) row[j] = f[0] * D.Dd[0][j] + f[1] * D.Dd[1][j] + f[2] * D.Dd[2][j] - fk * nR[j];
    J[2 + a][0] = -fk * nu0;
    J[2 + a][1] = -fk * nv0;
    if (R) {  // dd/dl0, dd/dl1 (zero without the gradient terms)
      J[2 + a][0] += f[0] * (T)R->Du[0] + f[1] * (T)R->Du[1] + f[2] * (T)R->Du[2];
      J[2 + a][1] += f[0] * (T)R->Dv[0] + f[1] * (T)R->Dv[1] + f[2] * (T)R->Dv[2];
    }
    J[2 + a][2] = dot3(row, gphi);
    J[2 + a][3] = dot3(row, gth);
    J[2 + a][4] = (T)dot3(f, D.dq) - fk * nrq;
  }
  // row t
  const T c = ib / nd;
  J[4][0] = -c * nu0;
  J[4][1] = -c * nv0;
  J[4][2] = -c * nRgphi;
  J[4][3] = -c * nRgth;
  J[4][4] = (T)D.tq - c * nrq;
}

// Covariance of a tip on LEAVING its module: V5 noise on (phi, theta), then rule E, C <- J_E C J_E^T with
// J_E = diag(1, 1, 1, 1, g, 1).
CKF_HD void leave_module_cov(double C[21], const double dep[NDEP]) {
  C[tri(2, 2)] += dep[3];
  C[tri(3, 3)] += dep[4];
  const double g = dep[5];
#pragma unroll
  for (int i = 0; i < 6; ++i) C[tri(i, 4)] *= g;
  C[tri(4, 4)] *= g;
}

// C' = Jf C Jf^T on the packed upper triangle, Jf = full 6x6 built from the 5x5 block (see arrival_jacobian).
template <typename T>
CKF_HD void transport_cov(const T J[5][5], const T C[21], T Co[21]) {
  // rows of Jf: 0..3 -> J[0..3] over cols 0..4;  4 -> e_4;  5 -> J[4] over cols 0..4 plus 1 at col 5
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    T t[6];  // row i of Jf C
    if (i == 4) {
#pragma unroll
      for (int j = 0; j < 6; ++j) t[j] = C[tri(4, j)];
    } else {
      const int ri = (i == 5) ? 4 : i;
#pragma unroll
      for (int j = 0; j < 6; ++j) {
        T s = (i == 5) ? C[tri(5, j)] : T(0);
#pragma unroll
        for (int k = 0; k < 5; ++k) s += J[ri][k] * C[tri(k, j)];
        t[j] = s;
      }
    }
#pragma unroll
    for (int j = i; j < 6; ++j) {
      T s;
      if (j == 4) s = t[4];
      else {
        const int rj = (j == 5) ? 4 : j;
        s = (j == 5) ? t[5] : T(0);
#pragma unroll
        for (int k = 0; k < 5; ++k) s += t[k] * J[rj][k];
      }
      Co[tri(i, j)] = s;
    }
  }
}

// V1: chi2 of one measurement against predicted (l0, l1) [float64] and the 2x2 block of C.
template <typename T>
CKF_HD T predicted_chi2(double l0, double l1, T C00, T C01, T C11, T m0, T m1, T v0, T v1) {
  const T r0 = (T)((double)m0 - l0), r1 = (T)((double)m1 - l1);
  const T S00 = C00 + v0, S11 = C11 + v1;
  const T det = S00 * S11 - C01 * C01;
  return (r0 * r0 * S11 - T(2) * r0 * r1 * C01 + r1 * r1 * S00) / det;
}

// V1 + V2 gate of one measurement against a float64 prediction (l0, l1, C00, C01, C11).  M = element type of the
// measurement arrays.  M = float: a float32 pre-filter with a generous margin rejects the bulk of the slice; the few
// survivors are re-evaluated in float64, so the decision and the reported chi2 are float64 functions of the inputs
// (DESIGN.md §4).  M = double: one evaluation.
template <typename M>
CKF_HD bool gate_chi2(double l0, double l1, double C00, double C01, double C11, M m0, M m1, M v0, M v1, double chi2_max,
                      double& chi2) {
  if (sizeof(M) == 4) {
    const float c = predicted_chi2<float>(l0, l1, (float)C00, (float)C01, (float)C11, (float)m0, (float)m1, (float)v0, (float)v1);
    if (!(c < (float)chi2_max * 1.01f + 0.01f)) return false;
  }
  const double cd = predicted_chi2<double>(l0, l1, C00, C01, C11, (double)m0, (double)m1, (double)v0, (double)v1);
  chi2 = cd;
  return cd < chi2_max;
}

// V3: gain-form update, float64 in both modes (x, C packed upper triangle); M = element type of the measurement.
// C' = C - K H C cancels two to three digits when a precise hit meets a loose prediction.
template <typename M>
CKF_HD void kalman_update(const double x[6], const double C[21], M m0, M m1, M v0, M v1, double xo[6], double Co[21]) {
  const double r0 = (double)m0 - x[0], r1 = (double)m1 - x[1];
  const double S00 = C[tri(0, 0)] + (double)v0, S01 = C[tri(0, 1)], S11 = C[tri(1, 1)] + (double)v1;
  const double det = S00 * S11 - S01 * S01;
  const double I00 = S11 / det, I01 = -S01 / det, I11 = S00 / det;
  double K0[6], K1[6];
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    K0[i] = C[tri(i, 0)] * I00 + C[tri(i, 1)] * I01;
    K1[i] = C[tri(i, 0)] * I01 + C[tri(i, 1)] * I11;
  }
#pragma unroll
  for (int i = 0; i < 6; ++i) xo[i] = x[i] + (K0[i] * r0 + K1[i] * r1);
#pragma unroll
  for (int i = 0; i < 6; ++i)
#pragma unroll
    for (int j = i; j < 6; ++j)
      Co[tri(i, j)] = C[tri(i, j)] - (K0[i] * C[tri(0, j)] + K1[i] * C[tri(1, j)]);
  while (xo[2] > PI_D) xo[2] -= 2.0 * PI_D;
  while (xo[2] <= -PI_D) xo[2] += 2.0 * PI_D;
}

// ------------------------------------------------------------------------------------------ one move (step A)
// From bound x on module `from` to the next module: N2-N5 with P and J, as a per-tip state machine whose
// transitions are small functions.  The kernel (ckf_level_loop.cuh) keeps one Move per lane and calls the
// transitions at warp-wide service points: lanes fetch new tips, pick modules, run RKN4 trials and do the
// arrival algebra together, so every heavy piece of code runs converged.  The host test harness drives the
// very same transitions one tip at a time (move_to_next_module below) against the oracle.
//
//   START --pick--> PLANE | CYL | FIN(EXIT)         N2 overlap neighbour, else next layer's cylinder
//   CYL   --step--> CYL (one RKN4 trial) | LANDED    P3-P5 toward the portal cylinder of layer lp
//   LANDED--pick--> PLANE | CYL | FIN(EXIT)         N3/N4 module choice at the portal; a crack is not a hole;
//                                                   beyond every further layer's half length = EXIT (D11)
//   PLANE --step--> PLANE (one trial) | FIN          N5 toward the target module's plane
//   FIN   --arrive-> predicted bound parameters + 5x5 Jacobian block (J4, J5)
//   DISC  --step--> DISC | LANDED                   like CYL toward the plane of a disc layer (row f3)
//   CYL_IN / CYL_FAR (config.bidirectional, rules N3''): toward the outer envelope of an inner layer, crossed inward;
//                   toward the far side of the cylinder that bounds the tip's shell
enum MovePhase : int { PH_IDLE = 0, PH_START = 1, PH_CYL = 2, PH_LANDED = 3, PH_PLANE = 4, PH_FIN = 5, PH_DISC = 6,
                       PH_CYL_IN = 7, PH_CYL_FAR = 8 };

CKF_HD bool is_stepping(int phase) {
  return phase == PH_CYL || phase == PH_PLANE || phase == PH_DISC || phase == PH_CYL_IN || phase == PH_CYL_FAR;
}

template <typename T>
struct Move {
  Traj y;
  Jac<T> D;
  double tc[3], tn[3];  // target plane (PH_PLANE)
  double R;             // target cylinder radius (PH_CYL)
  double h, h_ctrl;
  double ib, dib;       // 1/beta and d(1/beta)/d(q/p): constant along the move (no energy loss)
  double B1[3];         // field at y.r, valid while `targeted` (read once per position, see move_target)
  int phase, from, tgt, n_steps;
  // navigation cursors, packed into one register (ckf_step sits at its register cap): they are touched once or twice
  // per move, never inside the trial loop
  int lp : 9;           // layer of the portal being targeted / just landed on
  int lb : 9;           // portals (N3'): last barrel cylinder inside the tip (the next one outward is lb + 1), -1 none
  int ld : 9;           // next disc candidate, -1 none
  int stop : 4;         // stop reason so far
  bool inward;          // the cylinder portal being targeted / just landed on is crossed inward (CYL_IN)
  bool targeted;        // the next trial's length m.h and B1 are set (P4 done for the current position)
};

// A move that also transports the two position columns of D (J2', config.field_gradient).
template <typename T>
struct MoveG : Move<T> {
  JacR<T> Dr;
};
template <typename M> struct MoveTraits;
template <typename T> struct MoveTraits<Move<T>> { typedef T Scalar; static constexpr bool kGrad = false; };
template <typename T> struct MoveTraits<MoveG<T>> { typedef T Scalar; static constexpr bool kGrad = true; };

// Departure state of a tip with bound parameters x on module `from` (J1, V5): global position and direction,
// the direction again for the bound->free Jacobian, the Highland variances to add to C[phi][phi], C[theta][theta] on
// leaving (dep[3], dep[4]) and, with rule E, q/p after the mean energy loss in the module (y.qop) with
// dep[5] = g = d(q/p)'/d(q/p) = (p/p')^3 (E'/E), the energy lost held fixed (1 when rule E is off).
// Returns STOP_NUMERIC for non-finite parameters, theta outside (0, pi), or a particle that would stop in the module.
CKF_HD int departure_state(const GeoDev& g, const CfgDev& cfg, int from, const double x[6], Traj& y, double dep[NDEP]) {
  bool ok = true;
#pragma unroll
  for (int i = 0; i < 6; ++i) ok = ok && isfinite(x[i]);
  ok = ok && (x[3] > 0.0 && x[3] < PI_D);
  if (!ok) return STOP_NUMERIC;
  ModuleLite k;
  load_module(g.mod + from, k);
  double sp, cp, st, ct;
  sincos(x[2], &sp, &cp);
  sincos(x[3], &st, &ct);
  y.d[0] = st * cp; y.d[1] = st * sp; y.d[2] = ct;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    y.r[i] = k.c[i] + x[0] * k.u[i] + x[1] * k.v[i];
    dep[i] = y.d[i];
  }
  y.t = x[5];
  y.qop = x[4];
  dep[3] = 0.0;  // q_phi
  dep[4] = 0.0;  // q_theta
  dep[5] = 1.0;  // g
  if (k.xx0 > 0.0) {
    const double cosi = fabs(dot3(y.d, k.n));
    const double th2 = highland_theta0_sq(k.xx0, cosi, y.qop, cfg.mass);   // V5: with the momentum the tip arrived with
    dep[4] = th2;
    dep[3] = th2 / (st * st);
    if (cfg.energy_loss) {
      const double p = 1.0 / fabs(y.qop), E = sqrt(p * p + cfg.mass * cfg.mass);
      const double dE = mean_dedx_silicon(p, cfg.mass) * (k.xx0 / cosi) * 21.82;
      const double E2 = E - dE, p2 = sqrt(E2 * E2 - cfg.mass * cfg.mass);
      y.qop = (y.qop < 0.0 ? -1.0 : 1.0) / p2;
      dep[5] = (p / p2) * (p / p2) * (p / p2) * (E2 / E);
      if (!isfinite(y.qop)) return STOP_NUMERIC;
    }
  }
  return STOP_NONE;
}

// Start of a move whose m.y holds the departure state: identity transport, fresh step control (P4, J3).
template <typename T>
CKF_HD void move_begin(Move<T>& m, const CfgDev& cfg, int from) {
  m.from = from; m.tgt = -1; m.lp = 0; m.lb = -1; m.ld = -1; m.n_steps = 0; m.targeted = false; m.inward = false; m.stop = STOP_NONE;
  m.h = 0.0; m.h_ctrl = cfg.h_max; m.R = 0.0;
  jac_identity(m.D);
  m.ib = inv_beta(m.y.qop, cfg.mass);
  m.dib = dinvbeta_dqop(m.y.qop, cfg.mass);
  m.phase = PH_START;
}

template <typename T>
CKF_HD void move_begin(MoveG<T>& m, const GeoDev& g, const CfgDev& cfg, int from) {
  move_begin(static_cast<Move<T>&>(m), cfg, from);
  jacr_begin(m.Dr, g.mod[from].u, g.mod[from].v);
}

// The 3x3 neighbourhood a move in PH_START / PH_LANDED wants tested.  Returns false when no module can be
// picked (portal point beyond the layer's half length).
struct PickRequest {
  int layer, iphi, iz, exclude;
  double s_min;
};
// N2 for a tip leaving module `from` at (r, d): nearest in-bounds overlap neighbour on the same layer, or -1.
CKF_HD int overlap_neighbour(const GeoDev& g, int from, const double r[3], const double d[3]) {
  const ModuleRec& k = g.mod[from];
  const int iz = from - g.layer[k.layer].offset - k.iphi * g.layer[k.layer].n_z;
  return pick_in_neighbourhood(g, k.layer, k.iphi, iz, from, r, d, 1e-3);
}

// What a move in PH_START / PH_LANDED needs next: PICK_TEST (test the 3x3 neighbourhood in q) or PICK_SKIP (the portal
// point lies outside the layer's acceptance: on to the next portal).  For a move that has just LANDED on a portal this
// also books the landing: the cylinder is passed (lb), the next disc of the side becomes the candidate (ld).
enum PickWhat : int { PICK_TEST = 1, PICK_SKIP = 0 };
CKF_HD int barrel_index_inside(const GeoDev& g, double rho) {   // last barrel layer with r <= rho, -1 if none
  int lb = -1;
  while (lb + 1 < g.n_barrel && g.layer[lb + 1].r <= rho) ++lb;
  return lb;
}
template <typename T>
CKF_HD int move_pick_request(Move<T>& m, const GeoDev& g, PickRequest& q) {
  if (m.phase == PH_START) {
    const ModuleRec& k = g.mod[m.from];
    q.layer = k.layer; q.iphi = k.iphi;
    q.iz = m.from - g.layer[k.layer].offset - k.iphi * g.layer[k.layer].n_z;
    q.exclude = m.from; q.s_min = 1e-3;
    return PICK_TEST;
  }
  const LayerRec L = g.layer[m.lp];
  q.layer = m.lp; q.exclude = -1; q.s_min = -1e-3; q.iphi = 0; q.iz = 0;
  double along;
  if (L.kind == 0) {
    m.lb = m.inward ? m.lp - 1 : m.lp;   // crossed inward: the shell below it
    if (fabs(m.y.r[2]) > L.half_z) return PICK_SKIP;
    along = m.y.r[2] + L.half_z;
  } else {
    const double rho = sqrt(m.y.r[0] * m.y.r[0] + m.y.r[1] * m.y.r[1]);
    m.ld = L.next_disc;
    m.lb = barrel_index_inside(g, rho);
    if (rho < L.r_min || rho > L.r) return PICK_SKIP;
    along = rho - L.r_min;
  }
  const double phix = atan2(m.y.r[1], m.y.r[0]);
  const int i = (int)nearbyint(phix * L.n_phi / (2.0 * PI_D));
  q.iphi = ((i % L.n_phi) + L.n_phi) % L.n_phi;
  const int j = (int)floor(along / L.len_z);
  q.iz = j < 0 ? 0 : (j > L.n_z - 1 ? L.n_z - 1 : j);
  return PICK_TEST;
}

// N3': the next PORTAL of a move that has no module to go to -- the cylinder of the next barrel layer or the plane of
// the next disc in the direction of d_z, whichever the straight line from here reaches first (tie -> the cylinder).
// A barrel layer whose half length is already behind a tip that moves away in z, and a disc whose plane is not ahead
// or whose outer radius is behind a tip that moves outward radially, are passed without propagating to them (reading
// D11, per layer).  No portal left = the tip has left the detector (EXIT).
template <typename T>
CKF_HD void choose_portal(Move<T>& m, const GeoDev& g) {
  if (g.n_barrel == g.n_layers && !g.bidir) {
    // barrel only, outward only (the BASELINE configs): the rule below reduces to "the next barrel cylinder whose half
    // length is not behind the tip" -- kept as its own short path because it runs once or twice per move of the hot
    // kernel (measured: the general code costs ckf_step 3-5 %)
    int lb = (m.phase == PH_START) ? g.mod[m.from].layer : m.lb;
    const double z = m.y.r[2];
    if (z * m.y.d[2] > 0.0)
      while (lb + 1 < g.n_barrel && fabs(z) > g.layer[lb + 1].half_z) ++lb;
    m.lb = lb;
    m.targeted = false;
    if (lb + 1 >= g.n_barrel) { m.stop = STOP_EXIT; m.phase = PH_FIN; return; }
    m.lp = lb + 1;
    m.R = g.layer[lb + 1].r;
    m.phase = PH_CYL;
    return;
  }
  const double z = m.y.r[2], dz = m.y.d[2];
  const double rho2 = m.y.r[0] * m.y.r[0] + m.y.r[1] * m.y.r[1], bxy = m.y.r[0] * m.y.d[0] + m.y.r[1] * m.y.d[1];
  if (m.phase == PH_START) {   // leaving a module: where the tip stands in the two families of portals
    const LayerRec L0 = g.layer[g.mod[m.from].layer];
    if (L0.kind == 0) {
      m.lb = g.mod[m.from].layer;
      if (g.bidir && bxy < 0.0) m.lb -= 1;   // N3'': leaving a barrel module inward, its own cylinder is behind already
      m.ld = dz > 0.0 ? g.first_disc[0] : (dz < 0.0 ? g.first_disc[1] : -1);
    } else {
      m.lb = barrel_index_inside(g, sqrt(rho2));
      m.ld = L0.next_disc;
    }
  }
  const bool inward = g.bidir && bxy < 0.0;
  while (!inward && m.lb + 1 < g.n_barrel && fabs(z) > g.layer[m.lb + 1].half_z && z * dz > 0.0) ++m.lb;
  while (m.ld >= 0 && ((g.layer[m.ld].half_z - z) * dz <= 0.0 || (rho2 > g.layer[m.ld].r * g.layer[m.ld].r && bxy > 0.0)))
    m.ld = g.layer[m.ld].next_disc;
  int lc = m.lb + 1 < g.n_barrel ? m.lb + 1 : -1;
  int kind = PH_CYL;
  double r_target = 0.0;
  const double a = m.y.d[0] * m.y.d[0] + m.y.d[1] * m.y.d[1];
  if (inward) {
    // N3'': the next inner layer's outer envelope if the straight line reaches it, else the far side of the first
    // cylinder from lb + 1 outward that the line meets at all
    int li = m.lb;
    while (li >= 0 && fabs(z) > g.layer[li].half_z && z * dz > 0.0) --li;
    if (li >= 0) r_target = g.layer[li].r_in;
    if (li >= 0 && bxy * bxy - a * (rho2 - r_target * r_target) >= 0.0) { lc = li; kind = PH_CYL_IN; }
    else {
      kind = PH_CYL_FAR;
      while (lc >= 0 && bxy * bxy - a * (rho2 - g.layer[lc].r * g.layer[lc].r) < 0.0) lc = lc + 1 < g.n_barrel ? lc + 1 : -1;
    }
  }
  if (kind != PH_CYL_IN && lc >= 0) r_target = g.layer[lc].r;
  if (lc < 0 && m.ld < 0) { m.stop = STOP_EXIT; m.phase = PH_FIN; return; }
  bool to_disc = false;
  if (m.ld >= 0) {
    const double s_d = (g.layer[m.ld].half_z - z) / dz;
    double s_c = INFINITY;
    if (lc >= 0) {
      const double cc = rho2 - r_target * r_target;
      const double disc = bxy * bxy - a * cc;
      if (kind == PH_CYL) { if (bxy > 0.0 && disc >= 0.0) s_c = -cc / (bxy + sqrt(disc)); }
      else if (kind == PH_CYL_IN) s_c = cc / (-bxy + sqrt(disc));
      else if (disc >= 0.0) s_c = (-bxy + sqrt(disc)) / a;
    }
    to_disc = lc < 0 || s_d < s_c;
  }
  m.targeted = false;
  m.inward = false;
  if (!to_disc) {
    m.lp = lc;
    m.R = r_target;
    m.phase = kind;
    m.inward = kind == PH_CYL_IN;
  } else {
    m.lp = m.ld;
    const double zd = g.layer[m.ld].half_z;
    m.tc[0] = 0.0; m.tc[1] = 0.0; m.tc[2] = zd;
    m.tn[0] = 0.0; m.tn[1] = 0.0; m.tn[2] = zd > 0.0 ? 1.0 : -1.0;
    m.phase = PH_DISC;
  }
}

// Result of the pick (module id or -1) -> next phase.
template <typename T>
CKF_HD void move_pick_apply(Move<T>& m, const GeoDev& g, int tgt) {
  if (tgt >= 0) {
    const ModuleRec& k = g.mod[tgt];
#pragma unroll
    for (int i = 0; i < 3; ++i) { m.tc[i] = k.c[i]; m.tn[i] = k.n[i]; }
    m.tgt = tgt;
    m.phase = PH_PLANE;
    return;
  }
  choose_portal(m, g);   // no module here (no overlap neighbour / outside the acceptance / a crack): the next portal
}

// P4: signed straight-line distance from the move's position to its target (plane or cylinder) along d.
// Returns STOP_NONE and s, or the stop reason (P6).
template <typename T>
CKF_HD int target_distance(const Move<T>& m, double& s) {
  if (m.phase == PH_PLANE || m.phase == PH_DISC) {
    const double dn = dot3(m.y.d, m.tn);
    if (!(fabs(dn) > 1e-12)) return STOP_NUMERIC;
    const double rel[3] = {m.tc[0] - m.y.r[0], m.tc[1] - m.y.r[1], m.tc[2] - m.y.r[2]};
    s = dot3(rel, m.tn) / dn;
  } else {
    const double a = m.y.d[0] * m.y.d[0] + m.y.d[1] * m.y.d[1];
    const double b = m.y.r[0] * m.y.d[0] + m.y.r[1] * m.y.d[1];
    const double cc = m.y.r[0] * m.y.r[0] + m.y.r[1] * m.y.r[1] - m.R * m.R;
    const double disc = b * b - a * cc;
    if (m.phase == PH_CYL_IN) {          // near root from outside, moving inward (signed once overshot)
      if (!(b < 0.0) || !(disc >= 0.0)) return STOP_NOT_OUTGOING;   // it turned before reaching it
      s = cc / (-b + sqrt(disc));
    } else if (m.phase == PH_CYL_FAR) {  // far root, written without cancellation for either sign of b
      if (!(disc >= 0.0)) return STOP_NOT_OUTGOING;
      const double sq = sqrt(disc);
      s = b < 0.0 ? (-b + sq) / a : -cc / (b + sq);
    } else {
      if (!(b > 0.0) || !(disc >= 0.0)) return STOP_NOT_OUTGOING;
      s = -cc / (b + sqrt(disc));
    }
  }
  return isfinite(s) ? STOP_NONE : STOP_NUMERIC;
}

// The next trial from the current position: its length (P4) and the field there -- stage 1 of that trial and of every
// retry of it (a rejected trial restarts from the same point).
template <typename T>
CKF_HD void set_trial(Move<T>& m, const FieldDev& fld, const CfgDev& cfg, double s) {
  const double hlim = fmin(m.h_ctrl, cfg.h_max);
  m.h = (fabs(s) <= hlim) ? s : (s > 0.0 ? hlim : -hlim);
  field_at(fld, m.y.r, m.B1);
  m.targeted = true;
}

// P5 / P6 once no further trial follows: stop, or close onto the surface with a field-free step.
template <typename M>
CKF_HD void land_or_stop(M& m, int st, double s) {
  if (st != STOP_NONE) { m.stop = st; m.phase = PH_FIN; return; }
  straight_close(m.y, m.D, s, m.ib, m.dib);
  if constexpr (MoveTraits<M>::kGrad) straight_close_r(m.Dr, s);
  m.phase = (m.phase == PH_PLANE) ? PH_FIN : PH_LANDED;
}

// One step of a move in PH_CYL / PH_PLANE: targeting + landing (P4, P5), else one RKN4 trial (P2, P3).  After an
// accepted trial the next one is targeted at once and its stage-1 field read is issued BEFORE the Jacobian columns of
// the accepted step are computed, so that the loads fly during that arithmetic.
template <typename T, typename M>
CKF_HD void move_step(M& m, const FieldDev& fld, const CfgDev& cfg, int& n_trials, int& n_accepted) {
  constexpr bool GRAD = MoveTraits<M>::kGrad;
  if (!m.targeted) {   // a fresh position (start of a phase)
    double s = 0.0;
    const int st = target_distance(m, s);
    if (st != STOP_NONE || fabs(s) <= cfg.surf_tol) { land_or_stop(m, st, s); return; }
    set_trial(m, fld, cfg, s);
  }
  if (++m.n_steps > cfg.max_rk_steps) { m.stop = STOP_STEP_LIMIT; m.phase = PH_FIN; return; }
  Trial<T> t;
  rk_trial<T, GRAD>(fld, m.y, m.B1, KAPPA * m.y.qop, m.h, t);
  ++n_trials;
  if (!isfinite(t.eps)) { m.stop = STOP_NUMERIC; m.phase = PH_FIN; return; }
  // P3 factor 0.9 (tol / eps)^(1/4) clamped to [0.25, 4]; eps = 0 gives +inf, which the upper clamp turns into the
  // rule's 4 (no branch).  It is evaluated inside each arm of the accept test, after the work that does not need it, so
  // that its division and two square roots overlap that work instead of preceding the branch.
  auto step_factor = [&]() {
    double f = 0.9 * sqrt(sqrt(cfg.rk_tol / t.eps));
    f = f < 0.25 ? 0.25 : f;
    return f > 4.0 ? 4.0 : f;
  };
  if (t.eps <= cfg.rk_tol) {
    const double h = m.h;
    StepGrad<T> sg;
    if constexpr (GRAD) step_gradients<T>(fld, m.y, h, t, sg);   // at the stage points of the step, from the state before it
    rk_accept_state<T>(m.y, h, t, m.ib);
    ++n_accepted;
    m.targeted = false;
    double s = 0.0;
    const int st = target_distance(m, s);
    m.h_ctrl = fabs(h) * step_factor();
    const bool more = st == STOP_NONE && fabs(s) > cfg.surf_tol;
    if (more) set_trial(m, fld, cfg, s);            // the loads of the next trial's stage 1 start here ...
    if constexpr (GRAD) rk_accept_jac_g<T>(m.y.qop, m.D, m.Dr, h, t, sg, m.dib);
    else rk_accept_jac<T>(m.y, m.D, h, t, m.dib);   // ... and fly while D <- D_step D is computed
    if (!more) land_or_stop(m, st, s);              // the closing drift acts on the updated D
  } else {
    m.h = m.h * step_factor();                      // retry from the same position: same B1
  }
}

// Arrival (J4, J5) of a move in PH_FIN with stop == NONE: predicted bound parameters and the 5x5 Jacobian
// block.  Returns the final stop reason (NUMERIC if a predicted parameter is not finite).
template <typename T>
CKF_HD int move_arrive(const Move<T>& m, const double dep[NDEP], const GeoDev& g, const FieldDev& fld, const CfgDev& cfg,
                       double xp[6], double J[5][5], const JacR<T>* R = nullptr) {
  ModuleLite k, m0;
  load_module(g.mod + m.tgt, k);
  load_module(g.mod + m.from, m0);
  double B[3];
  field_at(fld, m.y.r, B);
  arrival_jacobian<double, T>(m.D, m0.u, m0.v, dep, k, m.y, B, cfg.mass, J, R);
  const double rel[3] = {m.y.r[0] - k.c[0], m.y.r[1] - k.c[1], m.y.r[2] - k.c[2]};
  xp[0] = dot3(rel, k.u);
  xp[1] = dot3(rel, k.v);
  xp[2] = atan2(m.y.d[1], m.y.d[0]);
  xp[3] = atan2(sqrt(m.y.d[0] * m.y.d[0] + m.y.d[1] * m.y.d[1]), m.y.d[2]);
  xp[4] = m.y.qop;
  xp[5] = m.y.t;
  bool fin = true;
#pragma unroll
  for (int i = 0; i < 6; ++i) fin = fin && isfinite(xp[i]);
  return fin ? STOP_NONE : STOP_NUMERIC;
}

// One tip at a time (host test harness): the transitions above in their natural order.
template <typename T, typename M>
CKF_HD int move_to_next_module_impl(const GeoDev& g, const FieldDev& fld, const CfgDev& cfg, int from, const double x[6],
                                    int& target, double xp[6], double J[5][5], double& q_phi, double& q_theta, double& g_e,
                                    StepCtl& sc) {
  M m;
  double dep[NDEP];
  const int st0 = departure_state(g, cfg, from, x, m.y, dep);
  if (st0 != STOP_NONE) return st0;
  if constexpr (MoveTraits<M>::kGrad) move_begin(m, g, cfg, from);
  else move_begin(m, cfg, from);
  while (m.phase != PH_FIN) {
    if (m.phase == PH_START || m.phase == PH_LANDED) {
      PickRequest q;
      const int what = move_pick_request(m, g, q);
      const int tgt = what == PICK_TEST ? pick_in_neighbourhood(g, q.layer, q.iphi, q.iz, q.exclude, m.y.r, m.y.d, q.s_min) : -1;
      move_pick_apply(m, g, tgt);
    } else {
      move_step<T>(m, fld, cfg, sc.n_trials, sc.n_accepted);
    }
  }
  q_phi = dep[3];
  q_theta = dep[4];
  g_e = dep[5];
  if (m.stop != STOP_NONE) return m.stop;
  int st;
  if constexpr (MoveTraits<M>::kGrad) st = move_arrive<T>(m, dep, g, fld, cfg, xp, J, &m.Dr);
  else st = move_arrive<T>(m, dep, g, fld, cfg, xp, J);
  if (st == STOP_NONE) target = m.tgt;
  return st;
}
template <typename T>
CKF_HD int move_to_next_module(const GeoDev& g, const FieldDev& fld, const CfgDev& cfg, int from, const double x[6],
                               int& target, double xp[6], double J[5][5], double& q_phi, double& q_theta, double& g_e,
                               StepCtl& sc) {
  if (cfg.field_gradient) return move_to_next_module_impl<T, MoveG<T>>(g, fld, cfg, from, x, target, xp, J, q_phi, q_theta, g_e, sc);
  return move_to_next_module_impl<T, Move<T>>(g, fld, cfg, from, x, target, xp, J, q_phi, q_theta, g_e, sc);
}

}  // namespace ckf
