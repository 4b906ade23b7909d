// ckf_nav.cuh — navigation (N2-N5), arrival Jacobian (J4, J5), covariance transport, material (V5),
// chi2 (V1) and Kalman update (V3) of the CKF hot path.  See ckf_math.cuh for the conventions.
#pragma once
#include "ckf_math.cuh"

namespace ckf {

struct GeoDev {
  const ModuleRec* mod;
  const LayerRec* layer;
  int32_t n_layers, n_modules;
};

// Packed upper triangle of a symmetric 6x6: index of (i, j), i <= j.
CKF_HD constexpr int tri(int i, int j) { return i <= j ? i * 6 - (i * (i - 1)) / 2 + (j - i) : j * 6 - (j * (j - 1)) / 2 + (i - j); }

// N2 / N4: straight-line test of one module from (r, d).
CKF_HD bool line_hits_module(const ModuleRec& k, const double r[3], const double d[3], double s_min, double& s_out) {
  const double dn = dot3(d, k.n);
  if (dn <= 1e-6) return false;
  const double rel[3] = {k.c[0] - r[0], k.c[1] - r[1], k.c[2] - r[2]};
  const double s = dot3(rel, k.n) / dn;
  const double q[3] = {r[0] + s * d[0] - k.c[0], r[1] + s * d[1] - k.c[1], r[2] + s * d[2] - k.c[2]};
  if (!(fabs(dot3(q, k.u)) <= k.half_u)) return false;
  if (!(fabs(dot3(q, k.v)) <= k.half_v)) return false;
  if (!(s > s_min)) return false;
  s_out = s;
  return true;
}

// Nearest in-bounds module of the 3x3 neighbourhood (phi wraps, z clamps) of (iphi, iz) on `layer`.
CKF_HD int pick_in_neighbourhood(const GeoDev& g, int layer, int iphi, int iz, int exclude, const double r[3],
                                 const double d[3], double s_min) {
  const LayerRec L = g.layer[layer];
  int best = -1;
  double best_s = 0.0;
  for (int di = -1; di <= 1; ++di) {
    int ii = iphi + di;
    ii = ii < 0 ? ii + L.n_phi : (ii >= L.n_phi ? ii - L.n_phi : ii);
    for (int dj = -1; dj <= 1; ++dj) {
      const int jj = iz + dj;
      if (jj < 0 || jj >= L.n_z) continue;
      const int id = L.offset + ii * L.n_z + jj;
      if (id == exclude) continue;
      double s;
      if (!line_hits_module(g.mod[id], r, d, s_min, s)) continue;
      if (best < 0 || s < best_s || (s == best_s && id < best)) { best = id; best_s = s; }
    }
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

// J4 + J5: the non-trivial 5x5 block of the bound->bound Jacobian.  Rows (l0, l1, phi, theta, t), columns
// (l0, l1, phi, theta, q/p); the full 6x6 has row q/p = e_4, column t = e_5.
//   dep_u, dep_v : axes of the departure module;  dep_d : direction at departure (gives d d/d phi, d d/d theta)
//   arr          : arrival module;  y : state on its plane;  B : field there
template <typename T>
CKF_HD void arrival_jacobian(const Jac<T>& D, const double dep_u[3], const double dep_v[3], const T dep_d[3],
                             const ModuleRec& arr, const Traj& y, const double Bd[3], double mass, T J[5][5]) {
  const double lam = KAPPA * y.qop;
  double kd[3];
  cross3(y.d, Bd, kd);
  T k[3], n[3], u0[3], v0[3], dT[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    k[i] = (T)(lam * kd[i]);
    n[i] = (T)arr.n[i];
    u0[i] = (T)dep_u[i];
    v0[i] = (T)dep_v[i];
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
  const T nrq = dot3(n, D.rq), nu0 = dot3(n, u0), nv0 = dot3(n, v0);
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
    J[a][4] = dot3(wp, D.rq);
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
    J[2 + a][2] = dot3(row, gphi);
    J[2 + a][3] = dot3(row, gth);
    J[2 + a][4] = dot3(f, D.dq) - fk * nrq;
  }
  // row t
  const T c = ib / nd;
  J[4][0] = -c * nu0;
  J[4][1] = -c * nv0;
  J[4][2] = -c * nRgphi;
  J[4][3] = -c * nRgth;
  J[4][4] = D.tq - c * nrq;
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

// V1 + V2 gate of one measurement.  T = float: a float32 pre-filter with a generous margin rejects the bulk
// of the slice; the few survivors are re-evaluated in float64 so that the decision and the reported chi2 do
// not carry float32 cancellation error.  T = double: one evaluation.
template <typename T>
CKF_HD bool gate_chi2(double l0, double l1, T C00, T C01, T C11, T m0, T m1, T v0, T v1, T chi2_max, T& chi2) {
  const T c = predicted_chi2<T>(l0, l1, C00, C01, C11, m0, m1, v0, v1);
  if (sizeof(T) == 8) {
    chi2 = c;
    return c < chi2_max;
  }
  if (!(c < chi2_max * T(1.01) + T(0.01))) return false;
  const double cd = predicted_chi2<double>(l0, l1, (double)C00, (double)C01, (double)C11, (double)m0, (double)m1,
                                           (double)v0, (double)v1);
  chi2 = (T)cd;
  return cd < (double)chi2_max;
}

// V3: gain-form update.  x float64 in/out, C packed upper triangle in/out (stored as T).  The arithmetic is
// float64 in both modes: C' = C - K H C cancels two to three digits when a precise hit meets a loose
// prediction, and the update is < 2 % of the work, so it is not worth a float32 error budget.
template <typename T>
CKF_HD void kalman_update(const double x[6], const T C[21], T m0, T m1, T v0, T v1, double xo[6], T Co[21]) {
  const double r0 = (double)m0 - x[0], r1 = (double)m1 - x[1];
  const double S00 = (double)C[tri(0, 0)] + (double)v0, S01 = (double)C[tri(0, 1)], S11 = (double)C[tri(1, 1)] + (double)v1;
  const double det = S00 * S11 - S01 * S01;
  const double I00 = S11 / det, I01 = -S01 / det, I11 = S00 / det;
  double K0[6], K1[6];
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    K0[i] = (double)C[tri(i, 0)] * I00 + (double)C[tri(i, 1)] * I01;
    K1[i] = (double)C[tri(i, 0)] * I01 + (double)C[tri(i, 1)] * I11;
  }
#pragma unroll
  for (int i = 0; i < 6; ++i) xo[i] = x[i] + (K0[i] * r0 + K1[i] * r1);
#pragma unroll
  for (int i = 0; i < 6; ++i)
#pragma unroll
    for (int j = i; j < 6; ++j)
      Co[tri(i, j)] = (T)((double)C[tri(i, j)] - (K0[i] * (double)C[tri(0, j)] + K1[i] * (double)C[tri(1, j)]));
  while (xo[2] > PI_D) xo[2] -= 2.0 * PI_D;
  while (xo[2] <= -PI_D) xo[2] += 2.0 * PI_D;
}

// ------------------------------------------------------------------------------------------ one move (step A)
// From bound x on module `from` to the next module: N2-N5 with P and J.  Outputs the target module, the
// predicted bound parameters, the 5x5 Jacobian block and the Highland variances to add to C[phi][phi],
// C[theta][theta] before transport (V5, applied on leaving).  Work counters in sc.
template <typename T>
CKF_HD int move_to_next_module(const GeoDev& g, const FieldDev& fld, const CfgDev& cfg, int from, const double x[6],
                               int& target, double xp[6], T J[5][5], T& q_phi, T& q_theta, StepCtl& sc) {
#pragma unroll
  for (int i = 0; i < 6; ++i)
    if (!isfinite(x[i])) return STOP_NUMERIC;
  if (!(x[3] > 0.0 && x[3] < PI_D)) return STOP_NUMERIC;
  Traj y;
  Jac<T> D;
  T dep_d[3];
  double dep_u[3], dep_v[3];
  int layer, iphi, iz;
  {
    const ModuleRec& m = g.mod[from];
    double sp, cp, st, ct;
    sincos(x[2], &sp, &cp);
    sincos(x[3], &st, &ct);
    y.d[0] = st * cp; y.d[1] = st * sp; y.d[2] = ct;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      y.r[i] = m.c[i] + x[0] * m.u[i] + x[1] * m.v[i];
      dep_u[i] = m.u[i];
      dep_v[i] = m.v[i];
      dep_d[i] = (T)y.d[i];
    }
    y.t = x[5];
    y.qop = x[4];
    layer = m.layer;
    iphi = m.iphi;
    iz = from - g.layer[layer].offset - iphi * g.layer[layer].n_z;
    if (m.xx0 > 0.0) {
      const double th2 = highland_theta0_sq(m.xx0, fabs(dot3(y.d, m.n)), y.qop, cfg.mass);
      q_theta = (T)th2;
      q_phi = (T)(th2 / (st * st));
    } else {
      q_theta = T(0);
      q_phi = T(0);
    }
  }
  jac_identity(D);
  sc.h_ctrl = cfg.h_max;
  sc.n_steps = 0;
  // N2: overlap neighbour on the same layer
  int tgt = pick_in_neighbourhood(g, layer, iphi, iz, from, y.r, y.d, 1e-3);
  if (tgt < 0) {
    // N3 + N4: next layer's cylinder, module choice at the portal; a crack is not a hole
    int lp = layer + 1;
    for (;;) {
      if (lp >= g.n_layers) return STOP_EXIT;
      const LayerRec L = g.layer[lp];
      Target cyl;
      cyl.kind = 1;
      cyl.R = L.r;
      const int st = propagate_to(fld, cfg, cyl, y, D, sc);
      if (st != STOP_NONE) return st;
      if (fabs(y.r[2]) > L.half_z) { ++lp; continue; }
      const double phix = atan2(y.r[1], y.r[0]);
      int i = (int)nearbyint(phix * L.n_phi / (2.0 * PI_D));
      i = ((i % L.n_phi) + L.n_phi) % L.n_phi;
      int j = (int)floor((y.r[2] + L.half_z) / L.len_z);
      j = j < 0 ? 0 : (j > L.n_z - 1 ? L.n_z - 1 : j);
      tgt = pick_in_neighbourhood(g, lp, i, j, -1, y.r, y.d, -1e-3);
      if (tgt >= 0) break;
      ++lp;
    }
  }
  // N5: to the target's plane, then J4 / J5
  const ModuleRec& k = g.mod[tgt];
  {
    Target pl;
    pl.kind = 0;
#pragma unroll
    for (int i = 0; i < 3; ++i) { pl.c[i] = k.c[i]; pl.n[i] = k.n[i]; }
    const int st = propagate_to(fld, cfg, pl, y, D, sc);
    if (st != STOP_NONE) return st;
  }
  double B[3];
  field_at(fld, y.r, B);
  arrival_jacobian(D, dep_u, dep_v, dep_d, k, y, B, cfg.mass, J);
  const double rel[3] = {y.r[0] - k.c[0], y.r[1] - k.c[1], y.r[2] - k.c[2]};
  xp[0] = dot3(rel, k.u);
  xp[1] = dot3(rel, k.v);
  xp[2] = atan2(y.d[1], y.d[0]);
  xp[3] = atan2(sqrt(y.d[0] * y.d[0] + y.d[1] * y.d[1]), y.d[2]);
  xp[4] = y.qop;
  xp[5] = y.t;
#pragma unroll
  for (int i = 0; i < 6; ++i)
    if (!isfinite(xp[i])) return STOP_NUMERIC;
  target = tgt;
  return STOP_NONE;
}

}  // namespace ckf
