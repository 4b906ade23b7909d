// ckf_math.cuh — per-tip arithmetic of the CKF hot path (sm_100a), written from DESIGN.md §3.
//
// Everything here is register-resident, per-thread code: field read (F), RKN4 trial + block-sparse
// transport-Jacobian columns (P2, P3, J2, J3), targeting and landing (P4-P6), navigation over the
// per-layer phi/z grid (N2-N4), arrival Jacobian and covariance transport (J4, J5), Highland noise (V5),
// chi2 (V1) and the gain-form update (V3).
//
// Precision split: the trajectory (r, d, t, q/p, bound parameter vector) is always
// float64; `T` (float or double) is the type of the transport Jacobian, the covariance, the gain and chi2.
//
// The functions are __host__ __device__ so that tests/host_math_check.cu can run exactly this source on
// the CPU against the oracle; the product library only ever calls them from kernels.
#pragma once
#include <cmath>
#include <cstdint>

#if defined(__CUDACC__)
#define CKF_HD __host__ __device__ __forceinline__
#else
#define CKF_HD inline
#endif

namespace ckf {

constexpr double KAPPA = 2.99792458e-4;  // GeV / (T mm)
constexpr double PI_D = 3.14159265358979323846;

enum Stop : int { STOP_NONE = 0, STOP_EXIT = 1, STOP_HOLES = 2, STOP_NOT_OUTGOING = 3, STOP_STEP_LIMIT = 4,
                  STOP_NUMERIC = 5, STOP_LEVEL_LIMIT = 6 };

// ------------------------------------------------------------------------------------------ device stores
// a1 geometry store: one 128-byte record per module (one L2 line), one small record per layer.
struct alignas(128) ModuleRec {
  double c[3], u[3], v[3], n[3];
  double half_u, half_v, xx0;
  int32_t layer, iphi;
};
static_assert(sizeof(ModuleRec) == 128, "ModuleRec must be one 128-byte line");

struct LayerRec {
  double r, half_z, len_z;
  int32_t n_phi, n_z, offset, pad;
};

// a2 field store: uniform, or float4-padded copy of the float32 grid [ix][iy][iz] (w unused).
struct FieldDev {
  int32_t kind;
  int32_t n[3];
  double ub[3];
  double org[3];
  double inv[3];  // 1 / spacing
  const float4* grid;
};

struct CfgDev {
  double chi2_max;
  double rk_tol, surf_tol, h_max, mass;
  int32_t max_branches, max_cands, max_holes, min_meas, max_rk_steps, max_levels;
};

// ------------------------------------------------------------------------------------------ small algebra
template <typename A, typename B, typename C>
CKF_HD void cross3(const A a[3], const B b[3], C o[3]) {
  o[0] = a[1] * b[2] - a[2] * b[1];
  o[1] = a[2] * b[0] - a[0] * b[2];
  o[2] = a[0] * b[1] - a[1] * b[0];
}
template <typename A, typename B>
CKF_HD auto dot3(const A a[3], const B b[3]) -> decltype(a[0] * b[0]) {
  return a[0] * b[0] + a[1] * b[1] + a[2] * b[2];
}

CKF_HD float4 ldg4(const float4* p) {
#if defined(__CUDA_ARCH__)
  return __ldg(p);
#else
  return *p;
#endif
}

// ------------------------------------------------------------------------------------------ F: field read
// Trilinear, lerp along x then y then z, each as a + f (b - a); edge cells extrapolate.
CKF_HD void field_at(const FieldDev& f, const double r[3], double B[3]) {
  if (f.kind == 0) {
    B[0] = f.ub[0]; B[1] = f.ub[1]; B[2] = f.ub[2];
    return;
  }
  int idx[3];
  double fr[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double g = (r[a] - f.org[a]) * f.inv[a];
    int i = (int)floor(g);
    i = i < 0 ? 0 : i;
    i = i > f.n[a] - 2 ? f.n[a] - 2 : i;
    idx[a] = i;
    fr[a] = g - (double)i;
  }
  const long long s1 = f.n[2], s0 = (long long)f.n[1] * f.n[2];
  const float4* p = f.grid + idx[0] * s0 + idx[1] * s1 + idx[2];
  const float4 v000 = ldg4(p), v001 = ldg4(p + 1);
  const float4 v010 = ldg4(p + s1), v011 = ldg4(p + s1 + 1);
  const float4 v100 = ldg4(p + s0), v101 = ldg4(p + s0 + 1);
  const float4 v110 = ldg4(p + s0 + s1), v111 = ldg4(p + s0 + s1 + 1);
#define CKF_TRILERP(C)                                                                     \
  {                                                                                        \
    const double x00 = (double)v000.C + fr[0] * ((double)v100.C - (double)v000.C);         \
    const double x10 = (double)v010.C + fr[0] * ((double)v110.C - (double)v010.C);         \
    const double x01 = (double)v001.C + fr[0] * ((double)v101.C - (double)v001.C);         \
    const double x11 = (double)v011.C + fr[0] * ((double)v111.C - (double)v011.C);         \
    const double y0 = x00 + fr[1] * (x10 - x00);                                           \
    const double y1 = x01 + fr[1] * (x11 - x01);                                           \
    out = y0 + fr[2] * (y1 - y0);                                                          \
  }
  double out;
  CKF_TRILERP(x) B[0] = out;
  CKF_TRILERP(y) B[1] = out;
  CKF_TRILERP(z) B[2] = out;
#undef CKF_TRILERP
}

// ------------------------------------------------------------------------------------------ trajectory state
struct Traj {
  double r[3], d[3], t, qop;
};

// Block-sparse running transport Jacobian D = d(r,t,d,q/p)/d(r0,t0,d0,q/p0) (J3): only the d- and q-columns
// are non-trivial: Rd = dr/dd0, Dd = dd/dd0, rq = dr/dq, dq = dd/dq, tq = dt/dq.  25 numbers.
template <typename T>
struct Jac {
  T Rd[3][3], Dd[3][3], rq[3], dq[3], tq;
};

template <typename T>
CKF_HD void jac_identity(Jac<T>& J) {
#pragma unroll
  for (int i = 0; i < 3; ++i) {
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      J.Rd[i][j] = T(0);
      J.Dd[i][j] = (i == j) ? T(1) : T(0);
    }
    J.rq[i] = T(0);
    J.dq[i] = T(0);
  }
  J.tq = T(0);
}

CKF_HD double inv_beta(double qop, double mass) { return sqrt(1.0 + mass * mass * qop * qop); }
CKF_HD double dinvbeta_dqop(double qop, double mass) { return mass * mass * qop / sqrt(1.0 + mass * mass * qop * qop); }

// One RKN4 trial (P2): the four stage cross products cr_i (k_i = lam * cr_i), the three field values and the
// error estimate eps = h^2 |k1 - k2 - k3 + k4| (P3).
struct Trial {
  double cr1[3], cr2[3], cr3[3], cr4[3];
  double B1[3], B2[3], B4[3];
  double eps;
};

CKF_HD void rk_trial(const FieldDev& fld, const Traj& y, double lam, double h, Trial& t) {
  double w[3], p[3];
  field_at(fld, y.r, t.B1);
  cross3(y.d, t.B1, t.cr1);
  const double h2 = 0.5 * h, h8 = h * h * 0.125;
#pragma unroll
  for (int i = 0; i < 3; ++i) p[i] = y.r[i] + h2 * y.d[i] + h8 * (lam * t.cr1[i]);
  field_at(fld, p, t.B2);
#pragma unroll
  for (int i = 0; i < 3; ++i) w[i] = y.d[i] + h2 * (lam * t.cr1[i]);
  cross3(w, t.B2, t.cr2);
#pragma unroll
  for (int i = 0; i < 3; ++i) w[i] = y.d[i] + h2 * (lam * t.cr2[i]);
  cross3(w, t.B2, t.cr3);
  const double hh2 = h * h * 0.5;
#pragma unroll
  for (int i = 0; i < 3; ++i) p[i] = y.r[i] + h * y.d[i] + hh2 * (lam * t.cr3[i]);
  field_at(fld, p, t.B4);
#pragma unroll
  for (int i = 0; i < 3; ++i) w[i] = y.d[i] + h * (lam * t.cr3[i]);
  cross3(w, t.B4, t.cr4);
  double e2 = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    const double e = lam * t.cr1[i] - lam * t.cr2[i] - lam * t.cr3[i] + lam * t.cr4[i];
    e2 += e * e;
  }
  t.eps = h * h * sqrt(e2);
}

// J2 applied to one column (dr, dd) of the running Jacobian: the linearised RKN4 step with h fixed and the
// field gradient neglected.  WITH_Q adds the explicit q/p dependence kappa * cr_i (the q-column).
template <typename T, bool WITH_Q>
CKF_HD void jac_column(T lam, T h, const T B1[3], const T B2[3], const T B4[3], const T q1[3], const T q2[3],
                       const T q3[3], const T q4[3], T dr[3], T dd[3]) {
  T k1[3], k2[3], k3[3], k4[3], w[3];
  const T h2 = T(0.5) * h;
  cross3(dd, B1, k1);
#pragma unroll
  for (int i = 0; i < 3; ++i) k1[i] = WITH_Q ? lam * k1[i] + q1[i] : lam * k1[i];
#pragma unroll
  for (int i = 0; i < 3; ++i) w[i] = dd[i] + h2 * k1[i];
  cross3(w, B2, k2);
#pragma unroll
  for (int i = 0; i < 3; ++i) k2[i] = WITH_Q ? lam * k2[i] + q2[i] : lam * k2[i];
#pragma unroll
  for (int i = 0; i < 3; ++i) w[i] = dd[i] + h2 * k2[i];
  cross3(w, B2, k3);
#pragma unroll
  for (int i = 0; i < 3; ++i) k3[i] = WITH_Q ? lam * k3[i] + q3[i] : lam * k3[i];
#pragma unroll
  for (int i = 0; i < 3; ++i) w[i] = dd[i] + h * k3[i];
  cross3(w, B4, k4);
#pragma unroll
  for (int i = 0; i < 3; ++i) k4[i] = WITH_Q ? lam * k4[i] + q4[i] : lam * k4[i];
  const T h6 = h * T(1.0 / 6.0), hh6 = h * h * T(1.0 / 6.0);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    dr[i] = dr[i] + h * dd[i] + hh6 * (k1[i] + k2[i] + k3[i]);
    dd[i] = dd[i] + h6 * (k1[i] + T(2) * k2[i] + T(2) * k3[i] + k4[i]);
  }
}

// Accept a trial: D <- D_step D column by column (J2, J3), then the state (P2).
template <typename T>
CKF_HD void rk_accept(Traj& y, Jac<T>& J, double lam, double h, const Trial& t, double mass) {
  {
    T B1[3], B2[3], B4[3], q1[3], q2[3], q3[3], q4[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      B1[i] = (T)t.B1[i]; B2[i] = (T)t.B2[i]; B4[i] = (T)t.B4[i];
      q1[i] = (T)(KAPPA * t.cr1[i]); q2[i] = (T)(KAPPA * t.cr2[i]);
      q3[i] = (T)(KAPPA * t.cr3[i]); q4[i] = (T)(KAPPA * t.cr4[i]);
    }
    const T lamT = (T)lam, hT = (T)h;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      T dr[3] = {J.Rd[0][j], J.Rd[1][j], J.Rd[2][j]};
      T dd[3] = {J.Dd[0][j], J.Dd[1][j], J.Dd[2][j]};
      jac_column<T, false>(lamT, hT, B1, B2, B4, q1, q2, q3, q4, dr, dd);
#pragma unroll
      for (int i = 0; i < 3; ++i) { J.Rd[i][j] = dr[i]; J.Dd[i][j] = dd[i]; }
    }
    jac_column<T, true>(lamT, hT, B1, B2, B4, q1, q2, q3, q4, J.rq, J.dq);
    J.tq += (T)(h * dinvbeta_dqop(y.qop, mass));
  }
  const double h6 = h / 6.0, hh6 = h * h / 6.0;
  double dn[3], n2 = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    const double k1 = lam * t.cr1[i], k2 = lam * t.cr2[i], k3 = lam * t.cr3[i], k4 = lam * t.cr4[i];
    y.r[i] = y.r[i] + h * y.d[i] + hh6 * (k1 + k2 + k3);
    dn[i] = y.d[i] + h6 * (k1 + 2.0 * k2 + 2.0 * k3 + k4);
    n2 += dn[i] * dn[i];
  }
  const double nrm = sqrt(n2);
#pragma unroll
  for (int i = 0; i < 3; ++i) y.d[i] = dn[i] / nrm;
  y.t += h * inv_beta(y.qop, mass);
}

// P5: field-free closing step of length s.
template <typename T>
CKF_HD void straight_close(Traj& y, Jac<T>& J, double s, double mass) {
  const T sT = (T)s;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
#pragma unroll
    for (int j = 0; j < 3; ++j) J.Rd[i][j] += sT * J.Dd[i][j];
    J.rq[i] += sT * J.dq[i];
    y.r[i] += s * y.d[i];
  }
  J.tq += (T)(s * dinvbeta_dqop(y.qop, mass));
  y.t += s * inv_beta(y.qop, mass);
}

// ------------------------------------------------------------------------------------------ P4: targets
struct Target {
  int kind;  // 0 plane (c, n), 1 cylinder R
  double c[3], n[3], R;
};

CKF_HD bool target_distance(const Target& tg, const Traj& y, double& s, int& why) {
  if (tg.kind == 0) {
    const double dn = dot3(y.d, tg.n);
    if (!(fabs(dn) > 1e-12)) { why = STOP_NUMERIC; return false; }
    const double rel[3] = {tg.c[0] - y.r[0], tg.c[1] - y.r[1], tg.c[2] - y.r[2]};
    s = dot3(rel, tg.n) / dn;
    return true;
  }
  const double a = y.d[0] * y.d[0] + y.d[1] * y.d[1];
  const double b = y.r[0] * y.d[0] + y.r[1] * y.d[1];
  const double cc = y.r[0] * y.r[0] + y.r[1] * y.r[1] - tg.R * tg.R;
  const double disc = b * b - a * cc;
  if (!(b > 0.0) || !(disc >= 0.0)) { why = STOP_NOT_OUTGOING; return false; }
  s = -cc / (b + sqrt(disc));
  return true;
}

struct StepCtl {
  double h_ctrl;
  int n_steps;
  int n_trials, n_accepted;  // work counters
};

// P3-P6: adaptive stepping until the target is reached.
template <typename T>
CKF_HD int propagate_to(const FieldDev& fld, const CfgDev& cfg, const Target& tg, Traj& y, Jac<T>& J, StepCtl& sc) {
  const double lam = KAPPA * y.qop;
  for (;;) {
    double s;
    int why = STOP_NUMERIC;
    if (!target_distance(tg, y, s, why)) return why;
    if (!isfinite(s)) return STOP_NUMERIC;
    if (fabs(s) <= cfg.surf_tol) {
      straight_close(y, J, s, cfg.mass);
      return STOP_NONE;
    }
    const double hlim = fmin(sc.h_ctrl, cfg.h_max);
    double h = (fabs(s) <= hlim) ? s : (s > 0.0 ? hlim : -hlim);
    for (;;) {
      if (++sc.n_steps > cfg.max_rk_steps) return STOP_STEP_LIMIT;
      Trial t;
      rk_trial(fld, y, lam, h, t);
      ++sc.n_trials;
      if (!isfinite(t.eps)) return STOP_NUMERIC;
      double f;
      if (t.eps == 0.0) f = 4.0;
      else {
        f = 0.9 * sqrt(sqrt(cfg.rk_tol / t.eps));
        f = f < 0.25 ? 0.25 : f;
        f = f > 4.0 ? 4.0 : f;
      }
      if (t.eps <= cfg.rk_tol) {
        rk_accept(y, J, lam, h, t, cfg.mass);
        sc.h_ctrl = fabs(h) * f;
        ++sc.n_accepted;
        break;
      }
      h = h * f;
    }
  }
}

}  // namespace ckf
