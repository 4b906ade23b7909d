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

// kind 0: barrel cylinder of radius r, acceptance |z| <= half_z, modules on a (phi, z) grid of pitch len_z.
// kind 1 (row f3): disc in the plane z = half_z (signed), acceptance r_min <= rho <= r, modules on a (phi, ring)
// grid of ring pitch len_z, n_z rings; next_disc = the next disc of the same side (larger |z|) or -1.
// r_in (barrel): hypot(r, half_u), the outer envelope of the layer's flat modules = its portal for INWARD-moving tips.
struct LayerRec {
  double r, half_z, len_z, r_min, r_in;
  int32_t n_phi, n_z, offset, kind, next_disc, pad;
};

// a2 field store: uniform, or the float32 grid [ix][iy][iz] stored as (node, z-neighbour) pairs of 8 float32 (one
// 32-byte sector, one 256-bit load: ld_pair below) and widened to float64 in registers; the widening is exact, so the
// trilinear read returns the same float64 value as from a float64 copy of the grid.
struct FieldDev {
  int32_t kind;
  int32_t n[3];
  double ub[3];
  double org[3];
  double inv[3];  // 1 / spacing
  double nm2[3];  // (double)(n - 2): largest cell index
  const float* grid;   // [n0 * n1 * n2][8] float32: node (i, j, k) then node (i, j, k + 1), each (Bx, By, Bz, pad)
};

struct CfgDev {
  double chi2_max;
  double rk_tol, surf_tol, h_max, mass;
  int32_t max_branches, max_cands, max_holes, min_meas, max_rk_steps, max_levels;
  int32_t energy_loss;   // rule E: mean energy loss in every crossed module (BASELINE configs: 0)
  int32_t field_gradient;  // J2': field-gradient terms in the transport Jacobian (reading A13; BASELINE configs: 0)
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

struct D3 { double x, y, z; };
// One grid entry = the nodes (i, j, k) and (i, j, k + 1) as 8 float32 in a 32-byte sector: ONE 256-bit load
// (sm_100a: LDG.E.256) brings the two z-neighbours of a cell corner, so a cell is 4 loads.  The interpolation itself is
// float64 on the widened values -- the grid arrives as float32 (ckf_field.grid), widening is exact, so the result is
// the same as from a float64 copy of the grid.  History (profiles/r02_step_visit_update.md): the field read is the
// busiest user of the L1 data pipe in ckf_step, and what that pipe counts is load instructions x scattered lanes
// (wavefronts), not bytes: 16 loads of 128 + 64 bit per cell, then 8 of 256 bit (one node each), now 4.
// The asm is NOT volatile (that costs ckf_step 4 %): to the compiler it is a pure function of p, which it may hoist
// above the field-kind test of field_at -- it did in ckf_seed.  Hence every address field_at can form is readable: the
// index clamps keep it inside the grid, and a uniform field owns a 2 x 2 x 2 grid of its value (ckf_create).
CKF_HD void ld_pair(const float* p, D3& lo, D3& hi) {
#if defined(__CUDA_ARCH__)
  unsigned long long a, b, c, d;
  asm("ld.global.nc.v4.b64 {%0,%1,%2,%3}, [%4];" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p));
  lo.x = (double)__uint_as_float((unsigned)a); lo.y = (double)__uint_as_float((unsigned)(a >> 32));
  lo.z = (double)__uint_as_float((unsigned)b);
  hi.x = (double)__uint_as_float((unsigned)c); hi.y = (double)__uint_as_float((unsigned)(c >> 32));
  hi.z = (double)__uint_as_float((unsigned)d);
#else
  lo = D3{(double)p[0], (double)p[1], (double)p[2]};
  hi = D3{(double)p[4], (double)p[5], (double)p[6]};
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
    // i = clamp(floor(g), 0, n - 2) and fr = g - i with float64 adds only (no float<->int conversion
    // instructions): adding 1.5 * 2^52 rounds g to the nearest integer and leaves that integer in the low
    // mantissa bits.  Out-of-range g falls to the clamps.
    const double MAGIC = 6755399441055744.0;
    double ti = (g + MAGIC) - MAGIC;
    if (ti > g) ti -= 1.0;
    ti = ti < 0.0 ? 0.0 : ti;
    ti = ti > f.nm2[a] ? f.nm2[a] : ti;
#if defined(__CUDA_ARCH__)
    int i = __double2loint(ti + MAGIC);
#else
    int i = (ti == ti) ? (int)ti : 0;
#endif
    i = i < 0 ? 0 : i;                      // only a NaN position gets here out of range: keep the loads in bounds,
    i = i > f.n[a] - 2 ? f.n[a] - 2 : i;    // fr is NaN and the trial ends as STOP_NUMERIC
    idx[a] = i;
    fr[a] = g - ti;
  }
  const long long s1 = f.n[2], s0 = (long long)f.n[1] * f.n[2];
  const float* p = f.grid + 8 * (idx[0] * s0 + idx[1] * s1 + idx[2]);
  D3 v000, v001, v010, v011, v100, v101, v110, v111;
  ld_pair(p, v000, v001);
  ld_pair(p + 8 * s1, v010, v011);
  ld_pair(p + 8 * s0, v100, v101);
  ld_pair(p + 8 * (s0 + s1), v110, v111);
#define CKF_TRILERP(C)                                              \
  {                                                                 \
    const double x00 = v000.C + fr[0] * (v100.C - v000.C);          \
    const double x10 = v010.C + fr[0] * (v110.C - v010.C);          \
    const double x01 = v001.C + fr[0] * (v101.C - v001.C);          \
    const double x11 = v011.C + fr[0] * (v111.C - v011.C);          \
    const double y0 = x00 + fr[1] * (x10 - x00);                    \
    const double y1 = x01 + fr[1] * (x11 - x01);                    \
    out = y0 + fr[2] * (y1 - y0);                                   \
  }
  double out;
  CKF_TRILERP(x) B[0] = out;
  CKF_TRILERP(y) B[1] = out;
  CKF_TRILERP(z) B[2] = out;
#undef CKF_TRILERP
}

// J2' (config.field_gradient): G[i][j] = dB_i / dr_j, the exact derivative of the trilinear interpolant inside the cell
// field_at picks for r (piecewise constant along the differentiated axis); zero for a uniform field.
CKF_HD void field_gradient_at(const FieldDev& f, const double r[3], double G[3][3]) {
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) G[i][j] = 0.0;
  if (f.kind == 0) return;
  int idx[3];
  double fr[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double g = (r[a] - f.org[a]) * f.inv[a];
    double ti = floor(g);
    ti = ti < 0.0 ? 0.0 : ti;
    ti = ti > f.nm2[a] ? f.nm2[a] : ti;
    int i = (ti == ti) ? (int)ti : 0;
    i = i < 0 ? 0 : i;
    i = i > f.n[a] - 2 ? f.n[a] - 2 : i;
    idx[a] = i;
    fr[a] = g - ti;
  }
  const long long s1 = f.n[2], s0 = (long long)f.n[1] * f.n[2];
  const float* p = f.grid + 8 * (idx[0] * s0 + idx[1] * s1 + idx[2]);
  D3 v000, v001, v010, v011, v100, v101, v110, v111;
  ld_pair(p, v000, v001);
  ld_pair(p + 8 * s1, v010, v011);
  ld_pair(p + 8 * s0, v100, v101);
  ld_pair(p + 8 * (s0 + s1), v110, v111);
#define CKF_TRIGRAD(C, ROW)                                                                         \
  {                                                                                                 \
    /* d/dx: differences along x, then lerp along y and z */                                        \
    const double dx0 = (v100.C - v000.C) + fr[1] * ((v110.C - v010.C) - (v100.C - v000.C));         \
    const double dx1 = (v101.C - v001.C) + fr[1] * ((v111.C - v011.C) - (v101.C - v001.C));         \
    G[ROW][0] = (dx0 + fr[2] * (dx1 - dx0)) * f.inv[0];                                             \
    /* d/dy: lerp along x, difference along y, lerp along z */                                      \
    const double x00 = v000.C + fr[0] * (v100.C - v000.C), x10 = v010.C + fr[0] * (v110.C - v010.C); \
    const double x01 = v001.C + fr[0] * (v101.C - v001.C), x11 = v011.C + fr[0] * (v111.C - v011.C); \
    const double dy0 = x10 - x00, dy1 = x11 - x01;                                                  \
    G[ROW][1] = (dy0 + fr[2] * (dy1 - dy0)) * f.inv[1];                                             \
    /* d/dz: lerp along x and y, difference along z */                                              \
    const double y0 = x00 + fr[1] * (x10 - x00), y1 = x01 + fr[1] * (x11 - x01);                    \
    G[ROW][2] = (y1 - y0) * f.inv[2];                                                               \
  }
  CKF_TRIGRAD(x, 0)
  CKF_TRIGRAD(y, 1)
  CKF_TRIGRAD(z, 2)
#undef CKF_TRIGRAD
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

// J2': with the field-gradient terms the position columns of D are no longer trivial.  A move only needs them along
// the two local axes of its departure module (r0 = c + l0 u + l1 v): two tangent vectors (dr, dd), started at
// (u, 0) and (v, 0).  Without the gradient terms they stay there, which is what arrival_jacobian assumes by default.
template <typename T>
struct JacR {
  T Ru[3], Du[3], Rv[3], Dv[3];
};

template <typename T>
CKF_HD void jacr_begin(JacR<T>& R, const double u[3], const double v[3]) {
#pragma unroll
  for (int i = 0; i < 3; ++i) { R.Ru[i] = (T)u[i]; R.Rv[i] = (T)v[i]; R.Du[i] = T(0); R.Dv[i] = T(0); }
}

CKF_HD double inv_beta(double qop, double mass) { return sqrt(1.0 + mass * mass * qop * qop); }
CKF_HD double dinvbeta_dqop(double qop, double mass) { return mass * mass * qop / sqrt(1.0 + mass * mass * qop * qop); }

// One RKN4 trial (P2, P3).  What survives the trial is only what an accepted step needs, in the type it needs
// it in (keeps the live register set of the hot loop small): the three field values and the four
// q/p-derivative vectors kappa * cr_i as T for the Jacobian columns, the two stage sums
// s1 = k1 + k2 + k3, s2 = k1 + 2 k2 + 2 k3 + k4 (k_i = lam * cr_i) for the state, and the error estimate
// eps = h^2 |k1 - k2 - k3 + k4|.
template <typename T>
struct Trial {
  T B1[3], B2[3], B4[3];
  T q1[3], q2[3], q3[3], q4[3];
  double s1[3], s2[3];
  double eps;
  double rm[3], re[3];  // stage points, kept only by rk_trial<T, true> (J2' reads the field gradient there)
};

// B1 = field at y.r, read by the caller (move_target): it is the same for every retry of a rejected trial, and after an
// accepted step its loads are issued before the Jacobian columns are computed, which hides their latency.
template <typename T, bool GRAD = false>
CKF_HD void rk_trial(const FieldDev& fld, const Traj& y, const double B1[3], double lam, double h, Trial<T>& t) {
  // The stage loop is unrolled: three inlined copies of field_at.  In the monolithic level loop of r01b one rolled
  // copy was needed to stay inside the SM's instruction cache; in the per-phase ckf_step the three copies fit
  // (2,640 SASS instructions) and save the register moves of the rolled form: ckf_step 2.07 -> 1.89 ms per event.
  const double h2 = 0.5 * h, h8 = h * h * 0.125, hh2 = h * h * 0.5;
  double cr1[3], cr2[3], cr3[3], cr4[3];
#pragma unroll
  for (int st = 0; st < 3; ++st) {
    double p[3], B[3], w[3];
    if (st == 0) {
#pragma unroll
      for (int i = 0; i < 3; ++i) B[i] = B1[i];
    } else if (st == 1) {
#pragma unroll
      for (int i = 0; i < 3; ++i) p[i] = y.r[i] + h2 * y.d[i] + h8 * (lam * cr1[i]);
    } else {
#pragma unroll
      for (int i = 0; i < 3; ++i) p[i] = y.r[i] + h * y.d[i] + hh2 * (lam * cr3[i]);
    }
    if (GRAD && st != 0) {
#pragma unroll
      for (int i = 0; i < 3; ++i) (st == 1 ? t.rm : t.re)[i] = p[i];
    }
    if (st != 0) field_at(fld, p, B);
    if (st == 0) {
#pragma unroll
      for (int i = 0; i < 3; ++i) t.B1[i] = (T)B[i];
      cross3(y.d, B, cr1);
    } else if (st == 1) {
#pragma unroll
      for (int i = 0; i < 3; ++i) { t.B2[i] = (T)B[i]; w[i] = y.d[i] + h2 * (lam * cr1[i]); }
      cross3(w, B, cr2);
#pragma unroll
      for (int i = 0; i < 3; ++i) w[i] = y.d[i] + h2 * (lam * cr2[i]);
      cross3(w, B, cr3);
    } else {
#pragma unroll
      for (int i = 0; i < 3; ++i) { t.B4[i] = (T)B[i]; w[i] = y.d[i] + h * (lam * cr3[i]); }
      cross3(w, B, cr4);
    }
  }
  double e2 = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    const double k1 = lam * cr1[i], k2 = lam * cr2[i], k3 = lam * cr3[i], k4 = lam * cr4[i];
    const double e = k1 - k2 - k3 + k4;
    e2 += e * e;
    t.s1[i] = k1 + k2 + k3;
    t.s2[i] = k1 + 2.0 * k2 + 2.0 * k3 + k4;
    t.q1[i] = (T)(KAPPA * cr1[i]); t.q2[i] = (T)(KAPPA * cr2[i]);
    t.q3[i] = (T)(KAPPA * cr3[i]); t.q4[i] = (T)(KAPPA * cr4[i]);
  }
  t.eps = h * h * sqrt(e2);
}

// J2 applied to one column (dr, dd) of the running Jacobian: the linearised RKN4 step with h fixed and the
// field gradient neglected.  qf = 1 adds the explicit q/p dependence kappa * cr_i (the q-column), qf = 0 does
// not (adding qf * q = +0 leaves the d-columns' values unchanged).
template <typename T>
CKF_HD void jac_column_q(T lam, T h, T qf, const T B1[3], const T B2[3], const T B4[3], const T q1[3], const T q2[3],
                         const T q3[3], const T q4[3], T dr[3], T dd[3]) {
  T k1[3], k2[3], k3[3], k4[3], w[3];
  const T h2 = T(0.5) * h;
  cross3(dd, B1, k1);
#pragma unroll
  for (int i = 0; i < 3; ++i) k1[i] = lam * k1[i] + qf * q1[i];
#pragma unroll
  for (int i = 0; i < 3; ++i) w[i] = dd[i] + h2 * k1[i];
  cross3(w, B2, k2);
#pragma unroll
  for (int i = 0; i < 3; ++i) k2[i] = lam * k2[i] + qf * q2[i];
#pragma unroll
  for (int i = 0; i < 3; ++i) w[i] = dd[i] + h2 * k2[i];
  cross3(w, B2, k3);
#pragma unroll
  for (int i = 0; i < 3; ++i) k3[i] = lam * k3[i] + qf * q3[i];
#pragma unroll
  for (int i = 0; i < 3; ++i) w[i] = dd[i] + h * k3[i];
  cross3(w, B4, k4);
#pragma unroll
  for (int i = 0; i < 3; ++i) k4[i] = lam * k4[i] + qf * q4[i];
  const T h6 = h * T(1.0 / 6.0), hh6 = h * h * T(1.0 / 6.0);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    dr[i] = dr[i] + h * dd[i] + hh6 * (k1[i] + k2[i] + k3[i]);
    dd[i] = dd[i] + h6 * (k1[i] + T(2) * k2[i] + T(2) * k3[i] + k4[i]);
  }
}

// J2' applied to one column: jac_column_q plus the dependence of the field on the stage points,
//   k1 = lam [dd x B1 + w1 x (G1 dr)] + qf q1,          drm = dr + h/2 dd + h^2/8 k1
//   k2 = lam [(dd + h/2 k1) x B2 + w2 x (G2 drm)] + qf q2,   k3 likewise from k2 with w3
//   dre = dr + h dd + h^2/2 k3,    k4 = lam [(dd + h k3) x B4 + w4 x (G4 dre)] + qf q4
// w1 = d, w2 = d + h/2 k1, w3 = d + h/2 k2, w4 = d + h k3 of the trajectory itself (StepGrad).
template <typename T>
struct StepGrad {
  T G1[3][3], G2[3][3], G4[3][3];
  T w1[3], w2[3], w3[3], w4[3];
};

// Gradients at the three stage points and the stage directions of an accepted trial; y is the state BEFORE the step.
template <typename T>
CKF_HD void step_gradients(const FieldDev& fld, const Traj& y, double h, const Trial<T>& t, StepGrad<T>& sg) {
  double G[3][3];
  field_gradient_at(fld, y.r, G);
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) sg.G1[i][j] = (T)G[i][j];
  field_gradient_at(fld, t.rm, G);
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) sg.G2[i][j] = (T)G[i][j];
  field_gradient_at(fld, t.re, G);
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) sg.G4[i][j] = (T)G[i][j];
  // k_i = lam cr_i = q/p * (kappa cr_i) = q/p * q_i
  const double h2 = 0.5 * h;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    sg.w1[i] = (T)y.d[i];
    sg.w2[i] = (T)(y.d[i] + h2 * (y.qop * (double)t.q1[i]));
    sg.w3[i] = (T)(y.d[i] + h2 * (y.qop * (double)t.q2[i]));
    sg.w4[i] = (T)(y.d[i] + h * (y.qop * (double)t.q3[i]));
  }
}

template <typename T>
CKF_HD void jac_column_g(T lam, T h, T qf, const Trial<T>& t, const StepGrad<T>& sg, T dr[3], T dd[3]) {
  T k1[3], k2[3], k3[3], k4[3], w[3], gb[3], b[3], drs[3];
  const T h2 = T(0.5) * h, h8 = h * h * T(0.125), hh2 = h * h * T(0.5);
  auto gmul = [](const T G[3][3], const T v[3], T o[3]) {
#pragma unroll
    for (int i = 0; i < 3; ++i) o[i] = G[i][0] * v[0] + G[i][1] * v[1] + G[i][2] * v[2];
  };
  cross3(dd, t.B1, k1);
  gmul(sg.G1, dr, gb);
  cross3(sg.w1, gb, b);
#pragma unroll
  for (int i = 0; i < 3; ++i) k1[i] = lam * (k1[i] + b[i]) + qf * t.q1[i];
#pragma unroll
  for (int i = 0; i < 3; ++i) drs[i] = dr[i] + h2 * dd[i] + h8 * k1[i];
  gmul(sg.G2, drs, gb);
#pragma unroll
  for (int i = 0; i < 3; ++i) w[i] = dd[i] + h2 * k1[i];
  cross3(w, t.B2, k2);
  cross3(sg.w2, gb, b);
#pragma unroll
  for (int i = 0; i < 3; ++i) k2[i] = lam * (k2[i] + b[i]) + qf * t.q2[i];
#pragma unroll
  for (int i = 0; i < 3; ++i) w[i] = dd[i] + h2 * k2[i];
  cross3(w, t.B2, k3);
  cross3(sg.w3, gb, b);
#pragma unroll
  for (int i = 0; i < 3; ++i) k3[i] = lam * (k3[i] + b[i]) + qf * t.q3[i];
#pragma unroll
  for (int i = 0; i < 3; ++i) drs[i] = dr[i] + h * dd[i] + hh2 * k3[i];
  gmul(sg.G4, drs, gb);
#pragma unroll
  for (int i = 0; i < 3; ++i) w[i] = dd[i] + h * k3[i];
  cross3(w, t.B4, k4);
  cross3(sg.w4, gb, b);
#pragma unroll
  for (int i = 0; i < 3; ++i) k4[i] = lam * (k4[i] + b[i]) + qf * t.q4[i];
  const T h6 = h * T(1.0 / 6.0), hh6 = h * h * T(1.0 / 6.0);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    dr[i] = dr[i] + h * dd[i] + hh6 * (k1[i] + k2[i] + k3[i]);
    dd[i] = dd[i] + h6 * (k1[i] + T(2) * k2[i] + T(2) * k3[i] + k4[i]);
  }
}

// D <- D_step D with the gradient terms: the three d-columns, the q-column and the two position columns.
template <typename T>
CKF_HD void rk_accept_jac_g(double qop, Jac<T>& J, JacR<T>& R, double h, const Trial<T>& t, const StepGrad<T>& sg, double dib) {
  const T lamT = (T)(KAPPA * qop), hT = (T)h;
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    T dr[3] = {J.Rd[0][j], J.Rd[1][j], J.Rd[2][j]};
    T dd[3] = {J.Dd[0][j], J.Dd[1][j], J.Dd[2][j]};
    jac_column_g<T>(lamT, hT, T(0), t, sg, dr, dd);
#pragma unroll
    for (int i = 0; i < 3; ++i) { J.Rd[i][j] = dr[i]; J.Dd[i][j] = dd[i]; }
  }
  jac_column_g<T>(lamT, hT, T(1), t, sg, J.rq, J.dq);
  jac_column_g<T>(lamT, hT, T(0), t, sg, R.Ru, R.Du);
  jac_column_g<T>(lamT, hT, T(0), t, sg, R.Rv, R.Dv);
  J.tq += (T)(h * dib);
}

// Accept a trial, in two halves so that the caller can put the next field read between them: the state (P2), and
// D <- D_step D column by column (J2, J3).  The Jacobian half does not read the state's position or direction.
template <typename T>
CKF_HD void rk_accept_jac(const Traj& y, Jac<T>& J, double h, const Trial<T>& t, double dib) {
  {
    const T lamT = (T)(KAPPA * y.qop), hT = (T)h;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      T dr[3] = {J.Rd[0][j], J.Rd[1][j], J.Rd[2][j]};
      T dd[3] = {J.Dd[0][j], J.Dd[1][j], J.Dd[2][j]};
      jac_column_q<T>(lamT, hT, T(0), t.B1, t.B2, t.B4, t.q1, t.q2, t.q3, t.q4, dr, dd);
#pragma unroll
      for (int i = 0; i < 3; ++i) { J.Rd[i][j] = dr[i]; J.Dd[i][j] = dd[i]; }
    }
    jac_column_q<T>(lamT, hT, T(1), t.B1, t.B2, t.B4, t.q1, t.q2, t.q3, t.q4, J.rq, J.dq);
    J.tq += (T)(h * dib);
  }
}
template <typename T>
CKF_HD void rk_accept_state(Traj& y, double h, const Trial<T>& t, double ib) {
  const double h6 = h * (1.0 / 6.0), hh6 = h * h * (1.0 / 6.0);  // one rounding away from h / 6: far inside 1e-9
  double dn[3], n2 = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    y.r[i] = y.r[i] + h * y.d[i] + hh6 * t.s1[i];
    dn[i] = y.d[i] + h6 * t.s2[i];
    n2 += dn[i] * dn[i];
  }
  const double inrm = 1.0 / sqrt(n2);
#pragma unroll
  for (int i = 0; i < 3; ++i) y.d[i] = dn[i] * inrm;
  y.t += h * ib;
}

// P5: field-free closing step of length s.
template <typename T>
CKF_HD void straight_close(Traj& y, Jac<T>& J, double s, double ib, double dib) {
  const T sT = (T)s;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
#pragma unroll
    for (int j = 0; j < 3; ++j) J.Rd[i][j] += sT * J.Dd[i][j];
    J.rq[i] += sT * J.dq[i];
    y.r[i] += s * y.d[i];
  }
  J.tq += (T)(s * dib);
  y.t += s * ib;
}

template <typename T>
CKF_HD void straight_close_r(JacR<T>& R, double s) {
  const T sT = (T)s;
#pragma unroll
  for (int i = 0; i < 3; ++i) { R.Ru[i] += sT * R.Du[i]; R.Rv[i] += sT * R.Dv[i]; }
}

// ------------------------------------------------------------------------------------------ step control
struct StepCtl {
  double h_ctrl;
  int n_steps;
  int n_trials, n_accepted;  // work counters
};

}  // namespace ckf
