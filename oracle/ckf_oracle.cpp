// ckf_oracle.cpp — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, double-precision CPU implementation of combinatorial-Kalman-filter (CKF) track
// finding, written from the paper (arxiv 2505.22822, §2) and the
// textbook mathematics of the works it cites (refs [7],[8],[12]-[18]), following the
// step-by-step rules of SURVEY.md §8(c) (U, G, F, P1-P6, J1-J5, N1-N6, V1-V5, R9-R11, T) in that
// order and notation.  One seed at a time, std::vector + loops, dense 8x8 / 6x6 algebra, no blocking,
// no SIMD, no code shared with the CUDA path (paper_2505_22822_b200/csrc/).  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -fPIC -shared -pthread (oracle/build.py).
//
// Pins (tests/test_oracle_pins.py): analytic helix (P2-P5), finite-difference Jacobian (J1-J5),
// closed-form scalar gain + information-form identity (V1-V3), Highland values (V5), multilinear field
// (F), brute-force module sequence (N2-N5), brute-force CKF enumeration on a toy (R9-R11).
// KF fit + RTS smoother (rules K, tests/test_oracle_fit.py): scalar random walk against its information-form
// closed form, the smoothed states of real tracks against a dense Gaussian conditioning of the linearised
// model (numpy), forward pass = the CKF candidate's reported state.
// Round-2 pins (tests/test_oracle_pins2.py): RKN4 stage points and field per stage in a NON-uniform field against
// an independent DOP853 integration (analytic map through the pin hook `field kind 2`, and the float32 grid through
// scipy's multilinear interpolator); the material path factor x/X0 / |d.n| for inclined tracks; the closed form of
// R10 against a literal one-child-at-a-time greedy (which children survive, with branches finishing at different
// levels); reading D11 against the literal N3 walk (pin hook oracle_set_n3_literal_walk): same candidates.
// Energy loss (rule E, tests/test_oracle_eloss.py): minimum of the Bethe curve against the PDG table value for silicon
// (golden file), non-relativistic limit, energy conservation, g against finite differences of the kinematics, the
// whole move's Jacobian against finite differences.  Field-gradient Jacobian (J2', tests/test_oracle_pins2.py): finite
// differences of the bound->bound map in the analytic non-uniform field to 1e-5 with the terms on; the default
// matrix form of J2 against the tangent form with G = 0 (pin hook field_gradient = 2) in that field.
// Seeding + parameter estimation (rules S, tests/test_oracle_seed.py): S5 exact on three points of an analytic helix
// (tangent, theta, q/p at the bottom point to 1e-9); S1-S4 against an enumeration of all combinations with other
// textbook formulas (R = abc / 4A, circle centre from the bisectors), default and binding cuts.  Navigation with discs
// and bidirectional navigation (tests/test_oracle_endcap.py): visited-module sequences against brute force.
// Ambiguity resolution (rules AR, tests/test_oracle_resolve.py): the greedy's result against the unique fixed point of
// its defining property found by brute force over all subsets of a small candidate set; limits k = 0 and k = infinity.
// Parity unpinned (convention only, fixed by DESIGN.md): that R10 cuts in TIP order (the closed form itself is pinned),
// hole-only-when-nothing-passes (A5), outward-only navigation (A7), inclusive in-bounds edges (A10),
// min_measurements = 3 (A14).
#include <cmath>
#include <cstdint>
#include <cstring>
#include <algorithm>
#include <thread>
#include <vector>

namespace {

constexpr double KAPPA = 2.99792458e-4;  // GeV / (T mm)   (U)
constexpr double PI = 3.14159265358979323846;

// ---------------------------------------------------------------------------------- inputs (POD)
struct OGeometry {
  int32_t n_layers;
  const double* layer_r;
  const double* layer_half_z;
  const int32_t* n_phi;
  const int32_t* n_z;
  const int32_t* module_offset;  // [n_layers+1]
  int32_t n_modules;
  const double* center;  // [M][3]
  const double* axis_u;  // [M][3]
  const double* axis_v;  // [M][3]
  const double* half_u;
  const double* half_v;
  const double* x_over_x0;
  // endcap discs (row f3; both NULL = barrel only).  Barrel layers come first, by increasing radius.  For a disc layer
  // l: layer_half_z[l] = signed z of its plane, layer_r_min[l] .. layer_r[l] its radial acceptance, n_z[l] = rings,
  // module id = module_offset[l] + i_phi * n_z[l] + i_ring, ring pitch = 2 * half_v of its modules.
  const int32_t* layer_kind;   // [n_layers] 0 barrel cylinder, 1 disc
  const double* layer_r_min;   // [n_layers]
};

struct OField {
  int32_t kind;  // 0 uniform, 1 grid
  double uniform_b[3];
  int32_t n[3];
  double origin[3];
  double spacing[3];
  const float* grid;  // [n0][n1][n2][3]
};

struct OConfig {
  double chi2_max;
  int32_t max_branches_per_surface;
  int32_t max_candidates_per_seed;
  int32_t max_holes;
  int32_t min_measurements;
  double rk_tolerance_mm;
  double surface_tolerance_mm;
  double h_max_mm;
  double particle_mass_gev;
  int32_t max_rk_steps_per_surface;
  int32_t max_levels;
  int32_t energy_loss;      // 1: mean energy loss of rule E in every crossed module (0 = BASELINE configs: "no energy loss")
  int32_t field_gradient;   // 1: transport Jacobian with the field-gradient terms of PAPER.md ref [18] (reading A13; 0 = ref [17])
  int32_t bidirectional;    // 1: tips that move radially INWARD are navigated too (rules N3'' below); 0 = reading A7:
                            //    outward-only, such tips stop NOT_OUTGOING (BASELINE configs)
};

enum StopReason { STOP_NONE = 0, STOP_EXIT = 1, STOP_HOLES = 2, STOP_NOT_OUTGOING = 3, STOP_STEP_LIMIT = 4,
                  STOP_NUMERIC = 5, STOP_LEVEL_LIMIT = 6 };

struct Counters {
  long long visits = 0, rk_trials = 0, rk_accepted = 0, gate_tests = 0, updates = 0, tips = 0;
};

// ---------------------------------------------------------------------------------- small algebra
inline void cross(const double a[3], const double b[3], double o[3]) {
  o[0] = a[1] * b[2] - a[2] * b[1];
  o[1] = a[2] * b[0] - a[0] * b[2];
  o[2] = a[0] * b[1] - a[1] * b[0];
}
inline double dot(const double a[3], const double b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

// M(B) v := v x B  as a 3x3 matrix acting on v  (J2)
inline void cross_matrix(const double B[3], double M[3][3]) {
  M[0][0] = 0.0;   M[0][1] = B[2];  M[0][2] = -B[1];
  M[1][0] = -B[2]; M[1][1] = 0.0;   M[1][2] = B[0];
  M[2][0] = B[1];  M[2][1] = -B[0]; M[2][2] = 0.0;
}
inline void mat3_mul(const double A[3][3], const double B[3][3], double O[3][3]) {
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      double s = 0.0;
      for (int k = 0; k < 3; ++k) s += A[i][k] * B[k][j];
      O[i][j] = s;
    }
}

// ---------------------------------------------------------------------------------- F: field
// Trilinear read of the float32 grid; lerp along x, then y, then z, each as a + f (b - a).
void field_at(const OField& f, const double r[3], double B[3]) {
  if (f.kind == 0) {
    B[0] = f.uniform_b[0]; B[1] = f.uniform_b[1]; B[2] = f.uniform_b[2];
    return;
  }
  if (f.kind == 2) {
    // PIN HOOK (tests only; the product has no such field kind): the analytic map behind configs[2]'s grid,
    // Bz = B0 (1 - a z^2), Br = a B0 r z (BASELINE.json configs[2]), with B0 = uniform_b[2] and a = origin[0].
    // A smooth non-uniform field lets the stepping (P2-P5) be compared with an independent ODE integrator and
    // the Jacobian with finite differences without the kinks of the trilinear interpolant.
    const double B0 = f.uniform_b[2], a = f.origin[0];
    B[0] = a * B0 * r[0] * r[2];
    B[1] = a * B0 * r[1] * r[2];
    B[2] = B0 * (1.0 - a * r[2] * r[2]);
    return;
  }
  int idx[3];
  double fr[3];
  for (int a = 0; a < 3; ++a) {
    double g = (r[a] - f.origin[a]) / f.spacing[a];
    double fl = std::floor(g);
    int i = (int)fl;
    if (i < 0) i = 0;
    if (i > f.n[a] - 2) i = f.n[a] - 2;
    idx[a] = i;
    fr[a] = g - (double)i;
  }
  const long long s0 = (long long)f.n[1] * f.n[2] * 3, s1 = (long long)f.n[2] * 3, s2 = 3;
  const float* p = f.grid + idx[0] * s0 + idx[1] * s1 + idx[2] * s2;
  for (int c = 0; c < 3; ++c) {
    double v000 = p[c], v100 = p[s0 + c], v010 = p[s1 + c], v110 = p[s0 + s1 + c];
    double v001 = p[s2 + c], v101 = p[s0 + s2 + c], v011 = p[s1 + s2 + c], v111 = p[s0 + s1 + s2 + c];
    double x00 = v000 + fr[0] * (v100 - v000);
    double x10 = v010 + fr[0] * (v110 - v010);
    double x01 = v001 + fr[0] * (v101 - v001);
    double x11 = v011 + fr[0] * (v111 - v011);
    double y0 = x00 + fr[1] * (x10 - x00);
    double y1 = x01 + fr[1] * (x11 - x01);
    B[c] = y0 + fr[2] * (y1 - y0);
  }
}

// Gradient of the field, G[i][j] = dB_i / dr_j, for the optional gradient terms of the transport Jacobian (J2'):
// zero for a uniform field; the exact derivative of the trilinear interpolant inside its cell for a grid (piecewise
// constant along the differentiated axis); analytic for the pin hook `kind 2`.
void field_gradient_at(const OField& f, const double r[3], double G[3][3]) {
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) G[i][j] = 0.0;
  if (f.kind == 0) return;
  if (f.kind == 2) {
    const double B0 = f.uniform_b[2], a = f.origin[0];
    G[0][0] = a * B0 * r[2]; G[0][2] = a * B0 * r[0];
    G[1][1] = a * B0 * r[2]; G[1][2] = a * B0 * r[1];
    G[2][2] = -2.0 * a * B0 * r[2];
    return;
  }
  int idx[3];
  double fr[3];
  for (int a = 0; a < 3; ++a) {
    double g = (r[a] - f.origin[a]) / f.spacing[a];
    int i = (int)std::floor(g);
    if (i < 0) i = 0;
    if (i > f.n[a] - 2) i = f.n[a] - 2;
    idx[a] = i;
    fr[a] = g - (double)i;
  }
  const long long st[3] = {(long long)f.n[1] * f.n[2] * 3, (long long)f.n[2] * 3, 3};
  const float* p = f.grid + idx[0] * st[0] + idx[1] * st[1] + idx[2] * st[2];
  for (int c = 0; c < 3; ++c)
    for (int ax = 0; ax < 3; ++ax) {
      // d/d(axis ax): difference along ax of the corner values, bilinear in the other two axes
      const int o1 = (ax + 1) % 3, o2 = (ax + 2) % 3;
      double acc = 0.0;
      for (int b1 = 0; b1 < 2; ++b1)
        for (int b2 = 0; b2 < 2; ++b2) {
          const long long base = b1 * st[o1] + b2 * st[o2];
          const double diff = (double)p[base + st[ax] + c] - (double)p[base + c];
          acc += (b1 ? fr[o1] : 1.0 - fr[o1]) * (b2 ? fr[o2] : 1.0 - fr[o2]) * diff;
        }
      G[c][ax] = acc / f.spacing[ax];
    }
}

// ---------------------------------------------------------------------------------- free state + transport Jacobian
// Free vector y = (r[0..2], t, d[0..2], q/p)  (U);  D = d y / d y_departure (8x8, J3)
struct FreeState {
  double r[3], t, d[3], qop;
  double D[8][8];
  double h_ctrl;   // P3/P4: step-size proposal carried between steps
  int n_steps;     // attempted RKN4 steps since the tip left its module (P6)
};

void set_identity8(double D[8][8]) {
  for (int i = 0; i < 8; ++i)
    for (int j = 0; j < 8; ++j) D[i][j] = (i == j) ? 1.0 : 0.0;
}

// D <- Dstep * D
void apply_step_jacobian(double D[8][8], const double Ds[8][8]) {
  double O[8][8];
  for (int i = 0; i < 8; ++i)
    for (int j = 0; j < 8; ++j) {
      double s = 0.0;
      for (int k = 0; k < 8; ++k) s += Ds[i][k] * D[k][j];
      O[i][j] = s;
    }
  std::memcpy(D, O, sizeof(O));
}

inline double inv_beta(double qop, double mass) { return std::sqrt(1.0 + mass * mass * qop * qop); }
inline double dinvbeta_dqop(double qop, double mass) {
  return mass * mass * qop / std::sqrt(1.0 + mass * mass * qop * qop);
}

// P2 + P3 + J2: one RKN4 trial of signed length h.  Returns the error estimate eps; on request applies it.
struct Trial {
  double k1[3], k2[3], k3[3], k4[3], B1[3], B2[3], B4[3];
  double rm[3], re[3];   // stage points (for the gradient terms of J2')
  double eps;
};

void rk_trial(const OField& fld, const FreeState& y, double h, Trial& T) {
  const double lam = KAPPA * y.qop;
  double tmp[3], dd[3], rm[3], re[3];
  field_at(fld, y.r, T.B1);
  cross(y.d, T.B1, tmp);
  for (int i = 0; i < 3; ++i) T.k1[i] = lam * tmp[i];
  for (int i = 0; i < 3; ++i) rm[i] = y.r[i] + 0.5 * h * y.d[i] + h * h / 8.0 * T.k1[i];
  for (int i = 0; i < 3; ++i) T.rm[i] = rm[i];
  field_at(fld, rm, T.B2);
  for (int i = 0; i < 3; ++i) dd[i] = y.d[i] + 0.5 * h * T.k1[i];
  cross(dd, T.B2, tmp);
  for (int i = 0; i < 3; ++i) T.k2[i] = lam * tmp[i];
  for (int i = 0; i < 3; ++i) dd[i] = y.d[i] + 0.5 * h * T.k2[i];
  cross(dd, T.B2, tmp);
  for (int i = 0; i < 3; ++i) T.k3[i] = lam * tmp[i];
  for (int i = 0; i < 3; ++i) re[i] = y.r[i] + h * y.d[i] + h * h / 2.0 * T.k3[i];
  for (int i = 0; i < 3; ++i) T.re[i] = re[i];
  field_at(fld, re, T.B4);
  for (int i = 0; i < 3; ++i) dd[i] = y.d[i] + h * T.k3[i];
  cross(dd, T.B4, tmp);
  for (int i = 0; i < 3; ++i) T.k4[i] = lam * tmp[i];
  double e2 = 0.0;
  for (int i = 0; i < 3; ++i) {
    double e = T.k1[i] - T.k2[i] - T.k3[i] + T.k4[i];
    e2 += e * e;
  }
  T.eps = h * h * std::sqrt(e2);
}

// J2' (config.field_gradient = 1; reading A13, PAPER.md ref [18]): the step map of P2 differentiated stage by stage
// with h fixed INCLUDING the dependence of the field on the stage points.  Written as seven tangent vectors
// (dr, dd, dlam) -- one per column r_x, r_y, r_z, d_x, d_y, d_z, lambda -- pushed through the four stages:
//   dk1 = lam [dd x B1 + d x (G1 dr)] + dlam (d x B1)
//   drm = dr + h/2 dd + h^2/8 dk1
//   dk2 = lam [(dd + h/2 dk1) x B2 + (d + h/2 k1) x (G2 drm)] + dlam ((d + h/2 k1) x B2)      dk3 likewise from k2
//   dre = dr + h dd + h^2/2 dk3
//   dk4 = lam [(dd + h dk3) x B4 + (d + h k3) x (G4 dre)] + dlam ((d + h k3) x B4)
//   dr' = dr + h dd + h^2/6 (dk1 + dk2 + dk3),   dd' = dd + h/6 (dk1 + 2 dk2 + 2 dk3 + dk4)
// With G = 0 this is J2 (dr'/dr = I, dd'/dr = 0).
void step_jacobian_with_gradient(const OField& fld, const FreeState& y, double h, const Trial& T, double mass,
                                 bool zero_gradient, double Ds[8][8]) {
  const double lam = KAPPA * y.qop;
  double G1[3][3], G2[3][3], G4[3][3];
  field_gradient_at(fld, y.r, G1);
  field_gradient_at(fld, T.rm, G2);
  field_gradient_at(fld, T.re, G4);
  if (zero_gradient)   // PIN HOOK (field_gradient = 2): this tangent form with G = 0 must equal the matrix form of J2
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 3; ++j) G1[i][j] = G2[i][j] = G4[i][j] = 0.0;
  set_identity8(Ds);
  auto gmul = [](const double G[3][3], const double v[3], double o[3]) {
    for (int i = 0; i < 3; ++i) o[i] = G[i][0] * v[0] + G[i][1] * v[1] + G[i][2] * v[2];
  };
  for (int c = 0; c < 7; ++c) {
    double dr[3] = {0, 0, 0}, dd[3] = {0, 0, 0}, dlam = 0.0;
    if (c < 3) dr[c] = 1.0;
    else if (c < 6) dd[c - 3] = 1.0;
    else dlam = 1.0;
    double dk1[3], dk2[3], dk3[3], dk4[3], drm[3], dre[3], w[3], dw[3], a[3], b[3], gb[3];
    // stage 1
    cross(dd, T.B1, a);
    gmul(G1, dr, gb);
    cross(y.d, gb, b);
    cross(y.d, T.B1, w);
    for (int i = 0; i < 3; ++i) dk1[i] = lam * (a[i] + b[i]) + dlam * w[i];
    for (int i = 0; i < 3; ++i) drm[i] = dr[i] + 0.5 * h * dd[i] + h * h / 8.0 * dk1[i];
    // stage 2
    for (int i = 0; i < 3; ++i) { w[i] = y.d[i] + 0.5 * h * T.k1[i]; dw[i] = dd[i] + 0.5 * h * dk1[i]; }
    cross(dw, T.B2, a);
    gmul(G2, drm, gb);
    cross(w, gb, b);
    cross(w, T.B2, gb);
    for (int i = 0; i < 3; ++i) dk2[i] = lam * (a[i] + b[i]) + dlam * gb[i];
    // stage 3
    for (int i = 0; i < 3; ++i) { w[i] = y.d[i] + 0.5 * h * T.k2[i]; dw[i] = dd[i] + 0.5 * h * dk2[i]; }
    cross(dw, T.B2, a);
    gmul(G2, drm, gb);
    cross(w, gb, b);
    cross(w, T.B2, gb);
    for (int i = 0; i < 3; ++i) dk3[i] = lam * (a[i] + b[i]) + dlam * gb[i];
    for (int i = 0; i < 3; ++i) dre[i] = dr[i] + h * dd[i] + h * h / 2.0 * dk3[i];
    // stage 4
    for (int i = 0; i < 3; ++i) { w[i] = y.d[i] + h * T.k3[i]; dw[i] = dd[i] + h * dk3[i]; }
    cross(dw, T.B4, a);
    gmul(G4, dre, gb);
    cross(w, gb, b);
    cross(w, T.B4, gb);
    for (int i = 0; i < 3; ++i) dk4[i] = lam * (a[i] + b[i]) + dlam * gb[i];
    const int col = c < 3 ? c : (c < 6 ? 4 + (c - 3) : 7);
    const double scale = (c == 6) ? KAPPA : 1.0;   // d/d(q/p) = kappa d/dlam
    for (int i = 0; i < 3; ++i) {
      Ds[i][col] = scale * (dr[i] + h * dd[i] + h * h / 6.0 * (dk1[i] + dk2[i] + dk3[i]));
      Ds[4 + i][col] = scale * (dd[i] + h / 6.0 * (dk1[i] + 2.0 * dk2[i] + 2.0 * dk3[i] + dk4[i]));
    }
  }
  Ds[3][7] = h * dinvbeta_dqop(y.qop, mass);
}

void rk_accept(const OField& fld, const OConfig& cfg, FreeState& y, double h, const Trial& T, double mass) {
  const double lam = KAPPA * y.qop;
  if (cfg.field_gradient) {
    double Dg[8][8];
    step_jacobian_with_gradient(fld, y, h, T, mass, cfg.field_gradient == 2, Dg);
    apply_step_jacobian(y.D, Dg);
  } else {
  // ---- J2: step Jacobian, field gradient neglected, h fixed
  double M1[3][3], M2[3][3], M4[3][3], A1[3][3], A2[3][3], A3[3][3], A4[3][3], W[3][3], X[3][3];
  double a1[3], a2[3], a3[3], a4[3], dd[3], t1[3], t2[3];
  cross_matrix(T.B1, M1);
  cross_matrix(T.B2, M2);
  cross_matrix(T.B4, M4);
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) A1[i][j] = lam * M1[i][j];
  cross(y.d, T.B1, a1);
  // A2 = lam M(B2) (I + h/2 A1);  a2 = (d + h/2 k1) x B2 + lam (h/2 a1) x B2
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) W[i][j] = (i == j ? 1.0 : 0.0) + 0.5 * h * A1[i][j];
  mat3_mul(M2, W, X);
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) A2[i][j] = lam * X[i][j];
  for (int i = 0; i < 3; ++i) dd[i] = y.d[i] + 0.5 * h * T.k1[i];
  cross(dd, T.B2, t1);
  for (int i = 0; i < 3; ++i) dd[i] = 0.5 * h * a1[i];
  cross(dd, T.B2, t2);
  for (int i = 0; i < 3; ++i) a2[i] = t1[i] + lam * t2[i];
  // A3 from k2 (same B2)
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) W[i][j] = (i == j ? 1.0 : 0.0) + 0.5 * h * A2[i][j];
  mat3_mul(M2, W, X);
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) A3[i][j] = lam * X[i][j];
  for (int i = 0; i < 3; ++i) dd[i] = y.d[i] + 0.5 * h * T.k2[i];
  cross(dd, T.B2, t1);
  for (int i = 0; i < 3; ++i) dd[i] = 0.5 * h * a2[i];
  cross(dd, T.B2, t2);
  for (int i = 0; i < 3; ++i) a3[i] = t1[i] + lam * t2[i];
  // A4 from k3 with h and B4
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) W[i][j] = (i == j ? 1.0 : 0.0) + h * A3[i][j];
  mat3_mul(M4, W, X);
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) A4[i][j] = lam * X[i][j];
  for (int i = 0; i < 3; ++i) dd[i] = y.d[i] + h * T.k3[i];
  cross(dd, T.B4, t1);
  for (int i = 0; i < 3; ++i) dd[i] = h * a3[i];
  cross(dd, T.B4, t2);
  for (int i = 0; i < 3; ++i) a4[i] = t1[i] + lam * t2[i];

  double Ds[8][8];
  set_identity8(Ds);
  for (int i = 0; i < 3; ++i) {
    for (int j = 0; j < 3; ++j) {
      Ds[i][4 + j] = (i == j ? h : 0.0) + h * h / 6.0 * (A1[i][j] + A2[i][j] + A3[i][j]);
      Ds[4 + i][4 + j] = (i == j ? 1.0 : 0.0) + h / 6.0 * (A1[i][j] + 2.0 * A2[i][j] + 2.0 * A3[i][j] + A4[i][j]);
    }
    Ds[i][7] = KAPPA * (h * h / 6.0 * (a1[i] + a2[i] + a3[i]));
    Ds[4 + i][7] = KAPPA * (h / 6.0 * (a1[i] + 2.0 * a2[i] + 2.0 * a3[i] + a4[i]));
  }
  Ds[3][7] = h * dinvbeta_dqop(y.qop, mass);
  apply_step_jacobian(y.D, Ds);
  }

  // ---- P2: the state
  double dn[3], nrm2 = 0.0;
  for (int i = 0; i < 3; ++i) {
    y.r[i] = y.r[i] + h * y.d[i] + h * h / 6.0 * (T.k1[i] + T.k2[i] + T.k3[i]);
    dn[i] = y.d[i] + h / 6.0 * (T.k1[i] + 2.0 * T.k2[i] + 2.0 * T.k3[i] + T.k4[i]);
    nrm2 += dn[i] * dn[i];
  }
  const double nrm = std::sqrt(nrm2);
  for (int i = 0; i < 3; ++i) y.d[i] = dn[i] / nrm;
  y.t += h * inv_beta(y.qop, mass);
}

// P5: field-free closing step of length s
void straight_close(FreeState& y, double s, double mass) {
  double Ds[8][8];
  set_identity8(Ds);
  for (int i = 0; i < 3; ++i) Ds[i][4 + i] = s;
  Ds[3][7] = s * dinvbeta_dqop(y.qop, mass);
  apply_step_jacobian(y.D, Ds);
  for (int i = 0; i < 3; ++i) y.r[i] += s * y.d[i];
  y.t += s * inv_beta(y.qop, mass);
}

struct Target {
  int kind;      // 0 plane (c, n); cylinder of radius R around z: 1 crossed outward, 2 crossed INWARD from outside,
                 // 3 FAR crossing (the tip is inside or on it and leaves through its far side)
  double c[3], n[3], R;
};

// P4: signed straight-line distance to the target along d.  Returns false if unreachable (P6).
bool target_distance(const Target& tg, const FreeState& y, double& s, int& why) {
  if (tg.kind == 0) {
    double dn = dot(y.d, tg.n);
    if (!(std::fabs(dn) > 1e-12)) { why = STOP_NUMERIC; return false; }
    double rel[3] = {tg.c[0] - y.r[0], tg.c[1] - y.r[1], tg.c[2] - y.r[2]};
    s = dot(rel, tg.n) / dn;
    return true;
  }
  const double a = y.d[0] * y.d[0] + y.d[1] * y.d[1];
  const double b = y.r[0] * y.d[0] + y.r[1] * y.d[1];
  const double cc = y.r[0] * y.r[0] + y.r[1] * y.r[1] - tg.R * tg.R;
  const double disc = b * b - a * cc;
  if (tg.kind == 2) {
    // N3'': the cylinder is inside the tip's radius and the tip moves inward: near root of a s^2 + 2 b s + cc = 0,
    // s = cc / (-b + sqrt(disc)) (signed: negative once the tip has overshot to the inside)
    if (!(b < 0.0) || !(disc >= 0.0)) { why = STOP_NOT_OUTGOING; return false; }   // it turned before reaching it
    s = cc / (-b + std::sqrt(disc));
    return true;
  }
  if (tg.kind == 3) {
    // N3'': far root (-b + sqrt(disc)) / a, written without cancellation for either sign of b
    if (!(disc >= 0.0)) { why = STOP_NOT_OUTGOING; return false; }
    const double sq = std::sqrt(disc);
    s = b < 0.0 ? (-b + sq) / a : -cc / (b + sq);
    return true;
  }
  if (!(b > 0.0) || !(disc >= 0.0)) { why = STOP_NOT_OUTGOING; return false; }
  s = -cc / (b + std::sqrt(disc));
  return true;
}

// P3-P6: step until the target is reached.  Returns STOP_NONE on success.
int propagate_to(const OField& fld, const OConfig& cfg, const Target& tg, FreeState& y, Counters& cnt) {
  const double mass = cfg.particle_mass_gev;
  for (;;) {
    double s;
    int why = STOP_NUMERIC;
    if (!target_distance(tg, y, s, why)) return why;
    if (!std::isfinite(s)) return STOP_NUMERIC;
    if (std::fabs(s) <= cfg.surface_tolerance_mm) {
      straight_close(y, s, mass);
      return STOP_NONE;
    }
    const double hlim = std::min(y.h_ctrl, cfg.h_max_mm);
    double h = (std::fabs(s) <= hlim) ? s : (s > 0.0 ? hlim : -hlim);
    for (;;) {
      if (++y.n_steps > cfg.max_rk_steps_per_surface) return STOP_STEP_LIMIT;
      Trial T;
      rk_trial(fld, y, h, T);
      ++cnt.rk_trials;
      if (!std::isfinite(T.eps)) return STOP_NUMERIC;
      double f;
      if (T.eps == 0.0) f = 4.0;
      else {
        f = 0.9 * std::sqrt(std::sqrt(cfg.rk_tolerance_mm / T.eps));
        if (f < 0.25) f = 0.25;
        if (f > 4.0) f = 4.0;
      }
      if (T.eps <= cfg.rk_tolerance_mm) {
        rk_accept(fld, cfg, y, h, T, mass);
        y.h_ctrl = std::fabs(h) * f;
        ++cnt.rk_accepted;
        break;
      }
      h = h * f;
    }
  }
}

// ---------------------------------------------------------------------------------- bound <-> free
struct Module {
  int id, layer, iphi, iz;
  double c[3], u[3], v[3], n[3], half_u, half_v, x_over_x0;
};

Module get_module(const OGeometry& g, int id) {
  Module m;
  m.id = id;
  int l = 0;
  while (l + 1 < g.n_layers && id >= g.module_offset[l + 1]) ++l;
  m.layer = l;
  int loc = id - g.module_offset[l];
  m.iphi = loc / g.n_z[l];
  m.iz = loc % g.n_z[l];
  for (int i = 0; i < 3; ++i) {
    m.c[i] = g.center[3 * id + i];
    m.u[i] = g.axis_u[3 * id + i];
    m.v[i] = g.axis_v[3 * id + i];
  }
  cross(m.u, m.v, m.n);
  m.half_u = g.half_u[id];
  m.half_v = g.half_v[id];
  m.x_over_x0 = g.x_over_x0[id];
  return m;
}

// bound x = (l0, l1, phi, theta, q/p, t)
void bound_to_free(const Module& m, const double x[6], FreeState& y, double B2F[8][6]) {
  const double sp = std::sin(x[2]), cp = std::cos(x[2]), st = std::sin(x[3]), ct = std::cos(x[3]);
  for (int i = 0; i < 3; ++i) y.r[i] = m.c[i] + x[0] * m.u[i] + x[1] * m.v[i];
  y.t = x[5];
  y.d[0] = st * cp; y.d[1] = st * sp; y.d[2] = ct;
  y.qop = x[4];
  // J1
  for (int i = 0; i < 8; ++i)
    for (int j = 0; j < 6; ++j) B2F[i][j] = 0.0;
  for (int i = 0; i < 3; ++i) { B2F[i][0] = m.u[i]; B2F[i][1] = m.v[i]; }
  B2F[3][5] = 1.0;
  B2F[4][2] = -st * sp; B2F[5][2] = st * cp;  B2F[6][2] = 0.0;
  B2F[4][3] = ct * cp;  B2F[5][3] = ct * sp;  B2F[6][3] = -st;
  B2F[7][4] = 1.0;
}

// J4 + J5: arrival on plane of module m; outputs bound x', J (6x6) given B2F of the departure
void arrive(const OField& fld, const OConfig& cfg, const Module& m, const FreeState& y, const double B2F[8][6],
            double xo[6], double J[6][6]) {
  const double mass = cfg.particle_mass_gev;
  const double lam = KAPPA * y.qop;
  double B[3], dxB[3];
  field_at(fld, y.r, B);
  cross(y.d, B, dxB);
  // y' = (d, 1/beta, lam d x B, 0)
  double yp[8] = {y.d[0], y.d[1], y.d[2], inv_beta(y.qop, mass), lam * dxB[0], lam * dxB[1], lam * dxB[2], 0.0};
  const double nd = dot(m.n, y.d);
  // P = I - y' w^T / (n.d),  w = (n, 0, 0, 0, 0, 0)
  double P[8][8];
  set_identity8(P);
  for (int i = 0; i < 8; ++i)
    for (int j = 0; j < 3; ++j) P[i][j] -= yp[i] * m.n[j] / nd;
  // bound parameters on arrival (J5)
  double rel[3] = {y.r[0] - m.c[0], y.r[1] - m.c[1], y.r[2] - m.c[2]};
  const double phi = std::atan2(y.d[1], y.d[0]);
  const double theta = std::atan2(std::hypot(y.d[0], y.d[1]), y.d[2]);
  xo[0] = dot(rel, m.u); xo[1] = dot(rel, m.v); xo[2] = phi; xo[3] = theta; xo[4] = y.qop; xo[5] = y.t;
  const double sp = std::sin(phi), cp = std::cos(phi), st = std::sin(theta), ct = std::cos(theta);
  double F2B[6][8];
  for (int i = 0; i < 6; ++i)
    for (int j = 0; j < 8; ++j) F2B[i][j] = 0.0;
  for (int j = 0; j < 3; ++j) { F2B[0][j] = m.u[j]; F2B[1][j] = m.v[j]; }
  F2B[2][4] = -sp / st; F2B[2][5] = cp / st; F2B[2][6] = 0.0;
  F2B[3][4] = ct * cp;  F2B[3][5] = ct * sp; F2B[3][6] = -st;
  F2B[4][7] = 1.0;
  F2B[5][3] = 1.0;
  // J = F2B P D B2F
  double PD[8][8], PDB[8][6];
  for (int i = 0; i < 8; ++i)
    for (int j = 0; j < 8; ++j) {
      double s = 0.0;
      for (int k = 0; k < 8; ++k) s += P[i][k] * y.D[k][j];
      PD[i][j] = s;
    }
  for (int i = 0; i < 8; ++i)
    for (int j = 0; j < 6; ++j) {
      double s = 0.0;
      for (int k = 0; k < 8; ++k) s += PD[i][k] * B2F[k][j];
      PDB[i][j] = s;
    }
  for (int i = 0; i < 6; ++i)
    for (int j = 0; j < 6; ++j) {
      double s = 0.0;
      for (int k = 0; k < 8; ++k) s += F2B[i][k] * PDB[k][j];
      J[i][j] = s;
    }
}

void transport_cov(const double J[6][6], const double C[6][6], double Co[6][6]) {
  double JC[6][6], T[6][6];
  for (int i = 0; i < 6; ++i)
    for (int j = 0; j < 6; ++j) {
      double s = 0.0;
      for (int k = 0; k < 6; ++k) s += J[i][k] * C[k][j];
      JC[i][j] = s;
    }
  for (int i = 0; i < 6; ++i)
    for (int j = 0; j < 6; ++j) {
      double s = 0.0;
      for (int k = 0; k < 6; ++k) s += JC[i][k] * J[j][k];
      T[i][j] = s;
    }
  for (int i = 0; i < 6; ++i)
    for (int j = 0; j < 6; ++j) Co[i][j] = 0.5 * (T[i][j] + T[j][i]);
}

// ---------------------------------------------------------------------------------- V5: Highland
double highland_theta0(double p, double x_eff, double mass) {
  const double beta = p / std::sqrt(p * p + mass * mass);
  return 0.0136 / (beta * p) * std::sqrt(x_eff) * (1.0 + 0.038 * std::log(x_eff / (beta * beta)));
}

void add_material(const OConfig& cfg, const Module& m, const double x[6], double C[6][6]) {
  if (!(m.x_over_x0 > 0.0)) return;
  const double st = std::sin(x[3]), ct = std::cos(x[3]);
  const double d[3] = {st * std::cos(x[2]), st * std::sin(x[2]), ct};
  const double cosi = std::fabs(dot(d, m.n));
  const double p = 1.0 / std::fabs(x[4]);
  const double th0 = highland_theta0(p, m.x_over_x0 / cosi, cfg.particle_mass_gev);
  C[3][3] += th0 * th0;
  C[2][2] += th0 * th0 / (st * st);
}

// ---------------------------------------------------------------------------------- E: mean energy loss
// "effects from material interactions are evaluated by assuming muon trajectories".  BASELINE configs
// switch energy loss off; rule E adds the MEAN loss of the muon hypothesis in
// every crossed module, next to V5.  Mean stopping power of a heavy charged particle (Bethe, as tabulated by the PDG
// review "Passage of particles through matter"), density-effect correction neglected (reading):
//   -dE/dx = K (Z/A) / beta^2 [ 1/2 ln(2 me beta^2 gamma^2 Wmax / I^2) - beta^2 ],
//   Wmax = 2 me (beta gamma)^2 / (1 + 2 gamma me/M + (me/M)^2),      K = 0.307075 MeV cm^2 / mol.
// The modules are silicon (configs[0]: "0.15 mm silicon (x/X0 = 0.0016)"): Z/A = 0.49848 mol/g, I = 173 eV,
// X0 = 21.82 g/cm^2, so a module of x/X0 crossed at incidence |d.n| is (x/X0) / |d.n| * 21.82 g/cm^2 of silicon.
constexpr double EL_K = 0.307075e-3;      // GeV cm^2 / mol
constexpr double EL_Z_OVER_A = 0.49848;   // mol / g   (silicon)
constexpr double EL_I = 173.0e-9;         // GeV       (silicon mean excitation energy)
constexpr double EL_X0 = 21.82;           // g / cm^2  (silicon radiation length)
constexpr double EL_ME = 0.51099895e-3;   // GeV

// mean stopping power [GeV cm^2 / g] of a singly charged particle of mass M and momentum p in silicon
double bethe_dedx(double p, double M) {
  const double bg2 = (p * p) / (M * M);
  const double E = std::sqrt(p * p + M * M);
  const double beta2 = (p * p) / (E * E), gamma = E / M;
  const double r = EL_ME / M;
  const double wmax = 2.0 * EL_ME * bg2 / (1.0 + 2.0 * gamma * r + r * r);
  return EL_K * EL_Z_OVER_A / beta2 * (0.5 * std::log(2.0 * EL_ME * bg2 * wmax / (EL_I * EL_I)) - beta2);
}

// Rule E on leaving module m with bound parameters x: returns dE [GeV]; xo = x with q/p after the loss
// (E' = E - dE, p' = sqrt(E'^2 - M^2); not finite if the particle would stop), g = d(q/p)'/d(q/p) with dE held
// fixed (reading: like the field gradient in J2, the slow dependence of dE on p is neglected):
//   dE' = dE = (p/E) dp,  dp' = (E'/p') dE'   =>   g = (p/p')^3 (E'/E).
double energy_loss(const OConfig& cfg, const Module& m, const double x[6], double xo[6], double& g) {
  for (int i = 0; i < 6; ++i) xo[i] = x[i];
  g = 1.0;
  if (!cfg.energy_loss || !(m.x_over_x0 > 0.0)) return 0.0;
  const double M = cfg.particle_mass_gev;
  const double st = std::sin(x[3]), ct = std::cos(x[3]);
  const double d[3] = {st * std::cos(x[2]), st * std::sin(x[2]), ct};
  const double cosi = std::fabs(dot(d, m.n));
  const double p = 1.0 / std::fabs(x[4]);
  const double E = std::sqrt(p * p + M * M);
  const double dE = bethe_dedx(p, M) * (m.x_over_x0 / cosi) * EL_X0;
  const double E2 = E - dE;
  const double p2 = std::sqrt(E2 * E2 - M * M);     // NaN if E' < M: the tip then stops NUMERIC
  xo[4] = (x[4] < 0.0 ? -1.0 : 1.0) / p2;
  g = (p / p2) * (p / p2) * (p / p2) * (E2 / E);
  return dE;
}

// ---------------------------------------------------------------------------------- N: navigation
// PIN HOOK: 1 = walk the remaining portal cylinders literally as SURVEY.md N3 words it ("l' <- l' + 1 and repeat"),
// 0 (default) = reading D11: a tip beyond every further half-length and moving away in z stops EXIT at
// once.  tests/test_oracle_pins.py runs both and checks that the candidates are the same.
int g_n3_literal_walk = 0;

// straight-line test of one module from the point (r, d): N2 / N4
// (g_bidirectional, set per call from config.bidirectional: a module may also be crossed AGAINST its normal)
thread_local int g_bidirectional = 0;
bool line_hits_module(const Module& k, const double r[3], const double d[3], double s_min, double& s_out) {
  const double dn = dot(d, k.n);
  if (g_bidirectional ? std::fabs(dn) <= 1e-6 : dn <= 1e-6) return false;
  double rel[3] = {k.c[0] - r[0], k.c[1] - r[1], k.c[2] - r[2]};
  const double s = dot(rel, k.n) / dn;
  double q[3] = {r[0] + s * d[0] - k.c[0], r[1] + s * d[1] - k.c[1], r[2] + s * d[2] - k.c[2]};
  if (!(std::fabs(dot(q, k.u)) <= k.half_u)) return false;
  if (!(std::fabs(dot(q, k.v)) <= k.half_v)) return false;
  if (!(s > s_min)) return false;
  s_out = s;
  return true;
}

// nearest in-bounds module among the 3x3 neighbourhood of (iphi, iz) on `layer`, excluding `exclude`
int pick_in_neighbourhood(const OGeometry& g, int layer, int iphi, int iz, int exclude, const double r[3],
                          const double d[3], double s_min) {
  int best = -1;
  double best_s = 0.0;
  const int nphi = g.n_phi[layer], nz = g.n_z[layer];
  for (int di = -1; di <= 1; ++di)
    for (int dj = -1; dj <= 1; ++dj) {
      const int jj = iz + dj;
      if (jj < 0 || jj >= nz) continue;
      const int ii = ((iphi + di) % nphi + nphi) % nphi;
      const int id = g.module_offset[layer] + ii * nz + jj;
      if (id == exclude) continue;
      Module k = get_module(g, id);
      double s;
      if (!line_hits_module(k, r, d, s_min, s)) continue;
      if (best < 0 || s < best_s || (s == best_s && id < best)) { best = id; best_s = s; }
    }
  return best;
}

// One surface-to-surface move (N1-N5 + P + J): from bound (x, C) on module `from` to the next module.
// Material (V5) is added to C on leaving.  Returns STOP_NONE and (target, xp, Cp), or the stop reason.
int move_to_next_module(const OGeometry& g, const OField& fld, const OConfig& cfg, int from, const double x[6],
                        const double Cin[6][6], int& target, double xp[6], double Cp[6][6], double Jout[6][6],
                        Counters& cnt) {
  for (int i = 0; i < 6; ++i)
    if (!std::isfinite(x[i])) return STOP_NUMERIC;
  if (!(x[3] > 0.0 && x[3] < PI)) return STOP_NUMERIC;
  const Module m = get_module(g, from);
  g_bidirectional = cfg.bidirectional;
  double C[6][6];
  std::memcpy(C, Cin, sizeof(C));
  add_material(cfg, m, x, C);              // V5, with the momentum the tip arrived with
  double xd[6], gE = 1.0;                  // E: departure parameters after the mean energy loss, J_E = diag(1,1,1,1,gE,1)
  energy_loss(cfg, m, x, xd, gE);
  if (!std::isfinite(xd[4])) return STOP_NUMERIC;
  for (int i = 0; i < 6; ++i) { C[i][4] *= gE; C[4][i] *= gE; }   // C <- J_E C J_E^T (C[4][4] gets gE twice)
  FreeState y;
  double B2F[8][6];
  bound_to_free(m, xd, y, B2F);
  set_identity8(y.D);
  y.h_ctrl = cfg.h_max_mm;
  y.n_steps = 0;
  // N2: overlap neighbour on the same layer
  int tgt = pick_in_neighbourhood(g, m.layer, m.iphi, m.iz, m.id, y.r, y.d, 1e-3);
  if (tgt < 0) {
    // N3': the next PORTAL -- the cylinder of the next barrel layer, or the plane of the next disc in the direction of
    // d_z, whichever the straight line from here reaches first -- then N4 module choice on it.  Barrel only, this is
    // SURVEY's N3 with reading D11; discs (row f3) add the second family of portals.
    const bool has_discs = g.layer_kind != nullptr;
    auto is_disc = [&](int l) { return has_discs && g.layer_kind[l] == 1; };
    int n_barrel = 0;
    while (n_barrel < g.n_layers && !is_disc(n_barrel)) ++n_barrel;
    // next disc after disc layer `l` on its side (larger |z|), or the first disc ahead of z when l < 0
    auto disc_after = [&](int l, double z, double dz) {
      int best = -1;
      for (int k = n_barrel; k < g.n_layers; ++k) {
        const double zk = g.layer_half_z[k];
        bool ahead;
        if (l >= 0) ahead = (zk > 0.0) == (g.layer_half_z[l] > 0.0) && std::fabs(zk) > std::fabs(g.layer_half_z[l]);
        else ahead = dz != 0.0 && (zk - z) * dz > 0.0;
        if (ahead && (best < 0 || std::fabs(zk - z) < std::fabs(g.layer_half_z[best] - z))) best = k;
      }
      return best;
    };
    int lb, ld;   // radial shell: last barrel cylinder inside the tip (the next one outward is lb + 1, the next one
                  // inward is lb itself); next disc candidate (-1 = none)
    const bool bidir = cfg.bidirectional != 0;
    if (is_disc(m.layer)) {
      const double rho = std::hypot(y.r[0], y.r[1]);
      lb = -1;
      while (lb + 1 < n_barrel && g.layer_r[lb + 1] <= rho) ++lb;
      ld = disc_after(m.layer, y.r[2], y.d[2]);
    } else {
      lb = m.layer;
      // N3'': a tip that leaves a barrel module INWARD has its own layer's cylinder behind it already
      if (bidir && y.r[0] * y.d[0] + y.r[1] * y.d[1] < 0.0) lb = m.layer - 1;
      ld = disc_after(-1, y.r[2], y.d[2]);
    }
    for (;;) {
      // a barrel layer whose half length is already behind a tip that moves away in z cannot be crossed inside its
      // acceptance: it is passed without propagating to it (reading D11, per layer)
      const double a = y.d[0] * y.d[0] + y.d[1] * y.d[1], b = y.r[0] * y.d[0] + y.r[1] * y.d[1];
      const double rho2 = y.r[0] * y.r[0] + y.r[1] * y.r[1];
      const bool inward = bidir && b < 0.0;
      while (!inward && !g_n3_literal_walk && lb + 1 < n_barrel && std::fabs(y.r[2]) > g.layer_half_z[lb + 1] &&
             y.r[2] * y.d[2] > 0.0)
        ++lb;
      // likewise a disc whose plane is not ahead (any more), or whose outer radius is already behind a tip that moves
      // outward radially, is passed
      while (ld >= 0 && ((g.layer_half_z[ld] - y.r[2]) * y.d[2] <= 0.0 ||
                         (rho2 > g.layer_r[ld] * g.layer_r[ld] && b > 0.0)))
        ld = disc_after(ld, y.r[2], y.d[2]);
      int lc = lb + 1 < n_barrel ? lb + 1 : -1;
      int cyl_kind = 1;   // how the cylinder candidate is crossed: 1 outward, 2 inward, 3 through its far side
      double r_target = 0.0;
      if (inward) {
        // N3'': moving inward.  The candidate is the next inner cylinder (lb, or the first one below it whose half
        // length is not behind a tip moving away in z) if the straight line reaches it; otherwise the tip turns inside
        // its shell and leaves through the FAR side of the cylinder that bounds the shell from outside (lb + 1).
        // The flat modules of a layer lie OUTSIDE its cylinder, between r and hypot(r, half_u): a tip coming from
        // outside meets them before it meets the cylinder, so the inward portal of a layer is its outer envelope.
        int li = lb;
        while (!g_n3_literal_walk && li >= 0 && std::fabs(y.r[2]) > g.layer_half_z[li] && y.r[2] * y.d[2] > 0.0) --li;
        if (li >= 0) r_target = std::hypot(g.layer_r[li], g.half_u[g.module_offset[li]]);
        if (li >= 0 && b * b - a * (rho2 - r_target * r_target) >= 0.0) { lc = li; cyl_kind = 2; }
        else {
          cyl_kind = 3;   // first cylinder from lb + 1 outward that the straight line meets at all
          while (lc >= 0 && b * b - a * (rho2 - g.layer_r[lc] * g.layer_r[lc]) < 0.0) lc = lc + 1 < n_barrel ? lc + 1 : -1;
        }
      }
      if (cyl_kind != 2 && lc >= 0) r_target = g.layer_r[lc];
      if (lc < 0 && ld < 0) return STOP_EXIT;
      bool to_disc = false;
      if (ld >= 0) {
        const double s_d = (g.layer_half_z[ld] - y.r[2]) / y.d[2];
        double s_c = INFINITY;   // straight-line distance to the cylinder (P4), infinite when it is not ahead
        if (lc >= 0) {
          const double cc = rho2 - r_target * r_target;
          const double disc = b * b - a * cc;
          if (cyl_kind == 1) { if (b > 0.0 && disc >= 0.0) s_c = -cc / (b + std::sqrt(disc)); }
          else if (cyl_kind == 2) s_c = cc / (-b + std::sqrt(disc));
          else if (disc >= 0.0) s_c = (-b + std::sqrt(disc)) / a;
        }
        to_disc = lc < 0 || s_d < s_c;   // tie -> the cylinder
      }
      int lp;
      if (!to_disc) {
        lp = lc;
        Target cyl;
        cyl.kind = cyl_kind;
        cyl.R = r_target;
        int st = propagate_to(fld, cfg, cyl, y, cnt);
        if (st != STOP_NONE) return st;
        lb = cyl_kind == 2 ? lp - 1 : lp;   // crossed inward: the shell below it
        if (std::fabs(y.r[2]) > g.layer_half_z[lp]) continue;   // outside the layer's acceptance: on to the next portal
      } else {
        lp = ld;
        Target pl;
        pl.kind = 0;
        pl.c[0] = 0.0; pl.c[1] = 0.0; pl.c[2] = g.layer_half_z[lp];
        pl.n[0] = 0.0; pl.n[1] = 0.0; pl.n[2] = g.layer_half_z[lp] > 0.0 ? 1.0 : -1.0;
        int st = propagate_to(fld, cfg, pl, y, cnt);
        if (st != STOP_NONE) return st;
        ld = disc_after(lp, y.r[2], y.d[2]);
        const double rho = std::hypot(y.r[0], y.r[1]);
        lb = -1;
        while (lb + 1 < n_barrel && g.layer_r[lb + 1] <= rho) ++lb;
        if (rho < g.layer_r_min[lp] || rho > g.layer_r[lp]) continue;   // outside the disc's acceptance
      }
      // N4: module choice at the portal point, 3x3 around its (phi, z) or (phi, ring) bin
      const int nphi = g.n_phi[lp], nz = g.n_z[lp];
      const double len = 2.0 * g.half_v[g.module_offset[lp]];
      const double phix = std::atan2(y.r[1], y.r[0]);
      int i = (int)std::nearbyint(phix * nphi / (2.0 * PI));
      i = ((i % nphi) + nphi) % nphi;
      const double along = is_disc(lp) ? std::hypot(y.r[0], y.r[1]) - g.layer_r_min[lp] : y.r[2] + g.layer_half_z[lp];
      int j = (int)std::floor(along / len);
      if (j < 0) j = 0;
      if (j > nz - 1) j = nz - 1;
      tgt = pick_in_neighbourhood(g, lp, i, j, -1, y.r, y.d, -1e-3);
      if (tgt >= 0) break;
      // a crack is not a hole: on to the next portal
    }
  }
  // N5: to the target's plane
  const Module k = get_module(g, tgt);
  Target pl;
  pl.kind = 0;
  for (int i = 0; i < 3; ++i) { pl.c[i] = k.c[i]; pl.n[i] = k.n[i]; }
  int st = propagate_to(fld, cfg, pl, y, cnt);
  if (st != STOP_NONE) return st;
  double J[6][6];
  arrive(fld, cfg, k, y, B2F, xp, J);
  transport_cov(J, C, Cp);
  for (int i = 0; i < 6; ++i) {
    if (!std::isfinite(xp[i])) return STOP_NUMERIC;
    for (int j = 0; j < 6; ++j) {
      if (Jout) Jout[i][j] = J[i][j] * (j == 4 ? gE : 1.0);   // d(arrival) / d(parameters before the loss) = J J_E
      if (!std::isfinite(Cp[i][j])) return STOP_NUMERIC;
    }
  }
  target = tgt;
  return STOP_NONE;
}

// ---------------------------------------------------------------------------------- V: visit
// V1: chi2 of measurement (loc, var) against predicted (x, C)
double predicted_chi2(const double x[6], const double C[6][6], const double loc[2], const double var[2]) {
  const double r0 = loc[0] - x[0], r1 = loc[1] - x[1];
  const double S00 = C[0][0] + var[0], S01 = C[0][1], S11 = C[1][1] + var[1];
  const double det = S00 * S11 - S01 * S01;
  return (r0 * r0 * S11 - 2.0 * r0 * r1 * S01 + r1 * r1 * S00) / det;
}

// V3: gain-form update, upper triangle mirrored, phi wrapped to (-pi, pi]
void kalman_update(const double x[6], const double C[6][6], const double loc[2], const double var[2], double xo[6],
                   double Co[6][6]) {
  const double r0 = loc[0] - x[0], r1 = loc[1] - x[1];
  const double S00 = C[0][0] + var[0], S01 = C[0][1], S11 = C[1][1] + var[1];
  const double det = S00 * S11 - S01 * S01;
  const double I00 = S11 / det, I01 = -S01 / det, I11 = S00 / det;
  double K[6][2];
  for (int i = 0; i < 6; ++i) {
    K[i][0] = C[i][0] * I00 + C[i][1] * I01;
    K[i][1] = C[i][0] * I01 + C[i][1] * I11;
  }
  for (int i = 0; i < 6; ++i) xo[i] = x[i] + K[i][0] * r0 + K[i][1] * r1;
  for (int i = 0; i < 6; ++i)
    for (int j = i; j < 6; ++j) {
      const double v = C[i][j] - (K[i][0] * C[0][j] + K[i][1] * C[1][j]);
      Co[i][j] = v;
      Co[j][i] = v;
    }
  while (xo[2] > PI) xo[2] -= 2.0 * PI;
  while (xo[2] <= -PI) xo[2] += 2.0 * PI;
}

// ---------------------------------------------------------------------------------- R: CKF control
struct Link {
  int parent;   // index into the seed's link vector, -1 = root
  int meas;     // measurement index, -1 = hole
  double chi2;
};

struct Tip {
  double x[6], C[6][6];
  int module;
  int link;        // last link (-1 before level 0)
  int n_meas, n_holes;
  double chi2_sum;
  // snapshot at the last measurement (V3)
  double xs[6], Cs[6][6];
  int module_s;
};

struct Track {
  int seed, n_holes, last_module, stop_reason;
  double x[6], C[6][6], chi2_sum;
  std::vector<int> meas;
  std::vector<double> chi2;
};

struct Sel { double chi2; int idx; };

void run_seed(const OGeometry& g, const OField& fld, const OConfig& cfg, const int32_t* moff, const double* loc,
              const double* var, int seed, int seed_module, const double* sx, const double* sC,
              std::vector<Track>& out, Counters& cnt) {
  std::vector<Link> links;
  std::vector<Tip> tips(1);
  {
    Tip& t = tips[0];
    for (int i = 0; i < 6; ++i) {
      t.x[i] = sx[i];
      for (int j = 0; j < 6; ++j) t.C[i][j] = sC[6 * i + j];
    }
    t.module = seed_module; t.link = -1; t.n_meas = 0; t.n_holes = 0; t.chi2_sum = 0.0; t.module_s = -1;
    std::memset(t.xs, 0, sizeof(t.xs)); std::memset(t.Cs, 0, sizeof(t.Cs));
  }
  int finished = 0;
  auto emit = [&](const Tip& t, int reason) {
    ++finished;
    if (t.n_meas < cfg.min_measurements) return;
    Track tr;
    tr.seed = seed; tr.n_holes = t.n_holes; tr.last_module = t.module_s; tr.stop_reason = reason;
    std::memcpy(tr.x, t.xs, sizeof(tr.x)); std::memcpy(tr.C, t.Cs, sizeof(tr.C));
    tr.chi2_sum = t.chi2_sum;
    for (int l = t.link; l >= 0; l = links[l].parent)
      if (links[l].meas >= 0) { tr.meas.push_back(links[l].meas); tr.chi2.push_back(links[l].chi2); }
    std::reverse(tr.meas.begin(), tr.meas.end());
    std::reverse(tr.chi2.begin(), tr.chi2.end());
    out.push_back(std::move(tr));
  };

  for (int level = 0; !tips.empty(); ++level) {
    if (level >= cfg.max_levels) {
      for (const Tip& t : tips) emit(t, STOP_LEVEL_LIMIT);
      break;
    }
    const int n = (int)tips.size();
    cnt.tips += n;
    // ---- step A: move every tip to its next module (level 0: N6, the seed's own module, J = I)
    std::vector<int> stop(n, STOP_NONE), target(n, -1);
    std::vector<Tip> pred(tips);
    for (int i = 0; i < n; ++i) {
      if (level == 0) {
        const Tip& t = tips[i];
        bool ok = (t.x[3] > 0.0 && t.x[3] < PI);
        for (int a = 0; a < 6; ++a) ok = ok && std::isfinite(t.x[a]);
        if (!ok) stop[i] = STOP_NUMERIC;
        target[i] = t.module;
        continue;
      }
      int tg = -1;
      stop[i] = move_to_next_module(g, fld, cfg, tips[i].module, tips[i].x, tips[i].C, tg, pred[i].x, pred[i].C,
                                    nullptr, cnt);
      target[i] = tg;
    }
    // ---- step B: gate (V1, V2) -> wanted children
    std::vector<std::vector<Sel>> sel(n);
    std::vector<int> want(n, 0);
    for (int i = 0; i < n; ++i) {
      if (stop[i] != STOP_NONE) continue;
      ++cnt.visits;
      const int m = target[i];
      std::vector<Sel> pass;
      for (int k = moff[m]; k < moff[m + 1]; ++k) {
        ++cnt.gate_tests;
        const double c2 = predicted_chi2(pred[i].x, pred[i].C, loc + 2 * k, var + 2 * k);
        if (c2 < cfg.chi2_max) pass.push_back({c2, k});
      }
      std::stable_sort(pass.begin(), pass.end(), [](const Sel& a, const Sel& b) {
        return a.chi2 < b.chi2 || (a.chi2 == b.chi2 && a.idx < b.idx);
      });
      if ((int)pass.size() > cfg.max_branches_per_surface) pass.resize(cfg.max_branches_per_surface);
      if (pass.empty()) {
        // V4: hole
        if (tips[i].n_holes + 1 > cfg.max_holes) { stop[i] = STOP_HOLES; pred[i].n_holes = tips[i].n_holes + 1; }
        else want[i] = 1;
      } else {
        want[i] = (int)pass.size();
      }
      sel[i] = std::move(pass);
    }
    // ---- step C: per-seed cap (R10), greedy in tip order
    const int Rm = cfg.max_candidates_per_seed - (finished + n);
    long long P = 0;
    std::vector<int> keep(n, 0);
    for (int i = 0; i < n; ++i) {
      if (want[i] < 1) continue;
      const int e = want[i] - 1;
      const long long room = std::max<long long>(0, (long long)Rm - P);
      keep[i] = 1 + (int)std::min<long long>(e, room);
      P += e;
    }
    // ---- step D: finished tips emit (tip order), children are made (V3, V4)
    std::vector<Tip> next;
    for (int i = 0; i < n; ++i) {
      if (stop[i] != STOP_NONE) {
        Tip t = tips[i];
        if (stop[i] == STOP_HOLES) t.n_holes = pred[i].n_holes;
        emit(t, stop[i]);
        continue;
      }
      const int m = target[i];
      if (sel[i].empty()) {
        Tip c = pred[i];
        c.module = m;
        links.push_back({tips[i].link, -1, 0.0});
        c.link = (int)links.size() - 1;
        c.n_holes = tips[i].n_holes + 1;
        next.push_back(c);
        continue;
      }
      for (int j = 0; j < keep[i]; ++j) {
        Tip c = pred[i];
        const int k = sel[i][j].idx;
        kalman_update(pred[i].x, pred[i].C, loc + 2 * k, var + 2 * k, c.x, c.C);
        ++cnt.updates;
        c.module = m;
        links.push_back({tips[i].link, k, sel[i][j].chi2});
        c.link = (int)links.size() - 1;
        c.n_meas = tips[i].n_meas + 1;
        c.chi2_sum = tips[i].chi2_sum + sel[i][j].chi2;
        std::memcpy(c.xs, c.x, sizeof(c.x));
        std::memcpy(c.Cs, c.C, sizeof(c.C));
        c.module_s = m;
        next.push_back(c);
      }
    }
    tips.swap(next);
  }
}

// ====================================================================================== K: KF fit + RTS smoother
// "a Kalman Filter-based fitting [8], which runs a smoothing algorithm called the
// Rauch-Tung-Striebel (RTS) smoother [19], is applied additionally to the tracks to make all track parameters
// consider all measurements in the pattern"; the parameters at the FIRST measurement are the ones it names as
// wanted (vertex reconstruction).  The paper prints no formula; rules K1-K5 of DESIGN.md §3 restate the
// textbook filter/smoother of its refs [8], [19] on top of the P/J/N/V rules above.
//
// One visited module = one STATE: predicted (xp, Cp), filtered (xf, Cf), the bound->bound Jacobian J that made
// the prediction from the previous state's filtered one, and the measurement used (-1 = passed without one).
struct FitState {
  int module, meas;
  double chi2;
  double xp[6], Cp[6][6], xf[6], Cf[6][6], J[6][6];
  double qphi, qtheta;  // V5 variances added on leaving the PREVIOUS state (what made Cp = J (Cf + Q) J^T); 0 at state 0
};

// K2: forward filter = the CKF's own path with the branch choice replaced by the candidate's list: state 0 is the
// seed's module with the seed's (x, C) (N6); on every visited module the next unconsumed measurement of the list
// is used iff it lives on that module (V1 chi2, V3 update), otherwise the module is passed (filtered =
// predicted); then the N-rules move on (V5 material on leaving, J1-J5).  Ends when the list is consumed.
int fit_forward(const OGeometry& g, const OField& fld, const OConfig& cfg, const int32_t* moff, const double* loc,
                const double* var, int seed_module, const double* sx, const double* sC, const int32_t* meas, int n_meas,
                std::vector<FitState>& st, Counters& cnt) {
  double x[6], C[6][6];
  for (int i = 0; i < 6; ++i) {
    x[i] = sx[i];
    for (int j = 0; j < 6; ++j) C[i][j] = sC[6 * i + j];
  }
  int module = seed_module, next = 0;
  if (n_meas < 1) return STOP_NONE;
  for (int level = 0;; ++level) {
    if (level >= cfg.max_levels) return STOP_LEVEL_LIMIT;
    FitState s;
    if (level == 0) {
      bool ok = (x[3] > 0.0 && x[3] < PI);
      for (int a = 0; a < 6; ++a) ok = ok && std::isfinite(x[a]);
      if (!ok) return STOP_NUMERIC;
      std::memcpy(s.xp, x, sizeof(x));
      std::memcpy(s.Cp, C, sizeof(C));
      for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) s.J[i][j] = (i == j) ? 1.0 : 0.0;
      s.module = module;
      s.qphi = 0.0; s.qtheta = 0.0;
    } else {
      int tg = -1;
      {
        double Q[6][6];
        std::memset(Q, 0, sizeof(Q));
        add_material(cfg, get_module(g, module), x, Q);
        s.qphi = Q[2][2]; s.qtheta = Q[3][3];
      }
      const int stop = move_to_next_module(g, fld, cfg, module, x, C, tg, s.xp, s.Cp, s.J, cnt);
      if (stop != STOP_NONE) return stop;
      s.module = tg;
    }
    const int k = meas[next];
    if (k >= moff[s.module] && k < moff[s.module + 1]) {
      s.meas = k;
      s.chi2 = predicted_chi2(s.xp, s.Cp, loc + 2 * k, var + 2 * k);
      kalman_update(s.xp, s.Cp, loc + 2 * k, var + 2 * k, s.xf, s.Cf);
      ++next;
    } else {
      s.meas = -1;
      s.chi2 = 0.0;
      std::memcpy(s.xf, s.xp, sizeof(s.xp));
      std::memcpy(s.Cf, s.Cp, sizeof(s.Cp));
    }
    st.push_back(s);
    if (next == n_meas) return STOP_NONE;
    std::memcpy(x, s.xf, sizeof(x));
    std::memcpy(C, s.Cf, sizeof(C));
    module = s.module;
  }
}

// K4 helper: X = G^-1 B for a symmetric positive definite 6x6 G, by diagonal scaling (G_ii -> 1; the bound
// covariance mixes mm^2, rad^2 and GeV^-2, 10 orders of magnitude apart) and Cholesky G' = L L^T.
// Returns false when G is not positive definite.
bool spd_solve6(const double G[6][6], const double B[6][6], double X[6][6]) {
  double s[6], L[6][6];
  for (int i = 0; i < 6; ++i) {
    if (!(G[i][i] > 0.0)) return false;
    s[i] = 1.0 / std::sqrt(G[i][i]);
  }
  for (int j = 0; j < 6; ++j) {
    double d = G[j][j] * s[j] * s[j];
    for (int k = 0; k < j; ++k) d -= L[j][k] * L[j][k];
    if (!(d > 0.0)) return false;
    L[j][j] = std::sqrt(d);
    for (int i = j + 1; i < 6; ++i) {
      double v = G[i][j] * s[i] * s[j];
      for (int k = 0; k < j; ++k) v -= L[i][k] * L[j][k];
      L[i][j] = v / L[j][j];
    }
  }
  for (int c = 0; c < 6; ++c) {
    double z[6], w[6];
    for (int i = 0; i < 6; ++i) {  // L z = S b
      double v = B[i][c] * s[i];
      for (int k = 0; k < i; ++k) v -= L[i][k] * z[k];
      z[i] = v / L[i][i];
    }
    for (int i = 5; i >= 0; --i) {  // L^T w = z
      double v = z[i];
      for (int k = i + 1; k < 6; ++k) v -= L[k][i] * w[k];
      w[i] = v / L[i][i];
    }
    for (int i = 0; i < 6; ++i) X[i][c] = w[i] * s[i];
  }
  return true;
}

inline double wrap_pi(double a) {
  while (a > PI) a -= 2.0 * PI;
  while (a <= -PI) a += 2.0 * PI;
  return a;
}

// K4: RTS backward recursion [19] over states 0..n-1.  xs[n-1] = xf[n-1]; for k = n-2..0:
//   A_k = Cf[k] J[k+1]^T Cp[k+1]^-1;  xs[k] = xf[k] + A_k (xs[k+1] - xp[k+1]);
//   Cs[k] = Cf[k] + A_k (Cs[k+1] - Cp[k+1]) A_k^T   (symmetrised).
// The process noise (V5) enters Cp[k+1] = J (Cf[k] + Q_k) J^T only; the gain uses Cf[k] without it, because the
// noise of the step k -> k+1 is independent of state k.  Angle differences and results are wrapped to (-pi, pi].
bool rts_smooth(int n, const FitState* st, double (*xs)[6], double (*Cs)[6][6]) {
  if (n < 1) return true;
  std::memcpy(xs[n - 1], st[n - 1].xf, sizeof(double) * 6);
  std::memcpy(Cs[n - 1], st[n - 1].Cf, sizeof(double) * 36);
  for (int k = n - 2; k >= 0; --k) {
    const FitState& a = st[k];
    const FitState& b = st[k + 1];
    double M[6][6], X[6][6];  // M = J Cf[k];  X = Cp[k+1]^-1 M = A_k^T
    for (int i = 0; i < 6; ++i)
      for (int j = 0; j < 6; ++j) {
        double v = 0.0;
        for (int l = 0; l < 6; ++l) v += b.J[i][l] * a.Cf[l][j];
        M[i][j] = v;
      }
    if (!spd_solve6(b.Cp, M, X)) return false;
    double dx[6], dC[6][6], T[6][6];
    for (int i = 0; i < 6; ++i) dx[i] = xs[k + 1][i] - b.xp[i];
    dx[2] = wrap_pi(dx[2]);
    for (int i = 0; i < 6; ++i) {
      double v = 0.0;
      for (int j = 0; j < 6; ++j) v += X[j][i] * dx[j];
      xs[k][i] = a.xf[i] + v;
    }
    xs[k][2] = wrap_pi(xs[k][2]);
    for (int i = 0; i < 6; ++i)
      for (int j = 0; j < 6; ++j) dC[i][j] = Cs[k + 1][i][j] - b.Cp[i][j];
    for (int i = 0; i < 6; ++i)   // T = dC X
      for (int j = 0; j < 6; ++j) {
        double v = 0.0;
        for (int l = 0; l < 6; ++l) v += dC[i][l] * X[l][j];
        T[i][j] = v;
      }
    double R[6][6];
    for (int i = 0; i < 6; ++i)   // R = X^T T
      for (int j = 0; j < 6; ++j) {
        double v = 0.0;
        for (int l = 0; l < 6; ++l) v += X[l][i] * T[l][j];
        R[i][j] = a.Cf[i][j] + v;
      }
    for (int i = 0; i < 6; ++i)
      for (int j = 0; j < 6; ++j) Cs[k][i][j] = 0.5 * (R[i][j] + R[j][i]);
  }
  return true;
}

// K4': two-filter ("optimal") smoother, the variant PAPER.md:100 names as the more stable one [23, 24]: the smoothed
// state is the combination of the forward-filtered state with the information a BACKWARD filter has gathered from
// the later measurements.  It is run on the same linearised model as the RTS recursion (the stored J, xp, xf, Cf and
// the V5 noise), in deviations d_k = z_k - xf[k], so it needs no second propagation and must give the RTS result
// (pinned).  No difference of nearly equal covariances appears anywhere.
//   backward information (Y, y) about d_k from the measurements of the states after k; (0, 0) at the last state;
//   smoothed: Cf = B B^T (scaled Cholesky);  A = I + B^T Y B;  Cs = B A^-1 B^T;  xs = xf + B A^-1 B^T y;
//   step k -> k-1: add the measurement of state k (Y += H^T V^-1 H, y += H^T V^-1 (m - H xf[k]));
//     d_k = c + J (d_{k-1} + u), c = xp[k] - xf[k], u ~ N(0, Q) on (phi, theta):  Yz = J^T Y J, yz = J^T (y - Y c);
//     marginalise u:  Y' = Yz - Yz G (Qr^-1 + G^T Yz G)^-1 G^T Yz,  y' likewise  (2 x 2 inverse).
bool two_filter_smooth(int n, const FitState* st, const double* loc, const double* var, double (*xs)[6],
                       double (*Cs)[6][6]) {
  double Y[6][6], y[6];
  std::memset(Y, 0, sizeof(Y));
  std::memset(y, 0, sizeof(y));
  for (int k = n - 1; k >= 0; --k) {
    const FitState& a = st[k];
    // ---- smoothed state k
    double s[6], L[6][6], B[6][6];
    std::memset(L, 0, sizeof(L));
    for (int i = 0; i < 6; ++i) {
      if (!(a.Cf[i][i] > 0.0)) return false;
      s[i] = 1.0 / std::sqrt(a.Cf[i][i]);
    }
    for (int j = 0; j < 6; ++j) {  // Cholesky of S Cf S
      double d = a.Cf[j][j] * s[j] * s[j];
      for (int l = 0; l < j; ++l) d -= L[j][l] * L[j][l];
      if (!(d > 0.0)) return false;
      L[j][j] = std::sqrt(d);
      for (int i = j + 1; i < 6; ++i) {
        double v = a.Cf[i][j] * s[i] * s[j];
        for (int l = 0; l < j; ++l) v -= L[i][l] * L[j][l];
        L[i][j] = v / L[j][j];
      }
    }
    for (int i = 0; i < 6; ++i)
      for (int j = 0; j < 6; ++j) B[i][j] = L[i][j] / s[i];  // Cf = B B^T, B lower triangular
    double A[6][6], YB[6][6], t[6];
    for (int i = 0; i < 6; ++i)
      for (int j = 0; j < 6; ++j) {
        double v = 0.0;
        for (int l = 0; l < 6; ++l) v += Y[i][l] * B[l][j];
        YB[i][j] = v;
      }
    for (int i = 0; i < 6; ++i) {
      for (int j = 0; j < 6; ++j) {
        double v = (i == j) ? 1.0 : 0.0;
        for (int l = 0; l < 6; ++l) v += B[l][i] * YB[l][j];
        A[i][j] = v;
      }
      double v = 0.0;
      for (int l = 0; l < 6; ++l) v += B[l][i] * y[l];
      t[i] = v;
    }
    // X = A^-1 [B^T | t]: A is symmetric, >= I
    double R[6][6], Xm[6][6];
    for (int i = 0; i < 6; ++i)
      for (int j = 0; j < 6; ++j) R[i][j] = B[j][i];  // B^T
    if (!spd_solve6(A, R, Xm)) return false;   // Xm = A^-1 B^T
    double tt[6][6], Xt[6][6];
    for (int i = 0; i < 6; ++i)
      for (int j = 0; j < 6; ++j) tt[i][j] = (j == 0) ? t[i] : 0.0;
    if (!spd_solve6(A, tt, Xt)) return false;  // first column = A^-1 t
    for (int i = 0; i < 6; ++i) {
      double v = 0.0;
      for (int l = 0; l < 6; ++l) v += B[i][l] * Xt[l][0];
      xs[k][i] = a.xf[i] + v;
    }
    xs[k][2] = wrap_pi(xs[k][2]);
    double Rm[6][6];
    for (int i = 0; i < 6; ++i)
      for (int j = 0; j < 6; ++j) {
        double v = 0.0;
        for (int l = 0; l < 6; ++l) v += B[i][l] * Xm[l][j];
        Rm[i][j] = v;
      }
    for (int i = 0; i < 6; ++i)
      for (int j = 0; j < 6; ++j) Cs[k][i][j] = 0.5 * (Rm[i][j] + Rm[j][i]);
    if (k == 0) break;
    // ---- backward step k -> k - 1
    if (a.meas >= 0) {
      const double* m = loc + 2 * a.meas;
      const double* v = var + 2 * a.meas;
      for (int c = 0; c < 2; ++c) {
        Y[c][c] += 1.0 / v[c];
        y[c] += (m[c] - a.xf[c]) / v[c];
      }
    }
    double c6[6], yc[6];
    for (int i = 0; i < 6; ++i) c6[i] = a.xp[i] - a.xf[i];
    c6[2] = wrap_pi(c6[2]);
    for (int i = 0; i < 6; ++i) {
      double v = y[i];
      for (int l = 0; l < 6; ++l) v -= Y[i][l] * c6[l];
      yc[i] = v;
    }
    double YJ[6][6], Yz[6][6], yz[6];
    for (int i = 0; i < 6; ++i)
      for (int j = 0; j < 6; ++j) {
        double v = 0.0;
        for (int l = 0; l < 6; ++l) v += Y[i][l] * a.J[l][j];
        YJ[i][j] = v;
      }
    for (int i = 0; i < 6; ++i) {
      for (int j = 0; j < 6; ++j) {
        double v = 0.0;
        for (int l = 0; l < 6; ++l) v += a.J[l][i] * YJ[l][j];
        Yz[i][j] = v;
      }
      double v = 0.0;
      for (int l = 0; l < 6; ++l) v += a.J[l][i] * yc[l];
      yz[i] = v;
    }
    for (int i = 0; i < 6; ++i)
      for (int j = i + 1; j < 6; ++j) { const double m2 = 0.5 * (Yz[i][j] + Yz[j][i]); Yz[i][j] = m2; Yz[j][i] = m2; }
    if (a.qphi > 0.0 && a.qtheta > 0.0) {
      const double s00 = 1.0 / a.qphi + Yz[2][2], s01 = Yz[2][3], s11 = 1.0 / a.qtheta + Yz[3][3];
      const double det = s00 * s11 - s01 * s01;
      if (!(det > 0.0)) return false;
      const double i00 = s11 / det, i01 = -s01 / det, i11 = s00 / det;
      double K2[6], K3[6];   // Kg = Yz G Sg^-1
      for (int i = 0; i < 6; ++i) {
        K2[i] = Yz[i][2] * i00 + Yz[i][3] * i01;
        K3[i] = Yz[i][2] * i01 + Yz[i][3] * i11;
      }
      for (int i = 0; i < 6; ++i) {
        for (int j = 0; j < 6; ++j) Y[i][j] = Yz[i][j] - (K2[i] * Yz[2][j] + K3[i] * Yz[3][j]);
        y[i] = yz[i] - (K2[i] * yz[2] + K3[i] * yz[3]);
      }
      for (int i = 0; i < 6; ++i)
        for (int j = i + 1; j < 6; ++j) { const double m2 = 0.5 * (Y[i][j] + Y[j][i]); Y[i][j] = m2; Y[j][i] = m2; }
    } else {
      std::memcpy(Y, Yz, sizeof(Y));
      std::memcpy(y, yz, sizeof(y));
    }
  }
  return true;
}

struct Result {
  std::vector<Track> tracks;
  Counters cnt;
};

// ====================================================================================== AR: ambiguity resolution
// PAPER.md:98 (section 4): "Duplicate tracks arise when multiple tracks share the same or very similar hit patterns ...
// an additional algorithm -- known as ambiguity resolution -- will be integrated into the reconstruction chain to
// remove such tracks after the CKF stage."  The paper names the stage and gives no algorithm; rules AR1-AR3 of
// DESIGN.md 3 (readings) define a greedy shared-hit resolver over the candidates ckf_find reported:
//   AR1  a candidate's quality key is (number of measurements DESCENDING, chi2 sum rounded to float32 ASCENDING,
//        candidate index ASCENDING): longer first, then better chi2; the index makes the order total.
//   AR2  candidates are visited in that order; a measurement belongs to the first ACCEPTED candidate that holds it.
//   AR3  a candidate is accepted iff the number s of its measurements that already belong to accepted candidates
//        satisfies s <= max_shared_hits and s <= max_shared_fraction * n_meas; an accepted candidate then takes its
//        free measurements; a rejected one takes nothing.
// Written out as exactly that loop.
void resolve_ambiguity(int n_tracks, const int32_t* offsets, const int32_t* meas, const double* chi2_sum, int n_meas_total,
                       int max_shared_hits, double max_shared_fraction, int32_t* accepted, int32_t* n_shared) {
  std::vector<int> order(n_tracks);
  for (int t = 0; t < n_tracks; ++t) order[t] = t;
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) {
    const int na = offsets[a + 1] - offsets[a], nb = offsets[b + 1] - offsets[b];
    if (na != nb) return na > nb;
    const float ca = (float)chi2_sum[a], cb = (float)chi2_sum[b];
    if (ca != cb) return ca < cb;
    return a < b;
  });
  std::vector<int> owner(n_meas_total, -1);
  for (int k = 0; k < n_tracks; ++k) {
    const int t = order[k];
    const int n = offsets[t + 1] - offsets[t];
    int s = 0;
    for (int e = offsets[t]; e < offsets[t + 1]; ++e)
      if (owner[meas[e]] >= 0) ++s;
    const bool ok = s <= max_shared_hits && (double)s <= max_shared_fraction * (double)n;
    accepted[t] = ok ? 1 : 0;
    n_shared[t] = s;
    if (ok)
      for (int e = offsets[t]; e < offsets[t + 1]; ++e)
        if (owner[meas[e]] < 0) owner[meas[e]] = t;
  }
}

}  // namespace

thread_local long long g_last_move_trials = 0;

// ====================================================================================== S: seeding + parameter estimation
// "The spacepoints are used in the seeding algorithm where triplets, a set of three spacepoints which can
// approximately form a helix, are found.  In the track parameter estimation algorithm, the position and momentum of
// tracks, called a seed, are estimated at the first spacepoint using the helix model."  The paper gives no cut and no
// formula; rules S0-S6 of DESIGN.md 3 (readings) are written out here as plain loops over all combinations.
struct OSeedConfig {
  int32_t layer_b, layer_m, layer_t;   // barrel layers of the bottom / middle / top spacepoint
  double dphi_max;     // S1: |phi_outer - phi_inner| of a doublet
  double cot_max;      // S1: |cot theta| of a doublet
  double z0_max;       // S1: |z at rho = 0| of a doublet's straight line in (rho, z)
  double dcot_max;     // S2: |cot theta (bottom, middle) - cot theta (middle, top)|
  double pt_min;       // S3: transverse momentum of the circle through the three points, GeV
  double d0_max;       // S4: distance of that circle from the z axis, mm
  double sigma_angle;  // S6: phi / theta standard deviation of a seed, rad
  double rel_sigma_qop;  // S6: relative standard deviation of q/p added to the sagitta-resolution term
  double cov_scale;    // S6: inflation of every variance (BASELINE seeds: 10)
};

struct SeedOut {
  int b, m, t;   // measurement indices
  int module;
  double x[6], C[36];
};

struct SpacePoint { int meas; double x, y, z, rho, phi; };

// S0: spacepoints of one layer = global positions of its measurements
std::vector<SpacePoint> layer_spacepoints(const OGeometry& g, int layer, const int32_t* moff, const double* loc) {
  std::vector<SpacePoint> out;
  for (int id = g.module_offset[layer]; id < g.module_offset[layer + 1]; ++id) {
    const Module k = get_module(g, id);
    for (int i = moff[id]; i < moff[id + 1]; ++i) {
      SpacePoint p;
      p.meas = i;
      p.x = k.c[0] + loc[2 * i] * k.u[0] + loc[2 * i + 1] * k.v[0];
      p.y = k.c[1] + loc[2 * i] * k.u[1] + loc[2 * i + 1] * k.v[1];
      p.z = k.c[2] + loc[2 * i] * k.u[2] + loc[2 * i + 1] * k.v[2];
      p.rho = std::hypot(p.x, p.y);
      p.phi = std::atan2(p.y, p.x);
      out.push_back(p);
    }
  }
  return out;
}

// S1: doublet (inner, outer) -> cot theta, or false
bool doublet_ok(const OSeedConfig& c, const SpacePoint& in, const SpacePoint& out, double& cot) {
  double dphi = out.phi - in.phi;
  while (dphi > PI) dphi -= 2.0 * PI;
  while (dphi <= -PI) dphi += 2.0 * PI;
  if (!(std::fabs(dphi) <= c.dphi_max)) return false;
  const double drho = out.rho - in.rho;
  if (!(drho > 0.0)) return false;
  cot = (out.z - in.z) / drho;
  if (!(std::fabs(cot) <= c.cot_max)) return false;
  const double z0 = in.z - in.rho * cot;
  return std::fabs(z0) <= c.z0_max;
}

// S3-S6 for one triplet that passed S1, S2: false if a cut fails
bool triplet_seed(const OGeometry& g, const OField& fld, const OSeedConfig& c, const int32_t* meas_module,
                  const double* loc, const double* var, const SpacePoint& B, const SpacePoint& M, const SpacePoint& T,
                  SeedOut& s) {
  // S3: circle through the three transverse points
  const double d = 2.0 * (B.x * (M.y - T.y) + M.x * (T.y - B.y) + T.x * (B.y - M.y));
  if (d == 0.0) return false;   // exactly collinear: no curvature to estimate
  const double b2 = B.x * B.x + B.y * B.y, m2 = M.x * M.x + M.y * M.y, t2 = T.x * T.x + T.y * T.y;
  const double xc = (b2 * (M.y - T.y) + m2 * (T.y - B.y) + t2 * (B.y - M.y)) / d;
  const double yc = (b2 * (T.x - M.x) + m2 * (B.x - T.x) + t2 * (M.x - B.x)) / d;
  const double R = std::hypot(B.x - xc, B.y - yc);
  const double rB[3] = {B.x, B.y, B.z};
  double Bf[3];
  field_at(fld, rB, Bf);
  const double pt = KAPPA * std::fabs(Bf[2]) * R;
  if (!(pt >= c.pt_min)) return false;
  // S4: distance of the circle from the z axis
  if (!(std::fabs(std::hypot(xc, yc) - R) <= c.d0_max)) return false;
  // S5: helix parameters at the bottom spacepoint
  double tx = -(B.y - yc) / R, ty = (B.x - xc) / R;   // tangent, oriented toward the middle point
  if (tx * (M.x - B.x) + ty * (M.y - B.y) < 0.0) { tx = -tx; ty = -ty; }
  const double cz = (M.x - B.x) * (T.y - M.y) - (M.y - B.y) * (T.x - M.x);   // turning sense of B -> M -> T
  const double q = (cz * Bf[2] < 0.0) ? 1.0 : -1.0;      // a positive charge turns clockwise in a field along +z (P1)
  const double chord = std::hypot(T.x - B.x, T.y - B.y);
  const double arc = 2.0 * R * std::asin(std::min(1.0, chord / (2.0 * R)));
  const double cot = (T.z - B.z) / arc;
  const double theta = std::atan2(1.0, cot);
  s.b = B.meas; s.m = M.meas; s.t = T.meas;
  s.module = meas_module[B.meas];
  s.x[0] = loc[2 * B.meas]; s.x[1] = loc[2 * B.meas + 1];
  s.x[2] = std::atan2(ty, tx);
  s.x[3] = theta;
  s.x[4] = q * std::sin(theta) / pt;
  s.x[5] = 0.0;
  // S6: diagonal covariance
  for (int i = 0; i < 36; ++i) s.C[i] = 0.0;
  s.C[0] = c.cov_scale * var[2 * B.meas];
  s.C[7] = c.cov_scale * var[2 * B.meas + 1];
  s.C[14] = c.cov_scale * c.sigma_angle * c.sigma_angle;
  s.C[21] = c.cov_scale * c.sigma_angle * c.sigma_angle;
  // q/p: what three points resolve -- the sagitta sag = M - (B + T) / 2 across the chord L has variance
  // var_M + (var_B + var_T) / 4 in the measured transverse coordinate, 1/R = 8 sag / L^2 -- plus a relative term for
  // the scattering between the layers
  const double var_sag = var[2 * M.meas] + 0.25 * (var[2 * B.meas] + var[2 * T.meas]);
  const double dcurv = 8.0 * std::sqrt(var_sag) / (chord * chord);                    // sigma(1/R), 1/mm
  const double sq_res = std::sin(theta) * dcurv / (KAPPA * std::fabs(Bf[2]));          // sigma(q/p) from the resolution
  s.C[28] = c.cov_scale * (sq_res * sq_res + (c.rel_sigma_qop * s.x[4]) * (c.rel_sigma_qop * s.x[4]));
  s.C[35] = 1.0;
  (void)g;
  return true;
}

struct SeedResult { std::vector<SeedOut> seeds; };

// ====================================================================================== C interface
extern "C" {

struct oracle_result;

// Runs the CKF over all seeds (static contiguous chunks over n_threads).  All pointers are HOST, double.
void* oracle_ckf_find(const OGeometry* g, const OField* f, const OConfig* cfg, int32_t n_meas,
                      const int32_t* module_offsets, const double* loc, const double* var, int32_t n_seeds,
                      const int32_t* seed_module, const double* seed_params, const double* seed_cov,
                      int32_t n_threads) {
  (void)n_meas;
  if (n_threads < 1) n_threads = 1;
  if (n_threads > n_seeds) n_threads = std::max(1, n_seeds);
  std::vector<std::vector<Track>> parts(n_threads);
  std::vector<Counters> cnts(n_threads);
  auto work = [&](int t) {
    const long long lo = (long long)n_seeds * t / n_threads, hi = (long long)n_seeds * (t + 1) / n_threads;
    for (long long s = lo; s < hi; ++s)
      run_seed(*g, *f, *cfg, module_offsets, loc, var, (int)s, seed_module[s], seed_params + 6 * s,
               seed_cov + 36 * s, parts[t], cnts[t]);
  };
  if (n_threads == 1) work(0);
  else {
    std::vector<std::thread> th;
    for (int t = 0; t < n_threads; ++t) th.emplace_back(work, t);
    for (auto& x : th) x.join();
  }
  Result* R = new Result();
  for (int t = 0; t < n_threads; ++t) {
    for (auto& tr : parts[t]) R->tracks.push_back(std::move(tr));
    R->cnt.visits += cnts[t].visits; R->cnt.rk_trials += cnts[t].rk_trials;
    R->cnt.rk_accepted += cnts[t].rk_accepted; R->cnt.gate_tests += cnts[t].gate_tests;
    R->cnt.updates += cnts[t].updates; R->cnt.tips += cnts[t].tips;
  }
  return R;
}

int32_t oracle_result_n_tracks(const void* r) { return (int32_t)((const Result*)r)->tracks.size(); }
int64_t oracle_result_n_entries(const void* r) {
  int64_t n = 0;
  for (const auto& t : ((const Result*)r)->tracks) n += (int64_t)t.meas.size();
  return n;
}
void oracle_result_counters(const void* r, int64_t out[6]) {
  const Counters& c = ((const Result*)r)->cnt;
  out[0] = c.visits; out[1] = c.rk_trials; out[2] = c.rk_accepted; out[3] = c.gate_tests; out[4] = c.updates;
  out[5] = c.tips;
}
void oracle_result_copy(const void* r, int32_t* track_offsets, int32_t* meas_idx, double* entry_chi2, int32_t* seed_id,
                        int32_t* n_holes, int32_t* last_module, int32_t* stop_reason, double* params, double* cov,
                        double* chi2_sum) {
  const Result* R = (const Result*)r;
  int32_t off = 0;
  for (size_t t = 0; t < R->tracks.size(); ++t) {
    const Track& tr = R->tracks[t];
    track_offsets[t] = off;
    for (size_t k = 0; k < tr.meas.size(); ++k) { meas_idx[off + k] = tr.meas[k]; entry_chi2[off + k] = tr.chi2[k]; }
    off += (int32_t)tr.meas.size();
    seed_id[t] = tr.seed; n_holes[t] = tr.n_holes; last_module[t] = tr.last_module; stop_reason[t] = tr.stop_reason;
    for (int i = 0; i < 6; ++i) {
      params[6 * t + i] = tr.x[i];
      for (int j = 0; j < 6; ++j) cov[36 * t + 6 * i + j] = tr.C[i][j];
    }
    chi2_sum[t] = tr.chi2_sum;
  }
  track_offsets[R->tracks.size()] = off;
}
void oracle_result_free(void* r) { delete (Result*)r; }

// ---- K: KF fit + RTS smoother over candidates given as a CSR list (the layout ckf_find reports).
// Per track: status (0 = fitted, else the stop reason of the forward pass, or STOP_NUMERIC when a predicted
// covariance is not positive definite), number of states, forward chi2 sum, the forward-filtered state at the
// last measurement (K2: equals the CKF candidate's), the smoothed covariance at the first measurement; per
// entry (measurement of the list): the smoothed parameters at that measurement's state.
void oracle_kf_fit(const OGeometry* g, const OField* f, const OConfig* cfg, const int32_t* module_offsets,
                   const double* loc, const double* var, const int32_t* seed_module, const double* seed_params,
                   const double* seed_cov, int32_t n_tracks, const int32_t* track_offsets, const int32_t* meas_idx,
                   const int32_t* seed_id, int32_t n_threads, int32_t* status, int32_t* n_states, double* chi2_sum,
                   double* last_x, double* last_C, double* first_C, double* entry_xs, int32_t smoother) {
  if (n_threads < 1) n_threads = 1;
  if (n_threads > n_tracks) n_threads = std::max(1, n_tracks);
  auto work = [&](int t) {
    const long long lo = (long long)n_tracks * t / n_threads, hi = (long long)n_tracks * (t + 1) / n_threads;
    Counters cnt;
    std::vector<FitState> st;
    std::vector<double> xs, Cs;
    for (long long tr = lo; tr < hi; ++tr) {
      const int e0 = track_offsets[tr], n = track_offsets[tr + 1] - e0, sd = seed_id[tr];
      st.clear();
      int rc = fit_forward(*g, *f, *cfg, module_offsets, loc, var, seed_module[sd], seed_params + 6 * sd,
                           seed_cov + 36 * sd, meas_idx + e0, n, st, cnt);
      const int ns = (int)st.size();
      n_states[tr] = ns;
      chi2_sum[tr] = 0.0;
      for (int i = 0; i < 6; ++i) last_x[6 * tr + i] = 0.0;
      for (int i = 0; i < 36; ++i) { last_C[36 * tr + i] = 0.0; first_C[36 * tr + i] = 0.0; }
      for (int e = 0; e < 6 * n; ++e) entry_xs[6 * (size_t)e0 + e] = 0.0;
      if (rc == STOP_NONE && ns > 0) {
        xs.assign((size_t)ns * 6, 0.0);
        Cs.assign((size_t)ns * 36, 0.0);
        const bool ok = smoother == 1
            ? two_filter_smooth(ns, st.data(), loc, var, (double(*)[6])xs.data(), (double(*)[6][6])Cs.data())
            : rts_smooth(ns, st.data(), (double(*)[6])xs.data(), (double(*)[6][6])Cs.data());
        if (!ok) rc = STOP_NUMERIC;
      }
      status[tr] = rc;
      if (rc != STOP_NONE || ns == 0) continue;
      double c2 = 0.0;
      int e = 0;
      bool first = true;
      for (int k = 0; k < ns; ++k) {
        if (st[k].meas < 0) continue;
        c2 += st[k].chi2;
        for (int i = 0; i < 6; ++i) entry_xs[6 * (size_t)(e0 + e) + i] = xs[(size_t)k * 6 + i];
        if (first) {
          for (int i = 0; i < 36; ++i) first_C[36 * tr + i] = Cs[(size_t)k * 36 + i];
          first = false;
        }
        ++e;
      }
      chi2_sum[tr] = c2;
      for (int i = 0; i < 6; ++i) last_x[6 * tr + i] = st[ns - 1].xf[i];
      for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) last_C[36 * tr + 6 * i + j] = st[ns - 1].Cf[i][j];
    }
  };
  if (n_threads == 1) work(0);
  else {
    std::vector<std::thread> th;
    for (int t = 0; t < n_threads; ++t) th.emplace_back(work, t);
    for (auto& x : th) x.join();
  }
}

// One track, every state (for the pins): returns the number of states (<= max_states are copied) or -stop.
int32_t oracle_kf_fit_states(const OGeometry* g, const OField* f, const OConfig* cfg, const int32_t* module_offsets,
                             const double* loc, const double* var, int32_t seed_module, const double* sx,
                             const double* sC, int32_t n_meas, const int32_t* meas, int32_t max_states,
                             int32_t* module, int32_t* meas_used, double* xp, double* Cp, double* xf, double* Cf,
                             double* J, double* xs, double* Cs, int32_t smoother) {
  Counters cnt;
  std::vector<FitState> st;
  const int rc = fit_forward(*g, *f, *cfg, module_offsets, loc, var, seed_module, sx, sC, meas, n_meas, st, cnt);
  if (rc != STOP_NONE) return -rc;
  const int ns = (int)st.size();
  std::vector<double> vx((size_t)ns * 6), vC((size_t)ns * 36);
  const bool ok = smoother == 1 ? two_filter_smooth(ns, st.data(), loc, var, (double(*)[6])vx.data(), (double(*)[6][6])vC.data())
                                : rts_smooth(ns, st.data(), (double(*)[6])vx.data(), (double(*)[6][6])vC.data());
  if (!ok) return -STOP_NUMERIC;
  for (int k = 0; k < ns && k < max_states; ++k) {
    module[k] = st[k].module; meas_used[k] = st[k].meas;
    std::memcpy(xp + 6 * k, st[k].xp, 48); std::memcpy(xf + 6 * k, st[k].xf, 48);
    std::memcpy(Cp + 36 * k, st[k].Cp, 288); std::memcpy(Cf + 36 * k, st[k].Cf, 288);
    std::memcpy(J + 36 * k, st[k].J, 288);
    std::memcpy(xs + 6 * k, &vx[(size_t)k * 6], 48); std::memcpy(Cs + 36 * k, &vC[(size_t)k * 36], 288);
  }
  return ns;
}

// The RTS recursion alone on caller-given states (closed-form pin).  Arrays [n][6] / [n][36]; J[k] leads into k.
int32_t oracle_rts_smooth(int32_t n, const double* xp, const double* Cp, const double* xf, const double* Cf,
                          const double* J, double* xs, double* Cs) {
  std::vector<FitState> st(n);
  for (int k = 0; k < n; ++k) {
    st[k].module = 0; st[k].meas = 0; st[k].chi2 = 0.0;
    std::memcpy(st[k].xp, xp + 6 * k, 48); std::memcpy(st[k].xf, xf + 6 * k, 48);
    std::memcpy(st[k].Cp, Cp + 36 * k, 288); std::memcpy(st[k].Cf, Cf + 36 * k, 288);
    std::memcpy(st[k].J, J + 36 * k, 288);
  }
  return rts_smooth(n, st.data(), (double(*)[6])xs, (double(*)[6][6])Cs) ? 0 : STOP_NUMERIC;
}

// ---- pieces exposed for the pins (tests/test_oracle_pins.py)
// AR1-AR3 on a CSR list of candidates (HOST arrays); accepted[t] in {0, 1}, n_shared[t] = s at the decision.
void oracle_resolve_ambiguity(int32_t n_tracks, const int32_t* track_offsets, const int32_t* meas_idx, const double* chi2_sum,
                              int32_t n_measurements, int32_t max_shared_hits, double max_shared_fraction,
                              int32_t* accepted, int32_t* n_shared) {
  resolve_ambiguity(n_tracks, track_offsets, meas_idx, chi2_sum, n_measurements, max_shared_hits, max_shared_fraction,
                    accepted, n_shared);
}

void oracle_set_n3_literal_walk(int32_t on) { g_n3_literal_walk = on ? 1 : 0; }

void oracle_field_at(const OField* f, const double r[3], double B[3]) { field_at(*f, r, B); }

// Free-state propagation to a plane (kind 0: c, n) or cylinder (kind 1: R).  y = (r, t, d, q/p) in/out;
// D (8x8 row-major) out.  Returns stop reason (0 = arrived); n_steps out.
int32_t oracle_propagate_free(const OField* f, const OConfig* cfg, int32_t kind, const double c[3], const double n[3],
                              double R, double y[8], double D[64], int32_t* n_steps) {
  FreeState s;
  for (int i = 0; i < 3; ++i) { s.r[i] = y[i]; s.d[i] = y[4 + i]; }
  s.t = y[3]; s.qop = y[7];
  set_identity8(s.D);
  s.h_ctrl = cfg->h_max_mm; s.n_steps = 0;
  Target tg;
  tg.kind = kind; tg.R = R;
  for (int i = 0; i < 3; ++i) { tg.c[i] = c ? c[i] : 0.0; tg.n[i] = n ? n[i] : 0.0; }
  Counters cnt;
  int st = propagate_to(*f, *cfg, tg, s, cnt);
  for (int i = 0; i < 3; ++i) { y[i] = s.r[i]; y[4 + i] = s.d[i]; }
  y[3] = s.t; y[7] = s.qop;
  if (D) std::memcpy(D, s.D, sizeof(s.D));
  if (n_steps) *n_steps = s.n_steps;
  return st;
}

// One full surface-to-surface move from module `from` (N1-N5, P, J, V5 material on leaving).
int32_t oracle_move(const OGeometry* g, const OField* f, const OConfig* cfg, int32_t from, const double x[6],
                    const double C[36], int32_t* target, double xp[6], double Cp[36], double J[36]) {
  double Ci[6][6], Co[6][6], Jo[6][6];
  std::memcpy(Ci, C, sizeof(Ci));
  Counters cnt;
  int tg = -1;
  int st = move_to_next_module(*g, *f, *cfg, from, x, Ci, tg, xp, Co, Jo, cnt);
  *target = tg;
  g_last_move_trials = cnt.rk_trials;
  if (st == STOP_NONE) {
    std::memcpy(Cp, Co, sizeof(Co));
    if (J) std::memcpy(J, Jo, sizeof(Jo));
  }
  return st;
}

// S: every triplet (bottom, middle, top) of spacepoints on the three seeding layers that passes S1-S4, as a seed (S5, S6).
// Order: by (bottom, middle, top) measurement index.  Threads split the bottom spacepoints.
void* oracle_seed_find(const OGeometry* g, const OField* f, const OSeedConfig* c, int32_t n_meas, const int32_t* module_offsets,
                       const double* loc, const double* var, int32_t n_threads) {
  std::vector<int32_t> meas_module(n_meas, -1);
  for (int id = 0; id < g->n_modules; ++id)
    for (int i = module_offsets[id]; i < module_offsets[id + 1]; ++i) meas_module[i] = id;
  const std::vector<SpacePoint> Bs = layer_spacepoints(*g, c->layer_b, module_offsets, loc);
  const std::vector<SpacePoint> Ms = layer_spacepoints(*g, c->layer_m, module_offsets, loc);
  const std::vector<SpacePoint> Ts = layer_spacepoints(*g, c->layer_t, module_offsets, loc);
  if (n_threads < 1) n_threads = 1;
  std::vector<std::vector<SeedOut>> parts(n_threads);
  auto work = [&](int th) {
    const size_t lo = Bs.size() * th / n_threads, hi = Bs.size() * (th + 1) / n_threads;
    std::vector<std::pair<int, double>> tops;
    for (size_t ib = lo; ib < hi; ++ib)
      for (size_t im = 0; im < Ms.size(); ++im) {
        double cot_bm;
        if (!doublet_ok(*c, Bs[ib], Ms[im], cot_bm)) continue;
        for (size_t it = 0; it < Ts.size(); ++it) {
          double cot_mt;
          if (!doublet_ok(*c, Ms[im], Ts[it], cot_mt)) continue;
          if (!(std::fabs(cot_bm - cot_mt) <= c->dcot_max)) continue;   // S2
          SeedOut s;
          if (triplet_seed(*g, *f, *c, meas_module.data(), loc, var, Bs[ib], Ms[im], Ts[it], s)) parts[th].push_back(s);
        }
      }
  };
  if (n_threads == 1) work(0);
  else {
    std::vector<std::thread> th;
    for (int t = 0; t < n_threads; ++t) th.emplace_back(work, t);
    for (auto& x : th) x.join();
  }
  SeedResult* R = new SeedResult();
  for (auto& p : parts)
    for (auto& s : p) R->seeds.push_back(s);
  std::sort(R->seeds.begin(), R->seeds.end(), [](const SeedOut& a, const SeedOut& b) {
    return a.b != b.b ? a.b < b.b : (a.m != b.m ? a.m < b.m : a.t < b.t);
  });
  return R;
}
int32_t oracle_seed_count(const void* r) { return (int32_t)((const SeedResult*)r)->seeds.size(); }
void oracle_seed_copy(const void* r, int32_t* triplets, int32_t* module, double* params, double* cov) {
  const SeedResult* R = (const SeedResult*)r;
  for (size_t i = 0; i < R->seeds.size(); ++i) {
    const SeedOut& s = R->seeds[i];
    triplets[3 * i] = s.b; triplets[3 * i + 1] = s.m; triplets[3 * i + 2] = s.t;
    module[i] = s.module;
    std::memcpy(params + 6 * i, s.x, sizeof(s.x));
    std::memcpy(cov + 36 * i, s.C, sizeof(s.C));
  }
}
void oracle_seed_free(void* r) { delete (SeedResult*)r; }

// RKN4 trials of the calling thread's last oracle_move (for the per-move comparison of the host-math test)
int64_t oracle_last_move_trials(void) { return g_last_move_trials; }

// Bound -> bound transport between two given modules, no navigation, no material (for the FD pin of J1-J5).
int32_t oracle_bound_to_bound(const OGeometry* g, const OField* f, const OConfig* cfg, int32_t from, int32_t to,
                              const double x[6], double xp[6], double J[36]) {
  const Module m = get_module(*g, from), k = get_module(*g, to);
  FreeState y;
  double B2F[8][6];
  bound_to_free(m, x, y, B2F);
  set_identity8(y.D);
  y.h_ctrl = cfg->h_max_mm; y.n_steps = 0;
  Target pl;
  pl.kind = 0;
  for (int i = 0; i < 3; ++i) { pl.c[i] = k.c[i]; pl.n[i] = k.n[i]; }
  Counters cnt;
  int st = propagate_to(*f, *cfg, pl, y, cnt);
  if (st != STOP_NONE) return st;
  double Jo[6][6];
  arrive(*f, *cfg, k, y, B2F, xp, Jo);
  if (J) std::memcpy(J, Jo, sizeof(Jo));
  return 0;
}

void oracle_transport_cov(const double J[36], const double C[36], double Co[36]) {
  double Jm[6][6], Cm[6][6], O[6][6];
  std::memcpy(Jm, J, sizeof(Jm)); std::memcpy(Cm, C, sizeof(Cm));
  transport_cov(Jm, Cm, O);
  std::memcpy(Co, O, sizeof(O));
}

double oracle_predicted_chi2(const double x[6], const double C[36], const double loc[2], const double var[2]) {
  double Cm[6][6];
  std::memcpy(Cm, C, sizeof(Cm));
  return predicted_chi2(x, Cm, loc, var);
}

void oracle_kalman_update(const double x[6], const double C[36], const double loc[2], const double var[2],
                          double xo[6], double Co[36]) {
  double Cm[6][6], O[6][6];
  std::memcpy(Cm, C, sizeof(Cm));
  kalman_update(x, Cm, loc, var, xo, O);
  std::memcpy(Co, O, sizeof(O));
}

double oracle_highland_theta0(double p, double x_eff, double mass) { return highland_theta0(p, x_eff, mass); }

double oracle_bethe_dedx(double p, double mass) { return bethe_dedx(p, mass); }

// rule E on module `module`: returns dE [GeV], xo[6] = parameters after the loss, *g = d(q/p)'/d(q/p)
double oracle_energy_loss(const OGeometry* g, const OConfig* cfg, int32_t module, const double x[6], double xo[6], double* gE) {
  return energy_loss(*cfg, get_module(*g, module), x, xo, *gE);
}

void oracle_add_material(const OGeometry* g, const OConfig* cfg, int32_t module, const double x[6], double C[36]) {
  double Cm[6][6];
  std::memcpy(Cm, C, sizeof(Cm));
  add_material(*cfg, get_module(*g, module), x, Cm);
  std::memcpy(C, Cm, sizeof(Cm));
}

}  // extern "C"
