// ckf_seed.cuh — triplet seeding and helix parameter estimation on the device (row f4, the stage in front of the CKF).
//
// "The spacepoints are used in the seeding algorithm where triplets, a set of three spacepoints which can
// approximately form a helix, are found.  In the track parameter estimation algorithm, the position and momentum of
// tracks, called a seed, are estimated at the first spacepoint using the helix model."  Rules S0-S6 of DESIGN.md 3.
//
// The measurement CSR is ordered by module id and a layer's modules are ordered (phi column, z row), so the measurements
// of one phi column of a layer are ONE contiguous index range: the spacepoints an inner spacepoint can pair with are the
// union of a few such ranges (the columns within dphi_max of it), visited in ascending index.  Everything is placed by
// count -> exclusive scan -> fill, in (bottom, middle, top) index order, so the seed list is deterministic and equals
// the oracle's enumeration of all combinations.
//   seed_spacepoints   thread per measurement of the three layers: global position, rho, phi (S0), float64
//   seed_doublets_mt   thread per middle spacepoint, two passes: the tops compatible with it (S1) -> CSR list (t, cot)
//   seed_triplets      warp per bottom spacepoint, two passes: lanes test the candidate middles (S1); for every passing
//                      middle the warp runs over its top list, 32 tops at a time (S2-S4); second pass writes the seeds
//                      (S5, S6) at their scanned offsets
//   seed_scan          single-block exclusive scan of the per-spacepoint counts
#pragma once
#include "ckf_nav.cuh"

namespace ckf {

struct SeedCfgDev {
  int32_t layer_b, layer_m, layer_t;
  double dphi_max, cot_max, z0_max, dcot_max, pt_min, d0_max, sigma_angle, rel_sigma_qop, cov_scale;
};

template <typename T>
struct SeedParams {
  GeoDev geo;
  FieldDev fld;
  SeedCfgDev cfg;
  int32_t n_meas;
  const int32_t* moff;
  const T* loc;   // [n][2]
  const T* var;   // [n][2]
  // workspace
  double* sp;          // [5][n_cap] x, y, z, rho, phi by measurement index
  int32_t n_cap;
  int32_t* cnt;        // [n_cap + 1] per-spacepoint counts, then exclusive offsets (in place)
  int32_t* mt_off;     // [n_cap + 1] offsets of the middle -> top lists
  int32_t* mt_t;       // [max_doublets]
  double* mt_cot;      // [max_doublets]
  int32_t max_doublets;
  int32_t* g;          // [4] totals: doublets, triplets
  // output (caller-owned device arrays)
  int32_t capacity;
  int32_t* o_n; int32_t* o_status; int32_t* o_module; T* o_params; T* o_cov; int32_t* o_triplets;
};

struct SP { double x, y, z, rho, phi; };
template <typename T>
__device__ __forceinline__ SP load_sp(const SeedParams<T>& p, int i) {
  const size_t N = (size_t)p.n_cap;
  return SP{p.sp[i], p.sp[N + i], p.sp[2 * N + i], p.sp[3 * N + i], p.sp[4 * N + i]};
}

// measurement index range [lo, hi) of a layer
template <typename T>
__device__ __forceinline__ void layer_range(const SeedParams<T>& p, int layer, int& lo, int& hi) {
  const LayerRec L = p.geo.layer[layer];
  lo = p.moff[L.offset];
  hi = p.moff[L.offset + L.n_phi * L.n_z];
}

template <typename T>
__global__ void seed_spacepoints(const SeedParams<T> p) {
  const int layers[3] = {p.cfg.layer_b, p.cfg.layer_m, p.cfg.layer_t};
  const size_t N = (size_t)p.n_cap;
  if (blockIdx.x == 0 && threadIdx.x < 4) p.g[threadIdx.x] = 0;
  for (int k = 0; k < 3; ++k) {
    const LayerRec L = p.geo.layer[layers[k]];
    for (int mod = L.offset + blockIdx.x; mod < L.offset + L.n_phi * L.n_z; mod += gridDim.x) {
      const ModuleRec& m = p.geo.mod[mod];
      for (int i = p.moff[mod] + threadIdx.x; i < p.moff[mod + 1]; i += blockDim.x) {
        const double l0 = (double)p.loc[2 * (size_t)i], l1 = (double)p.loc[2 * (size_t)i + 1];
        const double x = m.c[0] + l0 * m.u[0] + l1 * m.v[0];
        const double y = m.c[1] + l0 * m.u[1] + l1 * m.v[1];
        const double z = m.c[2] + l0 * m.u[2] + l1 * m.v[2];
        p.sp[i] = x; p.sp[N + i] = y; p.sp[2 * N + i] = z;
        p.sp[3 * N + i] = hypot(x, y);
        p.sp[4 * N + i] = atan2(y, x);
      }
    }
  }
}

// S1: doublet (inner, outer) -> cot theta
__device__ __forceinline__ bool doublet_ok(const SeedCfgDev& c, const SP& in, const SP& out, double& cot) {
  double dphi = out.phi - in.phi;
  while (dphi > PI_D) dphi -= 2.0 * PI_D;
  while (dphi <= -PI_D) dphi += 2.0 * PI_D;
  if (!(fabs(dphi) <= c.dphi_max)) return false;
  const double drho = out.rho - in.rho;
  if (!(drho > 0.0)) return false;
  cot = (out.z - in.z) / drho;
  if (!(fabs(cot) <= c.cot_max)) return false;
  const double z0 = in.z - in.rho * cot;
  return fabs(z0) <= c.z0_max;
}

// The phi columns of `layer` whose spacepoints can lie within dphi_max of azimuth phi: ascending column indices, as up
// to MAXCOL contiguous measurement ranges (a superset: the exact cut is applied per spacepoint).
constexpr int MAXCOL = 16;
template <typename T>
__device__ __forceinline__ int column_ranges(const SeedParams<T>& p, int layer, double phi, int lo[MAXCOL], int hi[MAXCOL]) {
  const LayerRec L = p.geo.layer[layer];
  const double half_u = p.geo.mod[L.offset].half_u;
  const double reach = p.cfg.dphi_max + atan2(half_u, L.r) + 1e-6;      // a spacepoint's phi vs its module's centre phi
  const double pitch = 2.0 * PI_D / L.n_phi;
  int w = (int)ceil(reach / pitch);
  const int ic = (int)nearbyint(phi / pitch);
  if (2 * w + 1 >= L.n_phi || 2 * w + 1 > MAXCOL) {   // the window covers the whole layer (or would not fit): one range
    lo[0] = p.moff[L.offset];
    hi[0] = p.moff[L.offset + L.n_phi * L.n_z];
    return 1;
  }
  int cols[MAXCOL], n = 0;
  for (int k = -w; k <= w; ++k) cols[n++] = (((ic + k) % L.n_phi) + L.n_phi) % L.n_phi;
  for (int a = 1; a < n; ++a) {   // ascending (a wrapped window is two runs)
    const int v = cols[a];
    int b = a - 1;
    while (b >= 0 && cols[b] > v) { cols[b + 1] = cols[b]; --b; }
    cols[b + 1] = v;
  }
  for (int a = 0; a < n; ++a) {
    lo[a] = p.moff[L.offset + cols[a] * L.n_z];
    hi[a] = p.moff[L.offset + (cols[a] + 1) * L.n_z];
  }
  return n;
}

// thread per middle spacepoint: its compatible tops.  WRITE = false counts, WRITE = true fills the list.
template <typename T, bool WRITE>
__global__ void seed_doublets_mt(const SeedParams<T> p) {
  int mlo, mhi;
  layer_range(p, p.cfg.layer_m, mlo, mhi);
  const bool overflow = WRITE && p.g[0] > p.max_doublets;
  for (int im = mlo + blockIdx.x * blockDim.x + threadIdx.x; im < mhi; im += gridDim.x * blockDim.x) {
    const SP M = load_sp(p, im);
    int lo[MAXCOL], hi[MAXCOL];
    const int nr = column_ranges(p, p.cfg.layer_t, M.phi, lo, hi);
    int n = 0;
    const int base = WRITE ? p.mt_off[im - mlo] : 0;
    for (int r = 0; r < nr; ++r)
      for (int it = lo[r]; it < hi[r]; ++it) {
        double cot;
        if (!doublet_ok(p.cfg, M, load_sp(p, it), cot)) continue;
        if (WRITE && !overflow) { p.mt_t[base + n] = it; p.mt_cot[base + n] = cot; }
        ++n;
      }
    if (!WRITE) p.cnt[im - mlo] = n;
  }
}

// single block: exclusive scan of cnt[0..n) into out[0..n], total into *total
__global__ void __launch_bounds__(1024) seed_scan(const int32_t* cnt, int32_t* out, int n, int32_t* total) {
  __shared__ int s_w[32];
  __shared__ int s_carry;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  if (tid == 0) s_carry = 0;
  __syncthreads();
  for (int i0 = 0; i0 < n; i0 += 1024) {
    const int i = i0 + tid;
    const int v = i < n ? cnt[i] : 0;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) s_w[w] = inc;
    __syncthreads();
    int base = s_carry, tot = 0;
#pragma unroll
    for (int k = 0; k < 32; ++k) {
      const int x = s_w[k];
      if (k < w) base += x;
      tot += x;
    }
    if (i < n) out[i] = base + inc - v;
    __syncthreads();
    if (tid == 0) s_carry += tot;
    __syncthreads();
  }
  if (tid == 0) { out[n] = s_carry; *total = s_carry; }
}

// S3-S6 of one triplet that passed S1, S2.  Returns false if a cut fails; fills x[6] and the six variances otherwise.
template <typename T>
__device__ __forceinline__ bool triplet_seed(const SeedParams<T>& p, const SP& B, const SP& M, const SP& Tp, int ib, int im,
                                             int it, double x[6], double dvar[6]) {
  const double d = 2.0 * (B.x * (M.y - Tp.y) + M.x * (Tp.y - B.y) + Tp.x * (B.y - M.y));
  if (d == 0.0) return false;
  const double b2 = B.x * B.x + B.y * B.y, m2 = M.x * M.x + M.y * M.y, t2 = Tp.x * Tp.x + Tp.y * Tp.y;
  const double xc = (b2 * (M.y - Tp.y) + m2 * (Tp.y - B.y) + t2 * (B.y - M.y)) / d;
  const double yc = (b2 * (Tp.x - M.x) + m2 * (B.x - Tp.x) + t2 * (M.x - B.x)) / d;
  const double R = hypot(B.x - xc, B.y - yc);
  const double rB[3] = {B.x, B.y, B.z};
  double Bf[3];
  field_at(p.fld, rB, Bf);
  const double pt = KAPPA * fabs(Bf[2]) * R;
  if (!(pt >= p.cfg.pt_min)) return false;
  if (!(fabs(hypot(xc, yc) - R) <= p.cfg.d0_max)) return false;
  double tx = -(B.y - yc) / R, ty = (B.x - xc) / R;
  if (tx * (M.x - B.x) + ty * (M.y - B.y) < 0.0) { tx = -tx; ty = -ty; }
  const double cz = (M.x - B.x) * (Tp.y - M.y) - (M.y - B.y) * (Tp.x - M.x);
  const double q = (cz * Bf[2] < 0.0) ? 1.0 : -1.0;
  const double chord = hypot(Tp.x - B.x, Tp.y - B.y);
  const double arc = 2.0 * R * asin(fmin(1.0, chord / (2.0 * R)));
  const double cot = (Tp.z - B.z) / arc;
  const double theta = atan2(1.0, cot);
  x[0] = (double)p.loc[2 * (size_t)ib]; x[1] = (double)p.loc[2 * (size_t)ib + 1];
  x[2] = atan2(ty, tx);
  x[3] = theta;
  x[4] = q * sin(theta) / pt;
  x[5] = 0.0;
  const double var_sag = (double)p.var[2 * (size_t)im] + 0.25 * ((double)p.var[2 * (size_t)ib] + (double)p.var[2 * (size_t)it]);
  const double dcurv = 8.0 * sqrt(var_sag) / (chord * chord);
  const double sq_res = sin(theta) * dcurv / (KAPPA * fabs(Bf[2]));
  const double k = p.cfg.cov_scale;
  dvar[0] = k * (double)p.var[2 * (size_t)ib];
  dvar[1] = k * (double)p.var[2 * (size_t)ib + 1];
  dvar[2] = k * p.cfg.sigma_angle * p.cfg.sigma_angle;
  dvar[3] = dvar[2];
  dvar[4] = k * (sq_res * sq_res + (p.cfg.rel_sigma_qop * x[4]) * (p.cfg.rel_sigma_qop * x[4]));
  dvar[5] = 1.0;
  return true;
}

// warp per bottom spacepoint.  WRITE = false: number of its triplets into cnt; WRITE = true: the seeds themselves at
// cnt[b] (now the exclusive offset) onward, in (middle, top) index order.
template <typename T, bool WRITE>
__global__ void __launch_bounds__(128) seed_triplets(const SeedParams<T> p) {
  int blo, bhi, mlo, mhi;
  layer_range(p, p.cfg.layer_b, blo, bhi);
  layer_range(p, p.cfg.layer_m, mlo, mhi);
  const int lane = threadIdx.x & 31;
  const int gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = (gridDim.x * blockDim.x) >> 5;
  const bool bad = p.g[0] > p.max_doublets;   // the doublet lists did not fit: no seeds, flagged by seed_finish
  for (int ib = blo + gw; ib < bhi; ib += nw) {
    const SP B = load_sp(p, ib);
    int lo[MAXCOL], hi[MAXCOL];
    const int nr = bad ? 0 : column_ranges(p, p.cfg.layer_m, B.phi, lo, hi);
    int n_trip = 0;
    const int out0 = WRITE ? p.cnt[ib - blo] : 0;
    for (int r = 0; r < nr; ++r)
      for (int m0 = lo[r]; m0 < hi[r]; m0 += 32) {
        const int im = m0 + lane;
        double cot_bm = 0.0;
        SP M = B;
        bool ok = false;
        if (im < hi[r]) { M = load_sp(p, im); ok = doublet_ok(p.cfg, B, M, cot_bm); }
        unsigned pass = __ballot_sync(0xffffffffu, ok);
        while (pass) {   // the passing middles of this chunk, in ascending index
          const int src = __ffs(pass) - 1;
          pass &= pass - 1;
          const int jm = m0 + src;
          const double cbm = __shfl_sync(0xffffffffu, cot_bm, src);
          const SP Mj = SP{__shfl_sync(0xffffffffu, M.x, src), __shfl_sync(0xffffffffu, M.y, src),
                           __shfl_sync(0xffffffffu, M.z, src), __shfl_sync(0xffffffffu, M.rho, src),
                           __shfl_sync(0xffffffffu, M.phi, src)};
          const int t_lo = p.mt_off[jm - mlo], t_hi = p.mt_off[jm - mlo + 1];
          for (int k0 = t_lo; k0 < t_hi; k0 += 32) {
            const int k = k0 + lane;
            bool good = false;
            int it = 0;
            double x[6], dv[6];
            if (k < t_hi && fabs(cbm - p.mt_cot[k]) <= p.cfg.dcot_max) {   // S2
              it = p.mt_t[k];
              good = triplet_seed<T>(p, B, Mj, load_sp(p, it), ib, jm, it, x, dv);
            }
            const unsigned gb = __ballot_sync(0xffffffffu, good);
            if (WRITE && good) {
              const int o = out0 + n_trip + __popc(gb & ((1u << lane) - 1u));
              if (o < p.capacity) {
                p.o_triplets[3 * (size_t)o] = ib; p.o_triplets[3 * (size_t)o + 1] = jm; p.o_triplets[3 * (size_t)o + 2] = it;
                int mod = 0;   // module of the bottom measurement: the CSR slice that holds it (binary search)
                {
                  const LayerRec L = p.geo.layer[p.cfg.layer_b];
                  int a = L.offset, b = L.offset + L.n_phi * L.n_z;   // moff[a] <= ib < moff[b]
                  while (b - a > 1) { const int mid = (a + b) >> 1; if (p.moff[mid] <= ib) a = mid; else b = mid; }
                  mod = a;
                }
                p.o_module[o] = mod;
#pragma unroll
                for (int i = 0; i < 6; ++i) p.o_params[6 * (size_t)o + i] = (T)x[i];
#pragma unroll
                for (int i = 0; i < 36; ++i) p.o_cov[36 * (size_t)o + i] = T(0);
#pragma unroll
                for (int i = 0; i < 6; ++i) p.o_cov[36 * (size_t)o + 7 * i] = (T)dv[i];
              }
            }
            n_trip += __popc(gb);
          }
        }
      }
    if (!WRITE && lane == 0) p.cnt[ib - blo] = n_trip;
  }
}

template <typename T>
__global__ void seed_finish(const SeedParams<T> p) {
  const int total = p.g[1];
  int status = 0;
  if (p.g[0] > p.max_doublets) status |= 2;
  if (total > p.capacity) status |= 1;
  *p.o_n = status & 2 ? 0 : (total < p.capacity ? total : p.capacity);
  *p.o_status = status;
}

}  // namespace ckf
