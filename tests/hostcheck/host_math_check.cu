// host_math_check.cu — TEST ONLY.  Runs the per-tip arithmetic of the CUDA path (csrc/ckf_math.cuh,
// ckf_nav.cuh: the very source the kernels inline) on the host CPU, so that the GPU-less test tier can compare
// it element by element with the oracle.  It is not part of libckf.so and the product never calls it.
#include <cuda_runtime.h>

#include <cstring>
#include <vector>

#include "../../paper_2505_22822_b200/csrc/ckf_host_geom.h"
#include "../../paper_2505_22822_b200/csrc/ckf_nav.cuh"

using namespace ckf;

namespace {
struct Ctx {
  std::vector<ModuleRec> mods;
  std::vector<LayerRec> layers;
  std::vector<float> grid;
  GeoDev geo;
  FieldDev fld;
  CfgDev cfg;
};

template <typename T>
int move_t(Ctx* c, int from, const double* x, const double* C36, int* target, double* xp, double* Cp36, int* trials) {
  double J[5][5], qphi, qth, ge;
  StepCtl sc;
  sc.n_trials = 0; sc.n_accepted = 0;
  int tg = -1;
  int st = move_to_next_module<T>(c->geo, c->fld, c->cfg, from, x, tg, xp, J, qphi, qth, ge, sc);
  *target = tg;
  if (trials) *trials = sc.n_trials;
  if (st != STOP_NONE) return st;
  double C[21], Co[21];
  for (int i = 0; i < 6; ++i)
    for (int j = i; j < 6; ++j) C[tri(i, j)] = C36[6 * i + j];
  const double dep[NDEP] = {0.0, 0.0, 0.0, qphi, qth, ge};
  leave_module_cov(C, dep);
  transport_cov<double>(J, C, Co);
  for (int i = 0; i < 6; ++i)
    for (int j = 0; j < 6; ++j) Cp36[6 * i + j] = (double)Co[tri(i, j)];
  return st;
}

template <typename T>
void update_t(const double* x, const double* C36, const double* loc, const double* var, double* xo, double* Co36,
              double* chi2) {
  double C[21], Co[21];
  for (int i = 0; i < 6; ++i)
    for (int j = i; j < 6; ++j) C[tri(i, j)] = C36[6 * i + j];
  double c2 = 0.0;
  gate_chi2<T>(x[0], x[1], C[tri(0, 0)], C[tri(0, 1)], C[tri(1, 1)], (T)loc[0], (T)loc[1], (T)var[0], (T)var[1], 1e30, c2);
  *chi2 = c2;
  kalman_update<T>(x, C, (T)loc[0], (T)loc[1], (T)var[0], (T)var[1], xo, Co);
  for (int i = 0; i < 6; ++i)
    for (int j = 0; j < 6; ++j) Co36[6 * i + j] = (double)Co[tri(i, j)];
}
}  // namespace

extern "C" {

void* hm_create(const ckf_geometry* g, const ckf_field* f, const ckf_config* c) {
  Ctx* x = new Ctx();
  build_geometry_records(*g, x->mods, x->layers);
  x->geo.mod = x->mods.data(); x->geo.layer = x->layers.data(); x->geo.n_layers = g->n_layers; x->geo.n_modules = g->n_modules;
  fill_geo_summary(x->layers, x->geo);
  x->geo.bidir = c->bidirectional ? 1 : 0;
  std::memset(&x->fld, 0, sizeof(x->fld));
  x->fld.kind = f->kind;
  for (int a = 0; a < 3; ++a) {
    x->fld.ub[a] = f->uniform_b[a]; x->fld.n[a] = f->n[a]; x->fld.org[a] = f->origin[a];
    x->fld.inv[a] = f->kind == 1 ? 1.0 / f->spacing[a] : 0.0;
    x->fld.nm2[a] = (double)(f->n[a] - 2);
  }
  if (f->kind == 1) {
    fill_field_pairs(f->grid, f->n, x->grid);
    x->fld.grid = x->grid.data();
  }
  x->cfg.chi2_max = c->chi2_max; x->cfg.rk_tol = c->rk_tolerance_mm; x->cfg.surf_tol = c->surface_tolerance_mm;
  x->cfg.h_max = c->h_max_mm; x->cfg.mass = c->particle_mass_gev; x->cfg.max_branches = c->max_branches_per_surface;
  x->cfg.max_cands = c->max_candidates_per_seed; x->cfg.max_holes = c->max_holes; x->cfg.min_meas = c->min_measurements;
  x->cfg.max_rk_steps = c->max_rk_steps_per_surface; x->cfg.max_levels = c->max_levels;
  x->cfg.energy_loss = c->energy_loss ? 1 : 0;
  x->cfg.field_gradient = (c->field_gradient == 1 && f->kind == 1) ? 1 : 0;
  return x;
}
void hm_destroy(void* p) { delete (Ctx*)p; }

int hm_move(void* p, int precision, int from, const double* x, const double* C36, int* target, double* xp, double* Cp36,
            int* trials) {
  return precision == 32 ? move_t<float>((Ctx*)p, from, x, C36, target, xp, Cp36, trials)
                         : move_t<double>((Ctx*)p, from, x, C36, target, xp, Cp36, trials);
}
void hm_update(int precision, const double* x, const double* C36, const double* loc, const double* var, double* xo,
               double* Co36, double* chi2) {
  if (precision == 32) update_t<float>(x, C36, loc, var, xo, Co36, chi2);
  else update_t<double>(x, C36, loc, var, xo, Co36, chi2);
}
void hm_field(void* p, const double* r, double* B) { field_at(((Ctx*)p)->fld, r, B); }
void hm_field_gradient(void* p, const double* r, double* G9) {
  double G[3][3];
  field_gradient_at(((Ctx*)p)->fld, r, G);
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) G9[3 * i + j] = G[i][j];
}
}
