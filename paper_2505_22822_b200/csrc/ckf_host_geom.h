// ckf_host_geom.h — host-side packing of ckf_geometry into the device geometry store (a1).
#pragma once
#include <cmath>
#include <vector>

#include "../../include/ckf.h"
#include "ckf_nav.cuh"

namespace ckf {

inline void build_geometry_records(const ckf_geometry& g, std::vector<ModuleRec>& mods, std::vector<LayerRec>& layers) {
  layers.resize(g.n_layers);
  for (int l = 0; l < g.n_layers; ++l) {
    LayerRec& L = layers[l];
    L.r = g.layer_r[l];
    L.half_z = g.layer_half_z[l];
    L.n_phi = g.n_phi[l];
    L.n_z = g.n_z[l];
    L.offset = g.module_offset[l];
    L.len_z = 2.0 * g.half_v[g.module_offset[l]];
    L.pad = 0;
    L.kind = g.layer_kind ? g.layer_kind[l] : 0;
    L.r_min = (g.layer_kind && g.layer_r_min) ? g.layer_r_min[l] : 0.0;
    L.next_disc = -1;
    L.r_in = std::sqrt(L.r * L.r + g.half_u[g.module_offset[l]] * g.half_u[g.module_offset[l]]);
  }
  // next disc of the same side: the one with the smallest |z| beyond this disc's
  for (int l = 0; l < g.n_layers; ++l) {
    if (layers[l].kind != 1) continue;
    for (int k = 0; k < g.n_layers; ++k) {
      if (layers[k].kind != 1 || (layers[k].half_z > 0.0) != (layers[l].half_z > 0.0)) continue;
      if (!(std::fabs(layers[k].half_z) > std::fabs(layers[l].half_z))) continue;
      if (layers[l].next_disc < 0 || std::fabs(layers[k].half_z) < std::fabs(layers[layers[l].next_disc].half_z))
        layers[l].next_disc = k;
    }
  }
  mods.resize(g.n_modules);
  int l = 0;
  for (int id = 0; id < g.n_modules; ++id) {
    while (l + 1 < g.n_layers && id >= g.module_offset[l + 1]) ++l;
    ModuleRec& m = mods[id];
    for (int i = 0; i < 3; ++i) {
      m.c[i] = g.center[3 * id + i];
      m.u[i] = g.axis_u[3 * id + i];
      m.v[i] = g.axis_v[3 * id + i];
    }
    m.n[0] = m.u[1] * m.v[2] - m.u[2] * m.v[1];
    m.n[1] = m.u[2] * m.v[0] - m.u[0] * m.v[2];
    m.n[2] = m.u[0] * m.v[1] - m.u[1] * m.v[0];
    m.half_u = g.half_u[id];
    m.half_v = g.half_v[id];
    m.xx0 = g.x_over_x0[id];
    m.layer = l;
    m.iphi = (id - g.module_offset[l]) / g.n_z[l];
  }
}

// barrel layers first (n_barrel of them), innermost disc of each side
inline void fill_geo_summary(const std::vector<LayerRec>& layers, GeoDev& geo) {
  geo.n_barrel = 0;
  while (geo.n_barrel < (int)layers.size() && layers[geo.n_barrel].kind == 0) ++geo.n_barrel;
  geo.first_disc[0] = geo.first_disc[1] = -1;
  for (int l = 0; l < (int)layers.size(); ++l) {
    if (layers[l].kind != 1) continue;
    const int side = layers[l].half_z > 0.0 ? 0 : 1;
    if (geo.first_disc[side] < 0 || std::fabs(layers[l].half_z) < std::fabs(layers[geo.first_disc[side]].half_z))
      geo.first_disc[side] = l;
  }
}

// Device layout of the field grid (ckf_math.cuh, ld_pair): entry (i, j, k) = node (i, j, k) then node (i, j, k + 1),
// each (Bx, By, Bz, 0) as float32; the last entry along z repeats its own node (no cell starts there).
inline void fill_field_pairs(const float* grid, const int32_t n[3], std::vector<float>& out) {
  const size_t n0 = n[0], n1 = n[1], n2 = n[2];
  out.assign(8 * n0 * n1 * n2, 0.0f);
  for (size_t i = 0; i < n0; ++i)
    for (size_t j = 0; j < n1; ++j)
      for (size_t k = 0; k < n2; ++k) {
        const size_t e = (i * n1 + j) * n2 + k, e1 = (i * n1 + j) * n2 + (k + 1 < n2 ? k + 1 : k);
        for (int c = 0; c < 3; ++c) { out[8 * e + c] = grid[3 * e + c]; out[8 * e + 4 + c] = grid[3 * e1 + c]; }
      }
}

}  // namespace ckf
