// ckf_resolve.cuh — ambiguity resolution after the CKF (row f4; "an additional algorithm -- known as
// ambiguity resolution -- will be integrated into the reconstruction chain to remove such [duplicate and fake] tracks
// after the CKF stage").  Rules AR1-AR3 of DESIGN.md 3: candidates ranked by (more measurements, smaller float32 chi2
// sum, lower index); in that order a candidate is accepted iff at most max_shared_hits (and at most
// max_shared_fraction of) its measurements already belong to accepted candidates, and then takes its free ones.
//
// The sequential greedy is reproduced EXACTLY by rounds that are parallel over the candidates: a candidate's decision
// depends only on the better-ranked candidates that share a measurement with it, so every candidate that is the best
// undecided one on ALL of its measurements can be decided in the same round (two such candidates cannot share a
// measurement, so their ownership writes never collide).  "Best undecided on a measurement" is an atomicMin of the
// 64-bit rank key per measurement, which is order-independent: the result is deterministic.  One cooperative launch,
// two grid-wide barriers per round (the per-measurement minima are double-buffered by round parity, so the reset of one
// buffer rides along with the decisions made from the other); the number of rounds is the longest chain of candidates linked by shared
// measurements (the candidates of one seed share its first hits, so about max_candidates_per_seed at worst).
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <cstdint>

namespace ckf {

constexpr int RESOLVE_NT = 256;
constexpr unsigned long long RANK_NONE = ~0ull;

template <typename T>
struct ResolveParams {
  const int32_t* n_tracks;   // device [1]
  const int32_t* offsets;    // CSR of the candidates (ckf_tracks)
  const int32_t* meas;
  const T* chi2sum;
  int32_t max_tracks;
  int32_t n_meas;
  int32_t max_shared;
  double max_frac;
  unsigned long long* key;   // [max_tracks] rank key of a candidate (smaller = better)
  unsigned long long* best;  // [2][n_meas] smallest key among the undecided candidates holding the measurement
  int32_t* owner;            // [n_meas] accepted candidate that owns the measurement, -1 = free
  int32_t* state;            // [max_tracks] 0 undecided, 1 accepted, 2 rejected, 3 / 4 the same, decided in the last round
  int32_t* g;                // [4] undecided candidates left after a round (three slots, by round % 3), accepted
  int32_t* o_accepted;       // [max_tracks] 1 / 0
  int32_t* o_nshared;        // [max_tracks] shared measurements at the decision
  int32_t* o_summary;        // [2] accepted candidates, rounds
};

// AR1: (255 - n_meas) : 8 | order-preserving bits of the float32 chi2 sum : 32 | candidate index : 24
__device__ __forceinline__ unsigned long long rank_key(int n, float chi2, int t) {
  unsigned int b = __float_as_uint(chi2);
  b = (chi2 != chi2) ? 0xffffffffu : ((b & 0x80000000u) ? ~b : (b | 0x80000000u));
  const unsigned int nn = (unsigned int)(255 - (n > 255 ? 255 : n));
  return ((unsigned long long)nn << 56) | ((unsigned long long)b << 24) | (unsigned long long)(t & 0xffffff);
}

template <typename T>
__global__ void __launch_bounds__(RESOLVE_NT) ckf_resolve_kernel(const ResolveParams<T> p) {
  namespace cg = cooperative_groups;
  cg::grid_group grid = cg::this_grid();
  const int nt = min(*p.n_tracks, p.max_tracks);
  const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
  for (int m = tid; m < p.n_meas; m += nth) { p.owner[m] = -1; p.best[m] = RANK_NONE; p.best[(size_t)p.n_meas + m] = RANK_NONE; }
  for (int t = tid; t < nt; t += nth) {
    p.key[t] = rank_key(p.offsets[t + 1] - p.offsets[t], (float)p.chi2sum[t], t);
    p.state[t] = 0;
  }
  if (tid == 0) { p.g[0] = 0; p.g[1] = 0; p.g[2] = 0; p.g[3] = 0; }
  grid.sync();
  for (int round = 0;; ++round) {
    unsigned long long* best = p.best + (size_t)(round & 1) * (size_t)p.n_meas;
    unsigned long long* best_next = p.best + (size_t)((round + 1) & 1) * (size_t)p.n_meas;
    // A: the best undecided candidate on every measurement
    for (int t = tid; t < nt; t += nth) {
      if (p.state[t] != 0) continue;
      const unsigned long long k = p.key[t];
      for (int e = p.offsets[t]; e < p.offsets[t + 1]; ++e) atomicMin(best + p.meas[e], k);
    }
    // three slots: slot (round + 1) % 3 was last READ after the second barrier of round - 2, so clearing it here cannot
    // race with a block that still reads the count of the previous round
    if (tid == 0) p.g[(round + 1) % 3] = 0;
    grid.sync();
    // B: decide every candidate that is the best undecided one on all of its measurements (AR2, AR3)
    int remaining = 0, acc = 0;
    for (int t = tid; t < nt; t += nth) {
      const int st = p.state[t];
      if (st == 1 || st == 2) continue;
      const int e0 = p.offsets[t], e1 = p.offsets[t + 1];
      if (st >= 3) {   // decided in the previous round: its keys are still in the other buffer, take them out
        for (int e = e0; e < e1; ++e) best_next[p.meas[e]] = RANK_NONE;
        p.state[t] = st - 2;
        continue;
      }
      const unsigned long long k = p.key[t];
      bool first = true;
      int s = 0;
      for (int e = e0; e < e1; ++e) {
        const int m = p.meas[e];
        first = first && best[m] == k;
        s += p.owner[m] >= 0 ? 1 : 0;
        best_next[m] = RANK_NONE;   // the other buffer holds the minima of the previous round: every candidate that wrote
      }                             // there (undecided then) clears its entries now, before next round's atomicMin
      if (!first) { ++remaining; continue; }
      const bool ok = s <= p.max_shared && (double)s <= p.max_frac * (double)(e1 - e0);
      p.o_accepted[t] = ok ? 1 : 0;
      p.o_nshared[t] = s;
      p.state[t] = ok ? 3 : 4;      // decided now; 1 / 2 once its keys are out of both buffers
      if (ok) {
        ++acc;
        for (int e = e0; e < e1; ++e) {
          const int m = p.meas[e];
          if (p.owner[m] < 0) p.owner[m] = t;   // no other candidate decided in this round holds m
        }
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      remaining += __shfl_xor_sync(0xffffffffu, remaining, o);
      acc += __shfl_xor_sync(0xffffffffu, acc, o);
    }
    if ((threadIdx.x & 31) == 0) {
      if (remaining) atomicAdd(p.g + (round % 3), remaining);
      if (acc) atomicAdd(p.g + 3, acc);
    }
    grid.sync();
    const int left = p.g[round % 3];
    if (left == 0) {
      if (tid == 0) { p.o_summary[0] = p.g[3]; p.o_summary[1] = round + 1; }
      break;
    }
  }
}

}  // namespace ckf
