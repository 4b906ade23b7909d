// ckf_peak.cuh — the roofline denominator of this library, MEASURED: plain-ALU FMA throughput of the device
// ("verify both the lane counts and the sustained clock with an FMA-chain microbenchmark on the
// box").  The CKF path runs on the FP32/FP64 ALUs, not on the tensor cores (north_star), and MEASURED_PEAKS.json
// holds no ALU peak, so bench.py calls ckf_measure_alu_peak and reports fractions "of measured".
#pragma once
#include <cuda_runtime.h>

namespace ckf {

// Every thread advances NF independent float chains and ND independent double chains x <- x * a + b; the chains of a
// thread are independent (ILP), 64 warps per SM hide the rest of the FMA latency.  Nothing is loaded; one store per
// thread at the end keeps the chains alive.
template <int NF, int ND>
__global__ void __launch_bounds__(256) ckf_fma_chain(double* out, int iters, float af, float bf, double ad, double bd) {
  float xf[NF > 0 ? NF : 1];
  double xd[ND > 0 ? ND : 1];
#pragma unroll
  for (int k = 0; k < NF; ++k) xf[k] = 1.0f + 1e-3f * (float)(threadIdx.x + k);
#pragma unroll
  for (int k = 0; k < ND; ++k) xd[k] = 1.0 + 1e-3 * (double)(threadIdx.x + k);
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
#pragma unroll
      for (int k = 0; k < NF; ++k) xf[k] = fmaf(xf[k], af, bf);
#pragma unroll
      for (int k = 0; k < ND; ++k) xd[k] = fma(xd[k], ad, bd);
    }
  }
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < NF; ++k) s += (double)xf[k];
#pragma unroll
  for (int k = 0; k < ND; ++k) s += xd[k];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace ckf
