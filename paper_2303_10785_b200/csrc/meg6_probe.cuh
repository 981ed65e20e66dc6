// meg6_probe.cuh -- FP64-pipe roof by measurement ("to be confirmed by a DFMA micro-benchmark").
// A register-resident loop of independent DFMA chains; nothing of the method is computed here.
#pragma once
#include <cuda_runtime.h>

namespace meg6 {

constexpr int PROBE_CHAINS = 8, PROBE_ITERS = 4096, PROBE_THREADS = 256;

__global__ void __launch_bounds__(PROBE_THREADS) k_dfma_probe(double a, double b, double* __restrict__ sink) {
  double x[PROBE_CHAINS];
#pragma unroll
  for (int q = 0; q < PROBE_CHAINS; ++q) x[q] = (double)(threadIdx.x + q) * 1e-3;
  for (int it = 0; it < PROBE_ITERS; ++it) {
#pragma unroll
    for (int q = 0; q < PROBE_CHAINS; ++q) x[q] = fma(x[q], a, b);   // PROBE_CHAINS independent dependency chains
  }
  double s = 0.0;
#pragma unroll
  for (int q = 0; q < PROBE_CHAINS; ++q) s += x[q];
  if (s == 123.456) sink[0] = s;   // keeps the loop alive; never true for the arguments used
}

}  // namespace meg6
