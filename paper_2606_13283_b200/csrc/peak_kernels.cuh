// peak_kernels.cuh -- microbenchmarks that MEASURE the two rooflines MEASURED_PEAKS.json does not hold: the fp64 FMA
// peak of the vector pipe (the bound of the Fermi-Dirac kernels and of the O(N_i N_g) ion-grid sums) and the L2 read
// bandwidth (the bound of the L2-resident grids c1/c2).  bench.py runs them in the same process as the timed steps and
// reports every "alu" / "l2" fraction against these numbers.
#pragma once
#include "common.cuh"

namespace arche {

// kChains independent dependent-FMA chains per thread: with 8 chains x 8 warps per scheduler the 4-8 cycle DFMA
// latency is covered many times over, so the kernel runs at the issue rate of the fp64 pipe.
constexpr int kPeakChains = 8;
__global__ void __launch_bounds__(256) fp64_fma_peak_kernel(long long iters, double a, double b, double *out) {
  double x[kPeakChains];
#pragma unroll
  for (int k = 0; k < kPeakChains; ++k) x[k] = 1.0 + 1e-3 * (threadIdx.x + k);
#pragma unroll 4
  for (long long i = 0; i < iters; ++i) {
#pragma unroll
    for (int k = 0; k < kPeakChains; ++k) x[k] = fma(x[k], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < kPeakChains; ++k) s += x[k];
  if (s == 12345.678) out[blockIdx.x * blockDim.x + threadIdx.x] = s;   // never true: keeps the chains alive
}

// every thread streams 16-byte words of a buffer that fits the L2 (grid-stride, `reps` sweeps)
__global__ void __launch_bounds__(256) l2_read_peak_kernel(const double2 *__restrict__ buf, long long n, int reps, double *out) {
  double s = 0.0;
  const long long stride = (long long)gridDim.x * blockDim.x, t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  for (int r = 0; r < reps; ++r) {
    long long g = t0;
    for (; g + 3 * stride < n; g += 4 * stride) {
      const double2 v0 = __ldcg(buf + g), v1 = __ldcg(buf + g + stride), v2 = __ldcg(buf + g + 2 * stride), v3 = __ldcg(buf + g + 3 * stride);
      s += (v0.x + v0.y) + (v1.x + v1.y) + (v2.x + v2.y) + (v3.x + v3.y);
    }
    for (; g < n; g += stride) { const double2 v = __ldcg(buf + g); s += v.x + v.y; }
  }
  if (s == 12345.678) out[t0] = s;
}

}  // namespace arche
