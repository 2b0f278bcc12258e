// peak.cuh -- FP64 issue-rate microbenchmarks behind chorus_fp64_peak (measurement only).
// mode 0: dependent-free DFMA chains on every warp;  mode 1: DMMA.8x8x4 chains on every warp;
// mode 2: even warps DFMA, odd warps DMMA (do the two share one pipe?).
#pragma once
#include <cuda_runtime.h>

namespace chorus {

template <int MODE>
__global__ void __launch_bounds__(256) fp64_peak_kernel(int iters, double seed, double* out) {
  const int warp = threadIdx.x >> 5;
  const bool mma = MODE == 1 || (MODE == 2 && (warp & 1));
  double acc[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) acc[k] = seed + k + threadIdx.x;
  const double a = 1.0 + 1e-9 * seed, b = 1e-9 + seed;
  if (!mma) {
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int rep = 0; rep < 4; ++rep)
#pragma unroll
        for (int k = 0; k < 16; ++k) acc[k] = fma(acc[k], a, b);     // 64 DFMA per thread per iteration
    }
  } else {
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int k = 0; k < 16; k += 2)                                 // 8 DMMA per warp per iteration = 8*256 FMA
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                     : "+d"(acc[k]), "+d"(acc[k + 1]) : "d"(a), "d"(b));
    }
  }
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < 16; ++k) s += acc[k];
  if (s == 12345.678) out[0] = s;   // keep the chains alive
}

}  // namespace chorus
