// kernels_probe.cuh - measurement helper (not on the search path): the FP32 FMA issue peak of the device
// at the clocks it runs at, the denominator of bench.py's "alu" roofline.
//
//   k_fp32_probe   every thread runs 8 independent FFMA chains (register operands, no memory traffic), 32
//                  FFMA per loop trip; 8 CTAs of 256 threads per SM = 64 resident warps.  On B200 this issues
//                  3.95 of the 4 warp-instructions per cycle per SM (profiles/r02_fp32_peak.md), i.e. the
//                  number it returns is what FMA-only code can reach, not a data-sheet figure.
#pragma once
#include "common.cuh"

namespace volks {

__global__ void __launch_bounds__(256) k_fp32_probe(float *out, int iters, float a, float b) {
  float x[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) x[k] = (float)(threadIdx.x + k) * 1e-3f;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int k = 0; k < 8; ++k) x[k] = fmaf(x[k], a, b);
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += x[k];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;   // keeps the chains alive
}

}  // namespace volks
