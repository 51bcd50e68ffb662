// kernels_allif.cuh - f2: VOLKS2's own fringe search, one delay across all IFs (Eq. 1).
//
//   k_allif   per (baseline, width, window): A[d] = sum_{t<w} Y[t0+t][d] (the coherent sum of the
//             per-AP all-IF delay spectra, step 6 of the paper), P = |A|^2, the first
//             argmax over the delay axis, and S1 = sum_d P (noise statistic, A3 on the
//             delay axis).  Y[t][d] is the zero-padded FFT of the AP's whole band (all IFs in
//             frequency order) written by the row kernels in their all-IF gather mode.
//
// Overlapping windows slide: A_{j+1} = A_j + sum_{t<s} (Y[t0+w+t] - Y[t0+t]) (no twiddle: rate 0 only;
// 2 s row reads per window instead of w), restarted from a direct sum every `seg` windows like
// kernels_slide.cuh; windows with 2 s > w are summed directly.  A sample leaves a rounding residue of
// about 6e-8 of its size in the running sum; when the window energy (from the per-AP energies, tracked
// as a float sliding sum, re-summed exactly at every restart: FP64 adds would cost more than the whole
// step on this part) falls below 1e-3 of the largest since the last exact sum, the window is summed
// directly again (a uniform decision: every thread evaluates the same scalars).
// A CTA owns all delay columns of its windows (thread = CP column pairs, packed FP32) - or, beyond 8192
// columns, one of the `gsplit` interleaved sub-rows of 8192: per 16 windows one barrier and fixed-order reductions;
// the parts' keys meet in an atomicMax (exact, order-free), their power sums in `gsplit` slots per
// window that the finalize adds in order (deterministic).
#pragma once
#include "common.cuh"

namespace volks {

constexpr int AI_MAXWARPS = 32;

struct AllifArgs {
  const float2 *Y;      // [nbl_chunk][nap][pitch] all-IF delay spectra, pair-interleaved rows
  u64 *keys;            // canonical window keys
  float *noise;         // canonical per-window noise = S1 / nfa
  const float *E;       // per-AP band energies [npairs_total][nap] (row kernel): detects energy collapse
  long long per_pair, offc, pair0;
  int nap, nf, w, stride, nwin, seg, nseg, pitch;
  int dlo, dhi;         // restricted delay search range (true bins, wrapping when dlo > dhi; dlo < 0: whole axis): the
                        // argmax looks at these bins only, the noise sum S1 runs over the whole axis
  int gsplit;           // nfa > 8192: nf = gsplit * 8192, column c of a row is sub-row rho = c / 8192, d' = c % 8192,
                        // delay d = gsplit d' + rho; one CTA per (baseline, segment, sub-row) (CP = 4);
                        // keys combine by atomicMax, the noise as gsplit partial sums added in order by the finalize
};

// CP = column pairs per thread (nf / gsplit / 2 / blockDim.x); SPLIT = (gsplit > 1), a compile-time switch
// so that the one-CTA form keeps its shorter address arithmetic
template <int CP, bool SPLIT>
__global__ void __launch_bounds__(1024) k_allif(AllifArgs a) {
  __shared__ u64 kslot[16][AI_MAXWARPS];
  __shared__ float sslot[16][AI_MAXWARPS];
  const int nwarps = blockDim.x >> 5, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int gs = SPLIT ? a.gsplit : 1;
  const int gpart = SPLIT ? blockIdx.x % gs : 0;
  const int sg = (blockIdx.x / gs) % a.nseg;
  const long long pl = blockIdx.x / (gs * a.nseg);
  const uint32_t pair_base = SPLIT ? (uint32_t)gpart * (uint32_t)(a.nf / 2 / gs) : 0u;   // first column pair of this part
  const char *ybase = (const char *)(a.Y + (size_t)pl * a.nap * a.pitch) + (size_t)pair_base * 16u;
  const size_t rowb = (size_t)a.pitch * 8u;
  const long long c0 = (a.pair0 + pl) * a.per_pair + a.offc;
  const int j0 = sg * a.seg, j1 = min(a.nwin, j0 + a.seg);
  const bool slide = 2 * a.stride <= a.w;

  f32x2 AX[CP], AY[CP];
  auto direct = [&](int t0) {
#pragma unroll
    for (int i = 0; i < CP; ++i) { AX[i] = pk(0.f, 0.f); AY[i] = pk(0.f, 0.f); }
    for (int t = 0; t < a.w; ++t) {
#pragma unroll
      for (int i = 0; i < CP; ++i) {
        f32x2 x, y;
        ldg2(ybase + (size_t)(t0 + t) * rowb + (size_t)(threadIdx.x + i * blockDim.x) * 16u, x, y);
        AX[i] = add2(AX[i], x); AY[i] = add2(AY[i], y);
      }
    }
  };
  const float *Ep = a.E + (a.pair0 + pl) * (long long)a.nap;
  float es = 0.f, esmax = 0.f;
  auto energy = [&](int t0) { float s = 0.f; for (int t = 0; t < a.w; ++t) s += __ldg(Ep + t0 + t); return s; };
  if (slide) {
    direct(j0 * a.stride);
    es = esmax = energy(j0 * a.stride);
  }

  for (int jb = j0; jb < j1; jb += 16) {
    const int nst = min(16, j1 - jb);
    for (int b = 0; b < nst; ++b) {
      const int j = jb + b;
      if (!slide) direct(j * a.stride);
      // energy of the NEXT window, loaded now so that the decision below does not wait on memory
      float es_next = es;
      if (slide && j + 1 < j1)
        for (int t = 0; t < a.stride; ++t)
          es_next += __ldg(Ep + j * a.stride + t + a.w) - __ldg(Ep + j * a.stride + t);
      // power, thread-local best (power bits, then lowest column) and power sum
      uint32_t pb = 0, db = 0xFFFFFFFFu;
      float ps = 0.f;
#pragma unroll
      for (int i = 0; i < CP; ++i) {
        const f32x2 pw = fma2(AY[i], AY[i], mul2(AX[i], AX[i]));
        // true delay bins of the pair (d' and d' + 1 of sub-row rho = gpart: d = psub d' + rho)
        const uint32_t dp = 2u * (uint32_t)(threadIdx.x + i * blockDim.x);
        const uint32_t d0 = SPLIT ? dp * (uint32_t)gs + (uint32_t)gpart : dp, d1 = d0 + (uint32_t)gs;
        const uint32_t p0 = __float_as_uint(lo32(pw)), p1 = __float_as_uint(hi32(pw));
        const bool in0 = a.dlo < 0 || (a.dlo <= a.dhi ? ((int)d0 >= a.dlo && (int)d0 <= a.dhi) : ((int)d0 >= a.dlo || (int)d0 <= a.dhi));
        const bool in1 = a.dlo < 0 || (a.dlo <= a.dhi ? ((int)d1 >= a.dlo && (int)d1 <= a.dhi) : ((int)d1 >= a.dlo || (int)d1 <= a.dhi));
        if (in0 && (p0 > pb || (p0 == pb && d0 < db))) { pb = p0; db = d0; }
        if (in1 && (p1 > pb || (p1 == pb && d1 < db))) { pb = p1; db = d1; }
        ps += lo32(pw) + hi32(pw);
      }
      const uint32_t km = __reduce_max_sync(0xffffffffu, pb);
      const uint32_t dm = __reduce_min_sync(0xffffffffu, pb == km ? db : 0xFFFFFFFFu);
#pragma unroll
      for (int o = 16; o >= 1; o >>= 1) ps += __shfl_xor_sync(0xffffffffu, ps, o);
      // (a warp none of whose columns lies in the range: dm = 2^32 - 1, the lowest key there is: it never wins)
      if (lane == 0) { kslot[b][warp] = dm == 0xFFFFFFFFu ? 0ull : make_key(__uint_as_float(km), dm); sslot[b][warp] = ps; }
      // next window
      if (slide && j + 1 < j1) {
        const int t0 = j * a.stride;
        es = es_next;
        if (es < 1e-3f * esmax) {         // energy collapse: the residue of what left would dominate - sum exactly
          direct(t0 + a.stride);
          es = esmax = energy(t0 + a.stride);
          continue;
        }
        esmax = es > esmax ? es : esmax;
        for (int t = 0; t < a.stride; ++t) {
#pragma unroll
          for (int i = 0; i < CP; ++i) {
            f32x2 xi, yi, xo, yo;
            const size_t co = (size_t)(threadIdx.x + i * blockDim.x) * 16u;
            ldg2(ybase + (size_t)(t0 + t + a.w) * rowb + co, xi, yi);
            ldg2(ybase + (size_t)(t0 + t) * rowb + co, xo, yo);
            AX[i] = add2(AX[i], sub2(xi, xo)); AY[i] = add2(AY[i], sub2(yi, yo));
          }
        }
      }
    }
    __syncthreads();
    if (threadIdx.x < nst) {      // (a warp-per-window shuffle tree here measured slower: 6.6 -> 7.1 ms per width)
      u64 k = kslot[threadIdx.x][0];
      float s = sslot[threadIdx.x][0];
      for (int i = 1; i < nwarps; ++i) {
        k = kslot[threadIdx.x][i] > k ? kslot[threadIdx.x][i] : k;
        s += sslot[threadIdx.x][i];
      }
      if (!SPLIT) a.keys[c0 + jb + threadIdx.x] = k;
      else atomicMax(a.keys + c0 + jb + threadIdx.x, k);
      a.noise[(c0 + jb + threadIdx.x) * gs + gpart] = s / (float)a.nf;
    }
    __syncthreads();
  }
}

}  // namespace volks
