// kernels_colfft.cuh - rate transform of windows with any stride, Nt = 16 * L1 (L1 = 2..32), as a
// two-pass Cooley-Tukey FFT through shared memory (the "multi-pass path" of configs[4]: the padded
// plane 512 x 2048 exceeds shared memory, so a CTA owns a 32-column strip of it).
//
//   k_colfft<L1>   a4+a5+a6 for every window of one width.
//
// Column d of window (t0, w) on the padded grid Nt = 16 * L1, with t = t2 + 16 t1 and r = rho + L1 s:
//   F[rho + L1 s] = sum_{t2<16} W_16^{s t2} [ W_Nt^{rho t2} Z_{t2}[rho] ],
//   Z_{t2}[rho]   = sum_{t1<L1} y[t0 + t2 + 16 t1] W_{L1}^{rho t1}          (zero for t2 + 16 t1 >= w)
// pass 1: warp t2 (16 warps), lane = column: L1-point packed DIF FFT (common.cuh FftDif2) over t1 in
//         registers, pruned at compile time to the NZ = ceil(w/16) (rounded up to a power of two) leading
//         non-zero inputs; the L1 outputs go to shared memory S[rho][t2][column].
// pass 2: warp <-> residues rho (L1/16 each... one or two per warp), lane = column: 16 shared loads,
//         the twiddle W_Nt^{rho t2} from a shared table, a 16-point DIF FFT in registers, |.|^2, the
//         tagged 32-bit peak key of kernels_slide.cuh (R1), warp redux, one slot per warp;
//         after the pass one thread combines the slots and issues the window's global atomicMax.
// Consecutive windows of a CTA overlap by w - stride samples: their rows stay in L1.
#pragma once
#include "common.cuh"

namespace volks {

constexpr int CF_WARPS = 16;

struct ColFftArgs {
  const float2 *Y;      // [npairs_chunk][nap][pitch]
  u64 *keys;            // canonical window keys
  const float4 *tw4;    // [nt] exp(-2 pi i k/nt), pre-broadcast (re, re, im, im)
  long long per_pair, offc, pair0;
  int nap, nf, w, stride, nt, nwin, pitch, paired;
  int split2;           // host side only: launch k_colfft2 (kernels_colfft2.cuh) where it exists
  int wpc;              // windows per CTA (consecutive)
  int nrange;           // ceil(nwin / wpc)
  uint32_t keymask;     // 0xFFFFFFF0 (register operand of the single-LOP3 key tag)
  // k_colfft2 SKIP (candidates-only mode): pre-threshold of every window of the chunk as float bits (k_winthr),
  // thr[pl * per_pair + offc + j]; nullptr = every (rate residue, column) is transformed
  const uint32_t *thr;
  int energy_first;     // host side only: with thr, launch k_colfft2e (the energies before the sums) instead of k_colfft2<SKIP>
};

// L1 = Nt/16 (2..32), NZ = leading non-zero inputs of the L1-point transform (power of two <= L1).
// Complex values travel as packed pairs (re, im): butterflies are FADD2, twiddles two FFMA2/FMUL2.
template <int L1, int NZ>
__global__ void __launch_bounds__(CF_WARPS * 32) k_colfft(ColFftArgs a) {
  extern __shared__ float4 cf_sm4[];
  float4 *tw4s = cf_sm4;                                // [nt] rate twiddles (re, re, im, im)
  f32x2 *S = (f32x2 *)(cf_sm4 + a.nt);                  // [L1][16][32]
  u64 *slots = (u64 *)(S + (size_t)L1 * 16 * 32);       // [L1] per-residue window keys
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int ntile = a.nf >> 5;
  long long u = blockIdx.x;
  const int rg = (int)(u % a.nrange); u /= a.nrange;
  const int tile = (int)(u % ntile);
  const long long pl = u / ntile;
  const int d = tile * 32 + lane;
  const size_t prow = (size_t)pl * a.nap;
  u64 *keyp = a.keys + ((a.pair0 + pl) * a.per_pair + a.offc);
  for (int i = threadIdx.x; i < a.nt; i += CF_WARPS * 32) tw4s[i] = a.tw4[i];
  const int j0 = rg * a.wpc, j1 = min(a.nwin, j0 + a.wpc);
  const int ntm = a.nt - 1;

  // pass-1 inputs of a window: rows t0 + warp + 16 t1 of this lane's column (zero beyond the window)
  f32x2 zin[NZ];
  auto load_window = [&](int j) {
    const int t0 = j * a.stride;
#pragma unroll
    for (int t1 = 0; t1 < NZ; ++t1) {
      const int t = warp + 16 * t1;
      zin[t1] = (j < j1 && t < a.w) ? c2_from(ld_y(a.Y, (prow + t0 + t) * a.pitch, d, a.paired)) : pk(0.f, 0.f);
    }
  };
  load_window(j0);

  for (int j = j0; j < j1; ++j) {
    // ---- pass 1: warp = t2, L1-point pruned FFT over t1 ----
    {
      const int t2 = warp;
      f32x2 z[L1];
#pragma unroll
      for (int t1 = 0; t1 < NZ; ++t1) z[t1] = zin[t1];
      FftDif2<L1, NZ, 0, L1>::run(z);
#pragma unroll
      for (int i = 0; i < L1; ++i) S[(brev<L1>(i) * 16 + t2) * 32 + lane] = z[i];
    }
    load_window(j + 1);   // in flight during pass 2
    __syncthreads();
    // ---- pass 2: warp = residue rho, 16-point FFT over t2, power, tagged key ----
    // (for L1 = 32 a warp owns two residues and works on both at once: twice the independent work
    //  under each shared-memory load and each dependent FFT stage)
    constexpr int RH = L1 > CF_WARPS ? L1 / CF_WARPS : 1;
    if (warp < L1) {
      f32x2 f[RH][16];
#pragma unroll
      for (int h = 0; h < RH; ++h) {
        const int rho = warp + h * CF_WARPS;
#pragma unroll
        for (int t2 = 0; t2 < 16; ++t2) {
          const f32x2 z = S[(rho * 16 + t2) * 32 + lane];
          const float4 w4 = tw4s[(rho * t2) & ntm];
          // z * w = (zx wx - zy wy, zx wy + zy wx)
          f[h][t2] = fma2(pk(-hi32(z), lo32(z)), pk(w4.z, w4.w), mul2(z, pk(w4.x, w4.y)));
        }
      }
#pragma unroll
      for (int h = 0; h < RH; ++h) FftDif2<16, 16, 0, 16>::run(f[h]);
#pragma unroll
      for (int h = 0; h < RH; ++h) {
        const int rho = warp + h * CF_WARPS;
        uint32_t best = 0;
#pragma unroll
        for (int i = 0; i < 16; ++i) {
          const f32x2 q = mul2(f[h][i], f[h][i]);
          const uint32_t k = (__float_as_uint(lo32(q) + hi32(q)) & a.keymask) | (uint32_t)(15 - brev<16>(i));
          best = max(best, k);
        }
        const uint32_t km = __reduce_max_sync(0xffffffffu, best);
        const uint32_t tied = __ballot_sync(0xffffffffu, best == km);
        if (lane == __ffs(tied) - 1) {
          const uint32_t s = 15u - (km & 15u);
          slots[rho] = make_key(__uint_as_float(km & 0xFFFFFFF0u), (uint32_t)(rho + L1 * s) * (uint32_t)a.nf + (uint32_t)d);
        }
      }
    }
    __syncthreads();
    if (warp == 0) {
      u64 k = lane < L1 ? slots[lane] : 0ull;
#pragma unroll
      for (int o = 16; o >= 1; o >>= 1) {
        const u64 other = __shfl_xor_sync(0xffffffffu, k, o);
        k = other > k ? other : k;
      }
      if (lane == 0) atomicMax(keyp + j, k);
    }
  }
}

}  // namespace volks
