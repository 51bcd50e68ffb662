// kernels_colfft2.cuh - k_colfft (kernels_colfft.cuh) for Nt = 256 / 512 (L1 = 16 / 32) with TWO delay columns
// per thread in the split format of kernels_slide.cuh: X = (Re z_a, Re z_b), Y = (Im z_a, Im z_b).
//
//   k_colfft2<L1, NZ>   a4+a5+a6 for every window of one width; the decomposition
//                       t = t2 + 16 t1, r = rho + L1 s is the one of k_colfft.
//
// Why: with one complex number per register pair every non-trivial twiddle (and the power) needs the
// (im, re) swap of the pair - register moves and ALU work next to each FMUL2/FFMA2 - and the pair-interleaved
// delay spectra (common.cuh ld_y) are gathered with two 32-bit loads per element.  In the split format a row
// of the pair is ONE 128-bit load, z * w is four FFMA2/FMUL2 for two columns with no moves, -i z is a
// renaming, and |z|^2 of both columns is FMUL2 + FFMA2.
//
// CTA = 512 threads = a 32-column strip (16 column pairs) x a range of consecutive windows.
// pass 1: thread = (t2, column pair, parity hb of rho); warp = (hb, t2 in {w/2, w/2 + 8}).  The first DIF
//         stage of the L1-point transform over t1 separates even and odd rho, so each parity is an
//         (L1/2)-point pruned FFT of its own: e[k] = z[k] + z[k + L1/2],  o[k] = (z[k] - z[k + L1/2]) W_L1^k.
//         Outputs go to shared memory S[rho][t2][pair] as (X, Y) = one float4.
// pass 2: thread = (rho, column pair); warp = two residues.  16 float4 loads, the twiddle W_Nt^{rho t2}
//         (shared table, pre-broadcast), a 16-point DIF FFT, powers, tagged keys (R1), warp max.
#pragma once
#include "common.cuh"
#include "kernels_colfft.cuh"

namespace volks {

// (X + i Y) * exp(-2 pi i K/N) for both columns; N in {2,..,32}, 0 <= K < N/2, compile time
template <int K, int N>
__device__ __forceinline__ void s2_mul_w(f32x2 &X, f32x2 &Y) {
  constexpr int k32 = K * (32 / N);
  static_assert(k32 >= 0 && k32 < 16, "first-half twiddles only");
  constexpr float H = 0.70710678118654752f;
  constexpr float C[16] = {1.f, 0.98078528040323043f, 0.92387953251128674f, 0.83146961230254524f, H, 0.55557023301960218f,
                           0.38268343236508977f, 0.19509032201612825f, 0.f, -0.19509032201612825f, -0.38268343236508977f,
                           -0.55557023301960218f, -H, -0.83146961230254524f, -0.92387953251128674f, -0.98078528040323043f};
  constexpr float S[16] = {0.f, 0.19509032201612825f, 0.38268343236508977f, 0.55557023301960218f, H, 0.83146961230254524f,
                           0.92387953251128674f, 0.98078528040323043f, 1.f, 0.98078528040323043f, 0.92387953251128674f,
                           0.83146961230254524f, H, 0.55557023301960218f, 0.38268343236508977f, 0.19509032201612825f};
  // (x + i y)(c - i s) = (x c + y s) + i (y c - x s)
  if constexpr (k32 == 0) return;
  else if constexpr (k32 == 8) { const f32x2 t = X; X = Y; Y = neg2(t); }
  else if constexpr (k32 == 4) { const f32x2 t = add2(X, Y); Y = mul2(sub2(Y, X), pk(H, H)); X = mul2(t, pk(H, H)); }
  else if constexpr (k32 == 12) { const f32x2 t = sub2(Y, X); Y = mul2(add2(X, Y), pk(-H, -H)); X = mul2(t, pk(H, H)); }
  else {
    constexpr float c = C[k32], s = S[k32];
    const f32x2 t = fma2(X, pk(c, c), mul2(Y, pk(s, s)));
    Y = fma2(Y, pk(c, c), mul2(X, pk(-s, -s)));
    X = t;
  }
}

// Split-format in-register radix-2 DIF FFT of N (<= 16) points (X, Y)[OFF .. OFF+N), forward, output
// BIT-REVERSED, only the first NZ inputs non-zero (NZ = N: the plain transform).
template <int N, int NZ, int OFF, int TOTAL>
struct FftDifS {
  template <int K>
  static __device__ __forceinline__ void stage(f32x2 (&X)[TOTAL], f32x2 (&Y)[TOTAL]) {
    if constexpr (K < N / 2) {
      if constexpr (NZ <= N / 2) {
        if constexpr (K < NZ) {
          X[OFF + K + N / 2] = X[OFF + K]; Y[OFF + K + N / 2] = Y[OFF + K];
          s2_mul_w<K, N>(X[OFF + K + N / 2], Y[OFF + K + N / 2]);
        }
      } else {
        const f32x2 ux = X[OFF + K], uy = Y[OFF + K], vx = X[OFF + K + N / 2], vy = Y[OFF + K + N / 2];
        X[OFF + K] = add2(ux, vx); Y[OFF + K] = add2(uy, vy);
        X[OFF + K + N / 2] = sub2(ux, vx); Y[OFF + K + N / 2] = sub2(uy, vy);
        s2_mul_w<K, N>(X[OFF + K + N / 2], Y[OFF + K + N / 2]);
      }
      stage<K + 1>(X, Y);
    }
  }
  static __device__ __forceinline__ void run(f32x2 (&X)[TOTAL], f32x2 (&Y)[TOTAL]) {
    if constexpr (N >= 2) {
      stage<0>(X, Y);
      constexpr int NZ2 = NZ < N / 2 ? NZ : N / 2;
      FftDifS<N / 2, NZ2, OFF, TOTAL>::run(X, Y);
      FftDifS<N / 2, NZ2, OFF + N / 2, TOTAL>::run(X, Y);
    }
  }
};

// (X, Y)[k] *= W_N^k for k < KN
template <int K, int KN, int N, int TOTAL>
struct S2Twiddle {
  static __device__ __forceinline__ void run(f32x2 (&X)[TOTAL], f32x2 (&Y)[TOTAL]) {
    if constexpr (K < KN) {
      s2_mul_w<K, N>(X[K], Y[K]);
      S2Twiddle<K + 1, KN, N, TOTAL>::run(X, Y);
    }
  }
};

__device__ __forceinline__ void cf2_lds(uint32_t addr, f32x2 &a, f32x2 &b) {
  asm volatile("ld.shared.v2.b64 {%0,%1}, [%2];" : "=l"(a), "=l"(b) : "r"(addr));
}
__device__ __forceinline__ void cf2_sts(uint32_t addr, f32x2 a, f32x2 b) {
  asm volatile("st.shared.v2.b64 [%0], {%1,%2};" ::"r"(addr), "l"(a), "l"(b) : "memory");
}

// pass 1 of one thread: parity HB of rho.  zx/zy: the NZ leading rows t2 + 16 t1 of the column pair.
// bytes between consecutive rho in the strip S[rho][t2][pair]: 256 CP, plus 32 for CP = 4 so that the two groups of
// a quarter warp (rho two apart, 64 B each) fall into different banks
template <int CP> __host__ __device__ constexpr uint32_t cf2_rho_stride() { return 256u * CP + (CP == 4 ? 32u : 0u); }

template <int L1, int NZ, int HB, int CP>
__device__ __forceinline__ void cf2_pass1(const f32x2 (&zx)[NZ], const f32x2 (&zy)[NZ], uint32_t sdst) {
  constexpr int H = L1 / 2;
  constexpr int NZH = NZ < H ? NZ : H;          // non-zero inputs of the half-size transform
  f32x2 X[H], Y[H];
  if constexpr (NZ <= H) {
#pragma unroll
    for (int k = 0; k < NZ; ++k) { X[k] = zx[k]; Y[k] = zy[k]; }
  } else {
#pragma unroll
    for (int k = 0; k < H; ++k) {
      X[k] = HB ? sub2(zx[k], zx[k + H]) : add2(zx[k], zx[k + H]);
      Y[k] = HB ? sub2(zy[k], zy[k + H]) : add2(zy[k], zy[k + H]);
    }
  }
  if constexpr (HB == 1) S2Twiddle<0, NZH, L1, H>::run(X, Y);
  FftDifS<H, NZH, 0, H>::run(X, Y);
  // output i of the half transform is m = brev(i); rho = 2 m + HB
#pragma unroll
  for (int i = 0; i < H; ++i) cf2_sts(sdst + (uint32_t)(2 * brev<H>(i) + HB) * cf2_rho_stride<CP>(), X[i], Y[i]);
}

#ifndef CF2_MIN_CTAS8
#define CF2_MIN_CTAS8 2   // CTAs per SM the CP = 8 variant is compiled for (register cap 128)
#endif
// CP = column pairs per CTA (16: a 32-column strip, 512 threads; 8: a 16-column strip, 256 threads, several CTAs per SM)
// SKIP (candidates-only mode): pass 2 of a (rate residue rho, column) is left out when none of its 16 bins can reach the
// window's pre-threshold.  The bins are F[rho + L1 s] = sum_{t2 < 16} W_16^{s t2} W_Nt^{rho t2} S[rho][t2]: unit-modulus
// multiples of the 16 pass-1 sums the thread has just loaded, so by the triangle and Cauchy-Schwarz inequalities
//   |F[rho + L1 s]|^2 <= (sum_t2 |S[rho][t2]|)^2 <= 16 sum_t2 |S[rho][t2]|^2      for every s.
// For noise the right-hand side lies about 4.8 deviations below the pre-threshold (0.98 of the power a candidate needs)
// whatever the width, so nearly every warp skips the twiddles, the 16-point transform and the powers; a window none of
// whose (rho, column) is evaluated keeps the zero key (not a candidate - all the mode promises).  A candidate's peak
// exceeds the pre-threshold, hence its (rho, column) passes the test and is evaluated exactly as without SKIP.
template <int L1, int NZ, int CP, bool SKIP = false>
__global__ void __launch_bounds__(CP * 32, CP == 8 ? CF2_MIN_CTAS8 : CP == 4 ? 2 * CF2_MIN_CTAS8 : 1) k_colfft2(ColFftArgs a) {
  static_assert(L1 == 16 || L1 == 32, "Nt = 256 or 512");
  static_assert(CP == 16 || CP == 8 || CP == 4, "strip of 32, 16 or 8 columns");
  constexpr int G = 32 / CP;                            // (t2 | rho) groups per warp
  constexpr int NW = CP;                                // warps per CTA
  extern __shared__ float4 cf_sm4[];
  float4 *tw4s = cf_sm4;                                // [NW][16][G] pass-2 twiddles W_Nt^{rho k} (re, re, im, im), rho = 2 (G (warp/2) + hi) + warp%2
  float4 *S4 = cf_sm4 + 512;                            // [L1][16][CP] (X, Y) of a column pair
  u64 *slots = (u64 *)((char *)S4 + (size_t)L1 * cf2_rho_stride<CP>());   // [NW] per-warp window keys
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int cp = lane & (CP - 1), hi = lane / CP;
  const int ntile = a.nf / (2 * CP);
  long long u = blockIdx.x;
  const int rg = (int)(u % a.nrange); u /= a.nrange;
  const int tile = (int)(u % ntile);
  const long long pl = u / ntile;
  const uint32_t rowb = (uint32_t)a.pitch * 8u;
  const char *ybase = (const char *)(a.Y + (size_t)pl * a.nap * a.pitch) + (size_t)(tile * CP + cp) * 16u;
  u64 *keyp = a.keys + ((a.pair0 + pl) * a.per_pair + a.offc);
  // per-warp twiddle rows: the G values a warp reads for one k are adjacent (one conflict-free wavefront, no index arithmetic)
  for (int i = threadIdx.x; i < 512; i += NW * 32) {
    const int wi = i / (16 * G);
    const uint32_t r = (uint32_t)(2 * (G * (wi >> 1) + i % G) + (wi & 1)), k = (uint32_t)((i / G) & 15);
    tw4s[i] = a.tw4[(r * k) & ((uint32_t)a.nt - 1u)];
  }
  const int j0 = rg * a.wpc, j1 = min(a.nwin, j0 + a.wpc);
  __syncthreads();   // twiddle rows visible to both halves
  const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(S4);
  const uint32_t twsrc = (uint32_t)__cvta_generic_to_shared(tw4s) + (uint32_t)(warp * 16 * G + hi) * 16u;
  // pass-1 role
  const int hb = warp & 1, t2 = G * (warp >> 1) + hi;   // the G rows of a warp are adjacent in S
  const uint32_t sdst = sbase + (uint32_t)(t2 * CP + cp) * 16u;
  // pass-2 role
  // the residues of a warp have the warp's parity hb: even and odd rho are two independent pipelines (pass 1 of
  // parity hb feeds only pass 2 of parity hb), each the even / odd warps of the CTA behind its own named barrier
  const uint32_t rho = (uint32_t)(2 * (G * (warp >> 1) + hi) + hb);
  const bool p2_active = (warp >> 1) < L1 / (2 * G);
  auto half_barrier = [&]() { asm volatile("bar.sync %0, %1;" ::"r"(1 + hb), "r"(NW * 16) : "memory"); };
  const uint32_t ssrc = sbase + rho * cf2_rho_stride<CP>() + (uint32_t)cp * 16u;
  constexpr bool PREFETCH = NZ <= 8;                    // NZ = 16 (+ pass 2's 64 registers) would spill

  f32x2 zx[NZ], zy[NZ];
  auto load_window = [&](int j) {
    const size_t t0 = (size_t)j * a.stride;
#pragma unroll
    for (int t1 = 0; t1 < NZ; ++t1) {
      const int t = t2 + 16 * t1;
      if (j < j1 && t < a.w) ldg2(ybase + (t0 + t) * rowb, zx[t1], zy[t1]);
      else { zx[t1] = pk(0.f, 0.f); zy[t1] = pk(0.f, 0.f); }
    }
  };
  if constexpr (PREFETCH) load_window(j0);

  for (int j = j0; j < j1; ++j) {
    if constexpr (!PREFETCH) load_window(j);
    if (hb) cf2_pass1<L1, NZ, 1, CP>(zx, zy, sdst);
    else cf2_pass1<L1, NZ, 0, CP>(zx, zy, sdst);
    if constexpr (PREFETCH) load_window(j + 1);   // in flight during pass 2
    half_barrier();
    if (p2_active) {
      f32x2 X[16], Y[16];
      bool go = true;
      if constexpr (SKIP) {
        const float thrj = __uint_as_float(__ldg(a.thr + pl * a.per_pair + a.offc + j));
        f32x2 e = pk(0.f, 0.f);
#pragma unroll
        for (int k = 0; k < 16; ++k) {
          cf2_lds(ssrc + (uint32_t)k * (16u * CP), X[k], Y[k]);
          e = fma2(X[k], X[k], e);
          e = fma2(Y[k], Y[k], e);
        }
        go = __any_sync(0xffffffffu, 16.0016f * fmaxf(lo32(e), hi32(e)) > thrj);   // warp-uniform
        if (go) {
#pragma unroll
          for (int k = 1; k < 16; ++k) {
            f32x2 wx, wy;
            cf2_lds(twsrc + (uint32_t)k * (16u * G), wx, wy);
            const f32x2 zx2 = X[k], zy2 = Y[k];
            X[k] = fma2(zx2, wx, mul2(zy2, neg2(wy)));
            Y[k] = fma2(zx2, wy, mul2(zy2, wx));
          }
        } else if (lane == 0) {
          slots[warp] = 0ull;
        }
      } else {
#pragma unroll
        for (int k = 0; k < 16; ++k) {
          f32x2 zx2, zy2, wx, wy;
          cf2_lds(ssrc + (uint32_t)k * (16u * CP), zx2, zy2);
          if (k == 0) { X[0] = zx2; Y[0] = zy2; continue; }   // W^0 = 1
          cf2_lds(twsrc + (uint32_t)k * (16u * G), wx, wy);
          // z * w = (zx wx - zy wy) + i (zx wy + zy wx)
          X[k] = fma2(zx2, wx, mul2(zy2, neg2(wy)));
          Y[k] = fma2(zx2, wy, mul2(zy2, wx));
        }
      }
      if (go) {
      FftDifS<16, 16, 0, 16>::run(X, Y);
      // untagged maximum (as k_slide for w >= 16): power and the delay column; the rate bin among the 16 of (rho, column)
      // is k_recover's exact re-evaluation (key = power bits, 2^31 | plane index of the column's bin s = 0)
      uint32_t ba = 0, bb = 0;
#pragma unroll
      for (int i = 0; i < 16; ++i) {
        const f32x2 pw = fma2(Y[i], Y[i], mul2(X[i], X[i]));
        ba = max(ba, __float_as_uint(lo32(pw)));
        bb = max(bb, __float_as_uint(hi32(pw)));
      }
      const bool colb = bb > ba;
      const uint32_t best = colb ? bb : ba;
      const uint32_t km = __reduce_max_sync(0xffffffffu, best);
      const uint32_t tied = __ballot_sync(0xffffffffu, best == km);
      if (lane == __ffs(tied) - 1)
        slots[warp] = ((u64)km << 32) |
                      (u64)(0xFFFFFFFFu - (0x80000000u | (rho * (uint32_t)a.nf + (uint32_t)(tile * 2 * CP + 2 * cp) + (colb ? 1u : 0u))));
      }
    }
    half_barrier();
    if (warp == hb) {   // warps 0 and 1: the slots of their parity
      u64 k = lane < L1 / (2 * G) && lane < NW / 2 ? slots[2 * lane + hb] : 0ull;
#pragma unroll
      for (int o = 8; o >= 1; o >>= 1) {
        const u64 other = __shfl_xor_sync(0xffffffffu, k, o);
        k = other > k ? other : k;
      }
      if (lane == 0) atomicMax(keyp + j, k);
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// k_colfft2e - the SKIP kernel with the energies first (candidates-only mode, 16-column strips).
// ncu on configs[4] had k_colfft2<.., SKIP> bound by the shared-memory data path (75 % busy): every pass-1 sum S[rho][t2]
// of a (window, strip) was written (16 B per column pair) and read back although the bound test only needs |S|^2.  Here a
// pass-1 thread keeps its 16 sums in registers and stores their ENERGIES (8 B per column pair: half the traffic each way);
// the pass-2 threads add the 16 energies of their (rho, column pair), test 16 sum |S|^2 against the window's
// pre-threshold (the Cauchy-Schwarz bound of k_colfft2) and raise a flag for their parity half of the CTA.  Only if the
// flag is up - a window that can hold a candidate in this strip: about one (window, strip) in a hundred - the sums
// themselves are stored, a third barrier is taken and the flagged warps run pass 2 exactly as k_colfft2 does.
#ifndef CF2_ENERGY_FIRST
#define CF2_ENERGY_FIRST 1
#endif
constexpr uint32_t CF2E_RHO = 1024u + 32u;   // bytes between consecutive rho in E[rho][t2][pair]: the two residue groups a
                                             // half warp reads (two rho apart) fall into different banks

template <int L1, int NZ, int HB>
__device__ __forceinline__ void cf2_pass1_keep(const f32x2 (&zx)[NZ], const f32x2 (&zy)[NZ], f32x2 (&X)[L1 / 2], f32x2 (&Y)[L1 / 2]) {
  constexpr int H = L1 / 2;
  constexpr int NZH = NZ < H ? NZ : H;
  if constexpr (NZ <= H) {
#pragma unroll
    for (int k = 0; k < NZ; ++k) { X[k] = zx[k]; Y[k] = zy[k]; }
  } else {
#pragma unroll
    for (int k = 0; k < H; ++k) {
      X[k] = HB ? sub2(zx[k], zx[k + H]) : add2(zx[k], zx[k + H]);
      Y[k] = HB ? sub2(zy[k], zy[k + H]) : add2(zy[k], zy[k + H]);
    }
  }
  if constexpr (HB == 1) S2Twiddle<0, NZH, L1, H>::run(X, Y);
  FftDifS<H, NZH, 0, H>::run(X, Y);          // output i is m = brev(i): rho = 2 m + HB
}

template <int L1, int NZ>
__global__ void __launch_bounds__(256, CF2_MIN_CTAS8) k_colfft2e(ColFftArgs a) {
  static_assert(L1 == 16 || L1 == 32, "Nt = 256 or 512");
  constexpr int CP = 8, G = 32 / CP, NW = CP, H = L1 / 2;
  extern __shared__ float4 cf_sm4[];
  float4 *tw4s = cf_sm4;                                // as in k_colfft2
  float4 *S4 = cf_sm4 + 512;                            // [L1][16][CP] (X, Y) of a column pair
  u64 *slots = (u64 *)((char *)S4 + (size_t)L1 * cf2_rho_stride<CP>());
  // the energy strip E[rho][t2][pair] behind the slots (not inside S: the two parity halves run windows apart, one may
  // store sums while the other still reads energies)
  const uint32_t ebase = (uint32_t)__cvta_generic_to_shared(slots + 16);
  __shared__ int flag_sm[2][2];                         // [parity half][window parity]: some warp of the half passed the test
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int cp = lane & (CP - 1), hi = lane / CP;
  const int ntile = a.nf / (2 * CP);
  long long u = blockIdx.x;
  const int rg = (int)(u % a.nrange); u /= a.nrange;
  const int tile = (int)(u % ntile);
  const long long pl = u / ntile;
  const uint32_t rowb = (uint32_t)a.pitch * 8u;
  const char *ybase = (const char *)(a.Y + (size_t)pl * a.nap * a.pitch) + (size_t)(tile * CP + cp) * 16u;
  u64 *keyp = a.keys + ((a.pair0 + pl) * a.per_pair + a.offc);
  for (int i = threadIdx.x; i < 512; i += NW * 32) {
    const int wi = i / (16 * G);
    const uint32_t r = (uint32_t)(2 * (G * (wi >> 1) + i % G) + (wi & 1)), k = (uint32_t)((i / G) & 15);
    tw4s[i] = a.tw4[(r * k) & ((uint32_t)a.nt - 1u)];
  }
  if (threadIdx.x < 4) ((int *)flag_sm)[threadIdx.x] = 0;
  const int j0 = rg * a.wpc, j1 = min(a.nwin, j0 + a.wpc);
  __syncthreads();
  const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(S4);
  const uint32_t twsrc = (uint32_t)__cvta_generic_to_shared(tw4s) + (uint32_t)(warp * 16 * G + hi) * 16u;
  const int hb = warp & 1, t2 = G * (warp >> 1) + hi;
  const uint32_t sdst = sbase + (uint32_t)(t2 * CP + cp) * 16u;
  const uint32_t edst = ebase + (uint32_t)(t2 * CP + cp) * 8u;
  const uint32_t rho = (uint32_t)(2 * (G * (warp >> 1) + hi) + hb);
  const bool p2_active = (warp >> 1) < L1 / (2 * G);
  auto half_barrier = [&]() { asm volatile("bar.sync %0, %1;" ::"r"(1 + hb), "r"(NW * 16) : "memory"); };
  const uint32_t ssrc = sbase + rho * cf2_rho_stride<CP>() + (uint32_t)cp * 16u;
  const uint32_t esrc = ebase + rho * CF2E_RHO + (uint32_t)cp * 8u;
  constexpr bool PREFETCH = NZ <= 8;                    // (as k_colfft2: NZ = 16 would spill)

  f32x2 zx[NZ], zy[NZ];
  auto load_window = [&](int j) {
    const size_t t0 = (size_t)j * a.stride;
#pragma unroll
    for (int t1 = 0; t1 < NZ; ++t1) {
      const int t = t2 + 16 * t1;
      if (j < j1 && t < a.w) ldg2(ybase + (t0 + t) * rowb, zx[t1], zy[t1]);
      else { zx[t1] = pk(0.f, 0.f); zy[t1] = pk(0.f, 0.f); }
    }
  };
  if constexpr (PREFETCH) load_window(j0);

  for (int j = j0; j < j1; ++j) {
    if constexpr (!PREFETCH) load_window(j);
    f32x2 SX[H], SY[H];                                 // this thread's pass-1 sums: rho = 2 brev(i) + hb, its t2, its column pair
    if (hb) cf2_pass1_keep<L1, NZ, 1>(zx, zy, SX, SY);
    else cf2_pass1_keep<L1, NZ, 0>(zx, zy, SX, SY);
#pragma unroll
    for (int i = 0; i < H; ++i) {
      const f32x2 en = fma2(SY[i], SY[i], mul2(SX[i], SX[i]));
      asm volatile("st.shared.b64 [%0], %1;" ::"r"(edst + (uint32_t)(2 * brev<H>(i) + hb) * CF2E_RHO), "l"(en) : "memory");
    }
    if constexpr (PREFETCH) load_window(j + 1);         // in flight during the test
    half_barrier();
    bool go = false;
    if (p2_active) {
      const float thrj = __uint_as_float(__ldg(a.thr + pl * a.per_pair + a.offc + j));
      f32x2 e = pk(0.f, 0.f);
#pragma unroll
      for (int k = 0; k < 16; ++k) {
        f32x2 en;
        asm volatile("ld.shared.b64 %0, [%1];" : "=l"(en) : "r"(esrc + (uint32_t)k * (8u * CP)));
        e = add2(e, en);
      }
      go = __any_sync(0xffffffffu, 16.0016f * fmaxf(lo32(e), hi32(e)) > thrj);   // warp-uniform
      if (go && lane == 0) flag_sm[hb][j & 1] = 1;
    }
    half_barrier();
    const bool any = flag_sm[hb][j & 1] != 0;           // uniform in the half
    if (warp == hb && lane == 0) flag_sm[hb][(j + 1) & 1] = 0;   // (last read before this window's first barrier)
    if (!any) continue;                                 // no candidate possible in this strip: the window keeps its key
#pragma unroll
    for (int i = 0; i < H; ++i) cf2_sts(sdst + (uint32_t)(2 * brev<H>(i) + hb) * cf2_rho_stride<CP>(), SX[i], SY[i]);
    half_barrier();
    if (p2_active) {
      if (go) {
        f32x2 X[16], Y[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) {
          f32x2 zx2, zy2, wx, wy;
          cf2_lds(ssrc + (uint32_t)k * (16u * CP), zx2, zy2);
          if (k == 0) { X[0] = zx2; Y[0] = zy2; continue; }   // W^0 = 1
          cf2_lds(twsrc + (uint32_t)k * (16u * G), wx, wy);
          X[k] = fma2(zx2, wx, mul2(zy2, neg2(wy)));
          Y[k] = fma2(zx2, wy, mul2(zy2, wx));
        }
        FftDifS<16, 16, 0, 16>::run(X, Y);
        uint32_t ba = 0, bb = 0;
#pragma unroll
        for (int i = 0; i < 16; ++i) {
          const f32x2 pw = fma2(Y[i], Y[i], mul2(X[i], X[i]));
          ba = max(ba, __float_as_uint(lo32(pw)));
          bb = max(bb, __float_as_uint(hi32(pw)));
        }
        const bool colb = bb > ba;
        const uint32_t best = colb ? bb : ba;
        const uint32_t km = __reduce_max_sync(0xffffffffu, best);
        const uint32_t tied = __ballot_sync(0xffffffffu, best == km);
        if (lane == __ffs(tied) - 1)
          slots[warp] = ((u64)km << 32) |
                        (u64)(0xFFFFFFFFu - (0x80000000u | (rho * (uint32_t)a.nf + (uint32_t)(tile * 2 * CP + 2 * cp) + (colb ? 1u : 0u))));
      } else if (lane == 0) {
        slots[warp] = 0ull;
      }
    }
    half_barrier();
    if (warp == hb) {   // warps 0 and 1: the slots of their parity
      u64 k = lane < L1 / (2 * G) && lane < NW / 2 ? slots[2 * lane + hb] : 0ull;
#pragma unroll
      for (int o = 8; o >= 1; o >>= 1) {
        const u64 other = __shfl_xor_sync(0xffffffffu, k, o);
        k = other > k ? other : k;
      }
      if (lane == 0) atomicMax(keyp + j, k);
    }
  }
}

}  // namespace volks
