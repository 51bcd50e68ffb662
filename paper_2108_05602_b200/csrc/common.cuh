// common.cuh - small device helpers shared by the fringe-search kernels (product path only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace volks {

typedef unsigned long long u64;

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
// acc += a*b
__device__ __forceinline__ void cmac(float2 &acc, float2 a, float2 b) {
  acc.x = fmaf(a.x, b.x, acc.x); acc.x = fmaf(-a.y, b.y, acc.x);
  acc.y = fmaf(a.x, b.y, acc.y); acc.y = fmaf(a.y, b.x, acc.y);
}
__device__ __forceinline__ float cnorm(float2 a) { return fmaf(a.x, a.x, a.y * a.y); }

// z * exp(-2 pi i K/N) for compile-time K, N (N | 16, 0 <= K < N).  Trivial factors cost nothing.
template <int K, int N>
__device__ __forceinline__ float2 mul_w(float2 z) {
  constexpr int k16 = K * (16 / N);
  static_assert(k16 >= 0 && k16 < 8, "only first-half twiddles");
  constexpr float C1 = 0.92387953251128674f, S1 = 0.38268343236508977f, H = 0.70710678118654752f;
  if constexpr (k16 == 0) return z;
  else if constexpr (k16 == 4) return make_float2(z.y, -z.x);
  else if constexpr (k16 == 2) return make_float2((z.x + z.y) * H, (z.y - z.x) * H);
  else if constexpr (k16 == 6) return make_float2((z.y - z.x) * H, -(z.x + z.y) * H);
  else {
    // general: W = (c, -s), z*W = (x c + y s, y c - x s)
    constexpr float c = (k16 == 1) ? C1 : (k16 == 3) ? S1 : (k16 == 5) ? -S1 : -C1 /*7*/;
    constexpr float s = (k16 == 1) ? S1 : (k16 == 3) ? C1 : (k16 == 5) ? C1 : S1 /*7*/;
    return make_float2(fmaf(z.x, c, z.y * s), fmaf(z.y, c, -z.x * s));
  }
}

// In-register radix-2 decimation-in-frequency FFT of N (power of two <= 16) points, forward
// (negative exponent).  Elements a[OFF + i*1], i < N.  Output is BIT-REVERSED: a[i] = X[brev(i)].
template <int N, int OFF, int TOTAL>
struct FftDif {
  template <int K>
  static __device__ __forceinline__ void stage(float2 (&a)[TOTAL]) {
    if constexpr (K < N / 2) {
      float2 u = a[OFF + K], v = a[OFF + K + N / 2];
      a[OFF + K] = cadd(u, v);
      a[OFF + K + N / 2] = mul_w<K, N>(csub(u, v));
      stage<K + 1>(a);
    }
  }
  static __device__ __forceinline__ void run(float2 (&a)[TOTAL]) {
    if constexpr (N >= 2) {
      stage<0>(a);
      FftDif<N / 2, OFF, TOTAL>::run(a);
      FftDif<N / 2, OFF + N / 2, TOTAL>::run(a);
    }
  }
};

template <int N>
__host__ __device__ constexpr int brev(int i) {
  int r = 0;
  for (int b = 1, n = N >> 1; n >= 1; b <<= 1, n >>= 1)
    if (i & b) r |= n;
  return r;
}

// Delay-spectrum intermediate Y.  Rows of `pitch` complex elements.  When `paired` the two columns
// 2c, 2c+1 of a row share one float4 (re[2c], re[2c+1], im[2c], im[2c+1]) - the layout the packed
// sliding kernel loads straight into (column a, column b) register pairs; otherwise plain float2.
__device__ __forceinline__ float2 ld_y(const float2 *Y, size_t row_elem_off, int d, int paired) {
  if (paired) {
    const float *p = (const float *)(Y + row_elem_off) + ((d >> 1) << 2) + (d & 1);
    return make_float2(__ldg(p), __ldg(p + 2));
  }
  return __ldg(Y + row_elem_off + d);
}

// Peak key: total order (power descending, plane index ascending) as one unsigned 64-bit max.
// power >= 0 so its IEEE bit pattern is monotone.
__device__ __forceinline__ u64 make_key(float p, uint32_t idx) {
  return ((u64)__float_as_uint(p) << 32) | (u64)(0xFFFFFFFFu - idx);
}
__device__ __forceinline__ float key_power(u64 k) { return __uint_as_float((uint32_t)(k >> 32)); }
__device__ __forceinline__ uint32_t key_index(u64 k) { return 0xFFFFFFFFu - (uint32_t)(k & 0xFFFFFFFFu); }

}  // namespace volks
