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

// ---- packed FP32 (sm_100a fma.rn.f32x2 / add / sub / mul .f32x2 -> SASS FFMA2 / FADD2 / FMUL2) ----
typedef unsigned long long f32x2;   // two packed floats (lo, hi) in one 64-bit register pair

__device__ __forceinline__ f32x2 pk(float lo, float hi) { f32x2 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ float lo32(f32x2 v) { float a, b; asm("mov.b64 {%0,%1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); (void)b; return a; }
__device__ __forceinline__ float hi32(f32x2 v) { float a, b; asm("mov.b64 {%0,%1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); (void)a; return b; }
__device__ __forceinline__ f32x2 neg2(f32x2 v) { return pk(-lo32(v), -hi32(v)); }   // folds into an operand modifier
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) { f32x2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) { f32x2 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
// 128-bit read-only load as two register pairs
__device__ __forceinline__ void ldg2(const void *p, f32x2 &a, f32x2 &b) {
  asm volatile("ld.global.nc.v2.b64 {%0,%1}, [%2];" : "=l"(a), "=l"(b) : "l"(p));
}

// complex numbers as packed pairs (lo = re, hi = im)
__device__ __forceinline__ f32x2 c2_from(float2 z) { return pk(z.x, z.y); }
// (y, -x) = -i z : a swap + sign operand modifier for the consuming instruction
__device__ __forceinline__ f32x2 c2_mulnegi(f32x2 z) { return pk(hi32(z), -lo32(z)); }
// z * (c - i s) for real constants c, s:  (x c + y s, y c - x s)
__device__ __forceinline__ f32x2 c2_mulcs(f32x2 z, float c, float s) { return fma2(c2_mulnegi(z), pk(s, s), mul2(z, pk(c, c))); }

// z * w, both packed (re, im):  z wx + (-zy, zx) wy
__device__ __forceinline__ f32x2 c2_mul(f32x2 z, f32x2 w) {
  return fma2(pk(-hi32(z), lo32(z)), pk(hi32(w), hi32(w)), mul2(z, pk(lo32(w), lo32(w))));
}

// w[m] = tab[m ts] for m = 1..15 (tab[k] = exp(-2 pi i k/n): powers of one root).  Only m = 1 and 4 are read
// - lanes read the table with a stride of m entries, and 15 such reads per thread saturate L1 (ncu: 60 % of
// k_rowbig's and 90 % of k_row3's L1 sectors) - the others are products, at most four deep.
__device__ __forceinline__ void c2_powers16(const float2 *tab, int ts, f32x2 (&w)[16]) {
  w[0] = pk(1.f, 0.f);
  w[1] = c2_from(__ldg(tab + ts)); w[4] = c2_from(__ldg(tab + 4 * ts));
  w[2] = c2_mul(w[1], w[1]); w[8] = c2_mul(w[4], w[4]);
  w[3] = c2_mul(w[2], w[1]); w[5] = c2_mul(w[4], w[1]); w[6] = c2_mul(w[4], w[2]); w[7] = c2_mul(w[4], w[3]);
#pragma unroll
  for (int m = 1; m < 8; ++m) w[8 + m] = c2_mul(w[8], w[m]);
}

// z * exp(-2 pi i K/N), N in {2,4,8,16,32}, 0 <= K < N/2, compile time
template <int K, int N>
__device__ __forceinline__ f32x2 c2_mul_w(f32x2 z) {
  constexpr int k32 = K * (32 / N);
  static_assert(k32 >= 0 && k32 < 16, "first-half twiddles only");
  constexpr float H = 0.70710678118654752f;
  constexpr float C[16] = {1.f, 0.98078528040323043f, 0.92387953251128674f, 0.83146961230254524f, H, 0.55557023301960218f,
                           0.38268343236508977f, 0.19509032201612825f, 0.f, -0.19509032201612825f, -0.38268343236508977f,
                           -0.55557023301960218f, -H, -0.83146961230254524f, -0.92387953251128674f, -0.98078528040323043f};
  constexpr float S[16] = {0.f, 0.19509032201612825f, 0.38268343236508977f, 0.55557023301960218f, H, 0.83146961230254524f,
                           0.92387953251128674f, 0.98078528040323043f, 1.f, 0.98078528040323043f, 0.92387953251128674f,
                           0.83146961230254524f, H, 0.55557023301960218f, 0.38268343236508977f, 0.19509032201612825f};
  if constexpr (k32 == 0) return z;
  else if constexpr (k32 == 8) return c2_mulnegi(z);
  else if constexpr (k32 == 4) return mul2(add2(z, c2_mulnegi(z)), pk(H, H));    // H (x + y, y - x)
  else if constexpr (k32 == 12) return mul2(sub2(c2_mulnegi(z), z), pk(H, H));   // H (y - x, -x - y)
  else return c2_mulcs(z, C[k32], S[k32]);
}

// Packed in-register radix-2 DIF FFT of N (<= 32) points a[OFF .. OFF+N), forward, output
// BIT-REVERSED, only the first NZ inputs non-zero (NZ = N: the plain transform).
template <int N, int NZ, int OFF, int TOTAL>
struct FftDif2 {
  template <int K>
  static __device__ __forceinline__ void stage(f32x2 (&a)[TOTAL]) {
    if constexpr (K < N / 2) {
      if constexpr (NZ <= N / 2) {
        if constexpr (K < NZ) a[OFF + K + N / 2] = c2_mul_w<K, N>(a[OFF + K]);
      } else {
        const f32x2 u = a[OFF + K], v = a[OFF + K + N / 2];
        a[OFF + K] = add2(u, v);
        a[OFF + K + N / 2] = c2_mul_w<K, N>(sub2(u, v));
      }
      stage<K + 1>(a);
    }
  }
  static __device__ __forceinline__ void run(f32x2 (&a)[TOTAL]) {
    if constexpr (N >= 2) {
      stage<0>(a);
      constexpr int NZ2 = NZ < N / 2 ? NZ : N / 2;
      FftDif2<N / 2, NZ2, OFF, TOTAL>::run(a);
      FftDif2<N / 2, NZ2, OFF + N / 2, TOTAL>::run(a);
    }
  }
};

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
