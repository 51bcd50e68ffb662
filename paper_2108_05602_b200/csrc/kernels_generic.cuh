// kernels_generic.cuh - the general (any width / stride / padding) multi-pass fringe-search kernels.
//
//   k_row_fft   a2+a3: slab load, zero-pad, delay FFT of every AP row (PAPER.md:133 step 5), and
//               the per-AP energy sum_k |V|^2 used for the noise statistic (Parseval, A3)
//   k_col<L>    a4+a5+a6: per (window, delay column): zero-padded rate DFT,
//               |.|^2, argmax; per-window max over a total order through 64-bit atomicMax keys
//
// The rate transform of one delay column d of window (t0, w) on the padded grid Nt = L*M is split
// by residue rho = r mod M (Cooley-Tukey, decimation in frequency):
//   F[rho + M s] = sum_{t2<L} e^{-2 pi i s t2/L} a_rho[t2],
//   a_rho[t2]    = sum_{t1: t2+L t1 < w} y[t0 + t2 + L t1] e^{-2 pi i rho (t2 + L t1)/Nt}
// so one thread folds the w samples of its column into L registers and runs an L-point FFT there.
#pragma once
#include <type_traits>
#include "common.cuh"

namespace volks {

// ------------------------------------------------------------------------------------------------
// Row (delay) FFT: radix-4 Stockham autosort passes in shared memory (+ one radix-2 pass when
// log2(nf) is odd).  One group of `tpr` threads per AP row, several rows per CTA.
// vis rows and Y rows are indexed by the flattened (pair, AP) row number.
// ------------------------------------------------------------------------------------------------
struct RowArgs {
  const float2 *vis;   // [rows_total][nchan]
  float2 *Y;           // [nrows][pitch] for rows row0 .. row0+nrows-1 (first nf of each row used)
  float *E;            // [rows_total] per-AP energy
  const float2 *twf;   // [nf] exp(-2 pi i k/nf)
  long long row0, nrows;
  int nchan, nf, tpr, rows_per_cta, pitch, paired;
  // width w == 1 (if the search has one): its plane is the row's delay spectrum repeated over every
  // rate bin, so the peak is max_d |Y[t][d]|^2 at r* = 0 (tie-break A8) and is emitted right here
  u64 *keys1;           // canonical key base of that width (keys + offc), or nullptr
  long long per_pair;   // windows per pair over all widths
  int nap, stride1, nwin1;
  // f1 dedispersion fused into the slab load: element (t, k) of pair (bl, ifq) is
  // read from AP t + shift[ifq][k] (zero beyond the slab); nullptr = no shift
  const int *shift;     // DEVICE [nif][nchan] or nullptr
  int nif;
  // f2 all-IF mode (kernels_allif.cuh): a row is the whole band of one (bl, AP): nchan = nif_src * nchan_src
  // frequency points gathered from vis[bl][n][t][j], m = n * nchan_src + j.  0 = off.
  int allif_nif, allif_nchan;
  // all-IF with nfa = psub * nf (nfa > 8192): AP row t is transformed as psub virtual rows rho = 0..psub-1,
  // delay d = psub d' + rho:  A[rho + psub d'] = sum_m (x[m] W_nfa^{m rho}) W_nf^{m d'};  premod = W_nfa table
  int psub;             // 1 = off
  const float2 *premod; // [psub * nf] exp(-2 pi i k/(psub nf))
  // initial calibration (Eq. 1's last two terms): element (pair, k) is multiplied by
  // cal[pair * nchan + k] (all-IF mode: pair = bl, k = n * nchan_src + j - the same memory layout
  // cf32[nbl][nif][nchan]); nullptr = none
  const float2 *cal;
  // restricted delay search range (volks_options.delay_lo / delay_hi): the delay spectra of the bins
  // outside dlo..dhi (wrapping when dlo > dhi) are written as ZERO, so that no rate kernel can find a peak there, while
  // the noise statistic (the per-AP energies, from the input side) is untouched.  dlo < 0: the whole axis.
  int dlo, dhi;
};

// delay bin d inside the searched range?
__device__ __forceinline__ bool delay_ok(int d, int dlo, int dhi) {
  return dlo < 0 || (dlo <= dhi ? (d >= dlo && d <= dhi) : (d >= dlo || d <= dhi));
}

// index of a row's per-AP energy: every row when psub == 1, else only the rho == 0 sub-row (-1 = none)
__device__ __forceinline__ long long e_index(const RowArgs &a, long long row) {
  if (a.psub == 1) return row;
  return row % a.psub == 0 ? row / a.psub : -1;
}

// Source of one AP row: plain (base pointer), dedispersed (per-channel row offsets), or the all-IF
// band of one (bl, AP) gathered across IFs (with or without dedispersion).
struct RowSrc {
  const float2 *base;   // vis + row * nchan (plain) or vis + pair * nap * nchan (dedispersed / all-IF: pair = bl * nif_src)
  const int *sh;        // shift row of this IF (all-IF: the whole [nif][nchan] table), or nullptr
  int t, nap, nchan, ai_nchan, rho;
  const float2 *premod;
  const float2 *calrow;   // calibration phasors of this row's pair, or nullptr
  bool gather;
  __device__ __forceinline__ RowSrc(const RowArgs &a, long long row) : nap(a.nap), nchan(a.nchan), ai_nchan(a.allif_nchan) {
    rho = 0; premod = nullptr; calrow = nullptr;
    if (a.psub > 1) { rho = (int)(row % a.psub); row /= a.psub; premod = a.premod; }   // uniform branch, rare
    if (a.cal) calrow = a.cal + (row / a.nap) * (long long)a.nchan;
    if (a.allif_nif) {
      const long long bl = row / a.nap;
      t = (int)(row - bl * a.nap);
      base = a.vis + bl * a.allif_nif * a.nap * (long long)a.allif_nchan;
      sh = a.shift; gather = true;
    } else if (a.shift) {
      const long long pair = row / a.nap;
      t = (int)(row - pair * a.nap);
      base = a.vis + pair * a.nap * (long long)a.nchan;
      sh = a.shift + (pair % a.nif) * a.nchan; gather = true;
    } else { base = a.vis + row * (long long)a.nchan; sh = nullptr; t = 0; gather = calrow != nullptr; }
  }
  __device__ __forceinline__ float2 fetch(int k) const {
    if (!sh && !ai_nchan) return __ldg(base + k);   // plain row (only the calibration is applied)
    const int ts = t + (sh ? __ldg(sh + k) : 0);
    if (ts < 0 || ts >= nap) return make_float2(0.f, 0.f);
    if (ai_nchan) {
      const int n = k / ai_nchan, j = k - n * ai_nchan;
      const float2 v = __ldg(base + ((long long)n * nap + ts) * ai_nchan + j);
      return rho ? cmul(v, __ldg(premod + (long long)k * rho)) : v;
    }
    return __ldg(base + (long long)ts * nchan + k);
  }
  __device__ __forceinline__ float2 operator()(int k) const {
    if (!gather) return __ldg(base + k);
    const float2 v = fetch(k);
    return calrow ? cmul(v, __ldg(calrow + k)) : v;
  }
  // The NZ elements k = k0 + m step (m < NZ) of the row, zero from `kmax` on (k_rowbig).  Same values as
  // operator(), but branch-free and without a division per element (the IF index and channel of k advance
  // by step / ai_nchan and step % ai_nchan), so that the NZ shift loads, then the NZ data loads, are all in
  // flight together instead of one dependent chain after another.
  template <int NZ>
  __device__ __forceinline__ void load_strided(int k0, int step, int kmax, float2 (&x)[NZ]) const {
    if (!gather) {
#pragma unroll
      for (int m = 0; m < NZ; ++m) {
        const int k = k0 + m * step;
        x[m] = k < kmax ? __ldg(base + k) : make_float2(0.f, 0.f);
      }
      return;
    }
    // (the mode tests below are uniform branches around whole loops, not per-element predicates)
    int ts[NZ];
    if (sh) {
#pragma unroll
      for (int m = 0; m < NZ; ++m) {
        const int k = k0 + m * step;
        ts[m] = t + __ldg(sh + (k < kmax ? k : 0));
      }
    } else {
#pragma unroll
      for (int m = 0; m < NZ; ++m) ts[m] = t;
    }
    const float2 *p[NZ];      // nullptr = zero
    if (ai_nchan) {
      int n = k0 / ai_nchan, j = k0 - n * ai_nchan;
      const int dq = step / ai_nchan, dr = step - dq * ai_nchan;
#pragma unroll
      for (int m = 0; m < NZ; ++m) {
        const bool ok = k0 + m * step < kmax && (unsigned)ts[m] < (unsigned)nap;
        p[m] = ok ? base + (long long)(n * nap + ts[m]) * ai_nchan + j : nullptr;
        n += dq; j += dr;
        if (j >= ai_nchan) { j -= ai_nchan; ++n; }
      }
    } else {
#pragma unroll
      for (int m = 0; m < NZ; ++m) {
        const int k = k0 + m * step;
        const bool ok = k < kmax && (unsigned)ts[m] < (unsigned)nap;
        p[m] = ok ? base + (long long)ts[m] * nchan + k : nullptr;
      }
    }
#pragma unroll
    for (int m = 0; m < NZ; ++m) x[m] = p[m] ? __ldg(p[m]) : make_float2(0.f, 0.f);
    if (rho) {
      // premodulation W^{k rho} = W^{k0 rho} W^{m step rho}: one strided table read per thread, the other
      // factor is the same address in every thread (a broadcast)
      const float2 pm0 = __ldg(premod + k0 * rho);
#pragma unroll
      for (int m = 0; m < NZ; ++m) x[m] = cmul(x[m], cmul(pm0, __ldg(premod + m * step * rho)));
    }
    if (calrow) {
#pragma unroll
      for (int m = 0; m < NZ; ++m) {
        const int k = k0 + m * step;
        x[m] = cmul(x[m], __ldg(calrow + (k < kmax ? k : 0)));
      }
    }
  }
};

__global__ void __launch_bounds__(512) k_row_fft(RowArgs a) {
  extern __shared__ float2 sm[];
  // a row never spans warps when tpr <= 32: a warp barrier is enough (rows of a CTA are independent)
#define ROW_SYNC() do { if (a.tpr <= 32) __syncwarp(); else __syncthreads(); } while (0)
  const int nf = a.nf, tpr = a.tpr;
  const int rl = threadIdx.x / tpr, lane = threadIdx.x % tpr;
  const long long rrel = (long long)blockIdx.x * a.rows_per_cta + rl;
  const bool live = rrel < a.nrows;
  float2 *buf0 = sm + (size_t)rl * nf;
  float2 *buf1 = sm + (size_t)(a.rows_per_cta + rl) * nf;
  float *esm = (float *)(sm + (size_t)2 * a.rows_per_cta * nf);   // [rows_per_cta][16] warp partials

  float e = 0.f;
  if (live) {
    const RowSrc src(a, a.row0 + rrel);
    for (int k = lane; k < nf; k += tpr) {
      float2 v = make_float2(0.f, 0.f);
      if (k < a.nchan) { v = src(k); e += cnorm(v); }
      buf0[k] = v;
    }
  }
  // energy: fixed tree (shuffle inside the row's lanes of a warp, then warp partials in order)
  {
    const int seg = tpr < 32 ? tpr : 32;
    for (int o = seg >> 1; o >= 1; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
    if (tpr <= 32) {
      if (live && lane == 0) { const long long ei = e_index(a, a.row0 + rrel); if (ei >= 0) a.E[ei] = e; }
    } else {
      if ((lane & 31) == 0) esm[rl * 16 + (lane >> 5)] = e;
    }
  }
  ROW_SYNC();
  if (tpr > 32 && live && lane == 0) {
    float s = 0.f;
    for (int i = 0; i < tpr / 32; ++i) s += esm[rl * 16 + i];
    const long long ei = e_index(a, a.row0 + rrel);
    if (ei >= 0) a.E[ei] = s;
  }

  float2 *in = buf0, *out = buf1;
  int Ns = 1;
  // radix-4 passes
  while (Ns * 4 <= nf) {
    const int nb = nf >> 2;
    if (live)
      for (int j = lane; j < nb; j += tpr) {
        const int k = j & (Ns - 1);
        const int tstep = nf / (Ns * 4);            // table stride for angle unit 1/(4 Ns)
        float2 v0 = in[j], v1 = in[j + nb], v2 = in[j + 2 * nb], v3 = in[j + 3 * nb];
        if (k) {
          v1 = cmul(v1, __ldg(a.twf + k * tstep));
          v2 = cmul(v2, __ldg(a.twf + 2 * k * tstep));
          v3 = cmul(v3, __ldg(a.twf + 3 * k * tstep));
        }
        float2 s02 = cadd(v0, v2), d02 = csub(v0, v2), s13 = cadd(v1, v3), d13 = csub(v1, v3);
        float2 md13 = make_float2(d13.y, -d13.x);   // -i * d13
        const int j0 = ((j - k) << 2) + k;
        out[j0] = cadd(s02, s13);
        out[j0 + Ns] = cadd(d02, md13);
        out[j0 + 2 * Ns] = csub(s02, s13);
        out[j0 + 3 * Ns] = csub(d02, md13);
      }
    ROW_SYNC();
    float2 *t = in; in = out; out = t;
    Ns <<= 2;
  }
  if (Ns < nf) {   // one radix-2 pass
    const int nb = nf >> 1;
    if (live)
      for (int j = lane; j < nb; j += tpr) {
        const int k = j & (Ns - 1);
        float2 v0 = in[j], v1 = in[j + nb];
        if (k) v1 = cmul(v1, __ldg(a.twf + k * (nf / (Ns * 2))));
        const int j0 = ((j - k) << 1) + k;
        out[j0] = cadd(v0, v1);
        out[j0 + Ns] = csub(v0, v1);
      }
    ROW_SYNC();
    float2 *t = in; in = out; out = t;
  }
  u64 key = 0;
  if (live) {
    float2 *dst = a.Y + rrel * (long long)a.pitch;
    if (a.paired) {
      for (int c = lane; c < (nf >> 1); c += tpr) {
        float2 v0 = in[2 * c], v1 = in[2 * c + 1];
        if (!delay_ok(2 * c, a.dlo, a.dhi)) v0 = make_float2(0.f, 0.f);
        if (!delay_ok(2 * c + 1, a.dlo, a.dhi)) v1 = make_float2(0.f, 0.f);
        ((float4 *)dst)[c] = make_float4(v0.x, v1.x, v0.y, v1.y);
        const u64 k0 = make_key(cnorm(v0), (uint32_t)(2 * c)), k1 = make_key(cnorm(v1), (uint32_t)(2 * c + 1));
        key = k0 > key ? k0 : key;
        key = k1 > key ? k1 : key;
      }
    } else {
      for (int k = lane; k < nf; k += tpr) {
        const float2 v = delay_ok(k, a.dlo, a.dhi) ? in[k] : make_float2(0.f, 0.f);
        dst[k] = v;
        const u64 kk = make_key(cnorm(v), (uint32_t)k);
        key = kk > key ? kk : key;
      }
    }
  }
  if (a.keys1) {   // uniform branch
    const int seg = tpr < 32 ? tpr : 32;
    for (int o = seg >> 1; o >= 1; o >>= 1) {
      const u64 other = __shfl_xor_sync(0xffffffffu, key, o);
      key = other > key ? other : key;
    }
    u64 *ksm = (u64 *)esm;                      // [rows_per_cta][16] warp partials (reuses the energy area)
    if (tpr > 32) {
      ROW_SYNC();
      if ((lane & 31) == 0) ksm[rl * 16 + (lane >> 5)] = key;
      ROW_SYNC();
      if (lane == 0) for (int i = 0; i < tpr / 32; ++i) key = ksm[rl * 16 + i] > key ? ksm[rl * 16 + i] : key;
    }
    if (live && lane == 0) {
      const long long row = a.row0 + rrel;
      const long long pair = row / a.nap;
      const int t = (int)(row - pair * a.nap);
      const int j = t / a.stride1;
      if (j * a.stride1 == t && j < a.nwin1) a.keys1[pair * a.per_pair + j] = key;
    }
  }
}
#undef ROW_SYNC

// ------------------------------------------------------------------------------------------------
// Row (delay) FFT, register form, for nf = N1 * N2 in {64, 128, 256}: n = n1 + N1 n2, k = N2 k1 + k2,
//   X[N2 k1 + k2] = sum_{n1} W_N1^{n1 k1} [ W_nf^{n1 k2} sum_{n2} x[n1 + N1 n2] W_N2^{n2 k2} ].
// A row is a group of N2 lanes (never spanning warps): step A, lane n1 < N1: N2-point packed DIF FFT
// over n2 in registers, pruned to the NZA leading non-zero inputs (only nchan of nf are non-zero),
// times W_nf^{n1 k2}, into shared memory; step C, lane k2: N1-point FFT over n1, paired store, the
// w = 1 peak.  One warp barrier per row instead of log4(nf) block barriers.
// ------------------------------------------------------------------------------------------------
template <int N1, int N2, int NZA>
__global__ void __launch_bounds__(256) k_row2(RowArgs a) {
  static_assert(N1 <= N2 && N2 <= 16, "row group = N2 lanes");
  constexpr int G = N2, RPC = 256 / G, EP = N2 + 1;
  __shared__ f32x2 ex[RPC * N1 * EP];
  const int g = threadIdx.x / G, l = threadIdx.x % G;
  const long long rrel = (long long)blockIdx.x * RPC + g;
  const bool live = rrel < a.nrows;
  f32x2 *E = ex + g * (N1 * EP);
  float e = 0.f;
  if (l < N1) {
    f32x2 z[N2];
    const RowSrc src(a, live ? a.row0 + rrel : a.row0);
    float2 v[NZA];
    if (!src.gather) {          // unswitched: the plain path keeps its independent, hoistable loads
#pragma unroll
      for (int n2 = 0; n2 < NZA; ++n2) {
        const int n = l + N1 * n2;
        v[n2] = (live && n < a.nchan) ? __ldg(src.base + n) : make_float2(0.f, 0.f);
      }
    } else {
      src.template load_strided<NZA>(l, N1, live ? a.nchan : 0, v);
    }
#pragma unroll
    for (int n2 = 0; n2 < NZA; ++n2) { e += cnorm(v[n2]); z[n2] = c2_from(v[n2]); }
    FftDif2<N2, NZA, 0, N2>::run(z);
    f32x2 w2[16];
    c2_powers16(a.twf, l, w2);                            // W_nf^{n1 m}: two coalesced reads, products (k_row3)
#pragma unroll
    for (int i = 0; i < N2; ++i) {
      const int k2 = brev<N2>(i);
      E[l * EP + k2] = k2 ? c2_mul(z[i], w2[k2]) : z[i];   // W_nf^{n1 k2}, n1 k2 < nf
    }
  }
#pragma unroll
  for (int o = G >> 1; o >= 1; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
  if (live && l == 0) { const long long ei = e_index(a, a.row0 + rrel); if (ei >= 0) a.E[ei] = e; }
  __syncwarp();
  f32x2 v[N1];
#pragma unroll
  for (int n1 = 0; n1 < N1; ++n1) v[n1] = E[n1 * EP + l];
  FftDif2<N1, N1, 0, N1>::run(v);
  u64 key = 0;
  float *dst = (float *)(a.Y + rrel * (long long)a.pitch);
  if (a.dlo >= 0) {   // uniform: restricted delay range - the spectra outside it are written as zero
#pragma unroll
    for (int i = 0; i < N1; ++i)
      if (!delay_ok(N2 * brev<N1>(i) + l, a.dlo, a.dhi)) v[i] = pk(0.f, 0.f);
  }
  // column 2c keeps (re, re') and column 2c + 1 keeps (im, im') of the pair's float4: one 64-bit store per lane
  float *dstl = dst + ((l >> 1) << 2) + ((l & 1) << 1);
#pragma unroll
  for (int i = 0; i < N1; ++i) {
    const float re = lo32(v[i]), im = hi32(v[i]);
    const float got = __shfl_xor_sync(0xffffffffu, (l & 1) ? re : im, 1);
    if (live) *(float2 *)(dstl + 2 * N2 * brev<N1>(i)) = (l & 1) ? make_float2(got, im) : make_float2(re, got);
  }
  if (a.keys1) {   // uniform branch: the w = 1 peaks (power, lowest column) of this row
    float bp = -1.f;
    int bc = 0;
#pragma unroll
    for (int i = 0; i < N1; ++i) {
      const int col = N2 * brev<N1>(i) + l;
      const float pw = fmaf(lo32(v[i]), lo32(v[i]), hi32(v[i]) * hi32(v[i]));
      if (pw > bp || (pw == bp && col < bc)) { bp = pw; bc = col; }
    }
    key = make_key(bp, (uint32_t)bc);
#pragma unroll
    for (int o = G >> 1; o >= 1; o >>= 1) {
      const u64 other = __shfl_xor_sync(0xffffffffu, key, o);
      key = other > key ? other : key;
    }
    if (live && l == 0) {
      const long long row = a.row0 + rrel;
      const long long pair = row / a.nap;
      const int t = (int)(row - pair * a.nap);
      const int j = t / a.stride1;
      if (j * a.stride1 == t && j < a.nwin1) a.keys1[pair * a.per_pair + j] = key;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Row (delay) FFT for nf = 128 as 16 x 8 (n = n1 + 16 n2, k = 8 k1 + k2): a row is a group of EIGHT lanes, every lane
// busy in both steps (k_row2<8, 16, .> leaves half of its 16 lanes idle in step A), four rows per warp, and a CTA walks
// ROW128_RB batches of 32 rows so that a thread's twiddles W_128^{n1 k2} (n1 = l, l + 8) are formed once, not per row.
// ncu on configs[3] (nchan 32): k_row2<8, 16, 4> issued 275 warp instructions per row at 61 % of the HBM bandwidth.
//   step A, lane l: for n1 = l and l + 8 the 8-point packed DIF FFT over n2 pruned to the NZA non-zero inputs (nchan <= 16 NZA),
//           times W_128^{n1 k2}, into shared memory E[n1][k2];  step C, lane k2 = l: 16-point FFT over n1, paired store,
//           per-AP energy, the w = 1 peak - as in k_row2.
// ------------------------------------------------------------------------------------------------
constexpr int ROW128_RB = 4;      // batches of 32 rows per CTA

__device__ __forceinline__ void c2_powers8(const float2 *tab, int ts, f32x2 (&w)[8]) {
  w[0] = pk(1.f, 0.f);
  w[1] = c2_from(__ldg(tab + ts)); w[4] = c2_from(__ldg(tab + 4 * ts));
  w[2] = c2_mul(w[1], w[1]); w[3] = c2_mul(w[2], w[1]);
  w[5] = c2_mul(w[4], w[1]); w[6] = c2_mul(w[4], w[2]); w[7] = c2_mul(w[4], w[3]);
}

template <int NZA>
__global__ void __launch_bounds__(256) k_row128(RowArgs a) {
  constexpr int N1 = 16, N2 = 8, G = 8, RPC = 256 / G, EP = N2 + 1;
  constexpr int GS = N1 * EP + 8;                         // f32x2 per row group: 16 banks between neighbours (no conflicts)
  __shared__ f32x2 ex[RPC * GS];
  const int g = threadIdx.x / G, l = threadIdx.x % G;
  f32x2 *E = ex + g * GS;
  f32x2 wA[8], wB[8];                                     // W_128^{n1 k2} for n1 = l and l + 8
  c2_powers8(a.twf, l, wA);
  c2_powers8(a.twf, l + 8, wB);
  float *dst0 = (float *)a.Y;
  for (int rb = 0; rb < ROW128_RB; ++rb) {
    const long long rfirst = ((long long)blockIdx.x * ROW128_RB + rb) * RPC;
    if (rfirst >= a.nrows) break;                         // (uniform)
    const long long rrel = rfirst + g;
    const bool live = rrel < a.nrows;
    float e = 0.f;
    const RowSrc src(a, live ? a.row0 + rrel : a.row0);
#pragma unroll
    for (int ia = 0; ia < 2; ++ia) {
      const int n1 = l + 8 * ia;
      f32x2 z[N2];
      float2 v[NZA];
      if (!src.gather) {
#pragma unroll
        for (int n2 = 0; n2 < NZA; ++n2) {
          const int n = n1 + N1 * n2;
          v[n2] = (live && n < a.nchan) ? __ldg(src.base + n) : make_float2(0.f, 0.f);
        }
      } else {
        src.template load_strided<NZA>(n1, N1, live ? a.nchan : 0, v);
      }
#pragma unroll
      for (int n2 = 0; n2 < NZA; ++n2) { e += cnorm(v[n2]); z[n2] = c2_from(v[n2]); }
      FftDif2<N2, NZA, 0, N2>::run(z);
#pragma unroll
      for (int i = 0; i < N2; ++i) {
        const int k2 = brev<N2>(i);
        E[n1 * EP + k2] = k2 ? c2_mul(z[i], ia ? wB[k2] : wA[k2]) : z[i];
      }
    }
#pragma unroll
    for (int o = G >> 1; o >= 1; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
    if (live && l == 0) { const long long ei = e_index(a, a.row0 + rrel); if (ei >= 0) a.E[ei] = e; }
    __syncwarp();
    f32x2 v[N1];
#pragma unroll
    for (int n1 = 0; n1 < N1; ++n1) v[n1] = E[n1 * EP + l];
    __syncwarp();                                         // E is rewritten by the next batch
    FftDif2<N1, N1, 0, N1>::run(v);
    float *dst = dst0 + rrel * (long long)a.pitch * 2;
    if (a.dlo >= 0) {   // uniform: restricted delay range - the spectra outside it are written as zero
#pragma unroll
      for (int i = 0; i < N1; ++i)
        if (!delay_ok(N2 * brev<N1>(i) + l, a.dlo, a.dhi)) v[i] = pk(0.f, 0.f);
    }
    // column 2c keeps (re, re') and column 2c + 1 keeps (im, im') of the pair's float4: one 64-bit store per lane
    float *dstl = dst + ((l >> 1) << 2) + ((l & 1) << 1);
#pragma unroll
    for (int i = 0; i < N1; ++i) {
      const float re = lo32(v[i]), im = hi32(v[i]);
      const float got = __shfl_xor_sync(0xffffffffu, (l & 1) ? re : im, 1);
      if (live) *(float2 *)(dstl + 2 * N2 * brev<N1>(i)) = (l & 1) ? make_float2(got, im) : make_float2(re, got);
    }
    if (a.keys1) {   // uniform branch: the w = 1 peaks (power, lowest column) of this row
      float bp = -1.f;
      int bc = 0;
#pragma unroll
      for (int i = 0; i < N1; ++i) {
        const int col = N2 * brev<N1>(i) + l;
        const float pw = fmaf(lo32(v[i]), lo32(v[i]), hi32(v[i]) * hi32(v[i]));
        if (pw > bp || (pw == bp && col < bc)) { bp = pw; bc = col; }
      }
      u64 key = make_key(bp, (uint32_t)bc);
#pragma unroll
      for (int o = G >> 1; o >= 1; o >>= 1) {
        const u64 other = __shfl_xor_sync(0xffffffffu, key, o);
        key = other > key ? other : key;
      }
      if (live && l == 0) {
        const long long row = a.row0 + rrel;
        const long long pair = row / a.nap;
        const int t = (int)(row - pair * a.nap);
        const int j = t / a.stride1;
        if (j * a.stride1 == t && j < a.nwin1) a.keys1[pair * a.per_pair + j] = key;
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Row (delay) FFT, register form, for nf = 256 * N3 (N3 = 2, 4, 8: nf = 512, 1024, 2048 = config 4).
// One row per CTA of 256 threads.  n = n' + 256 n3 (n' < 256), k = N3 k' + k3:
//   X[N3 k' + k3] = sum_{n'} W_256^{n' k'} [ W_nf^{n' k3} sum_{n3} x[n' + 256 n3] W_N3^{n3 k3} ]
// step 1, thread n': N3-point packed DIF FFT over n3 (pruned to the NZA non-zero inputs), twiddle,
//         V[k3][n'] to shared memory;
// step 2, 16-lane group k3: the 256-point transform over n' as in k_row2 (n' = n1 + 16 n2,
//         k' = 16 k1 + k2): lane n1: 16-point FFT over n2, W_256^{n1 k2}, exchange; lane k2: 16-point
//         FFT over n1; results to a shared row image in the pair-interleaved layout;
// step 3: coalesced 128-bit stores of the row, the w = 1 peak.
// ------------------------------------------------------------------------------------------------
template <int N3, int NZA>
__global__ void __launch_bounds__(256) k_row3(RowArgs a) {
  constexpr int NF = 256 * N3, EP = 17;
  __shared__ f32x2 V[NF];               // [k3][n']   (reused as the row image [NF] in step 2b)
  __shared__ f32x2 Ex[N3 * 16 * EP];    // [k3][n1][k2] padded
  __shared__ u64 kred[8];
  __shared__ float ered[8];
  const int tid = threadIdx.x;
  const long long rrel = blockIdx.x;     // one row per CTA; the grid is exactly nrows
  // ---- step 1 ----
  float e = 0.f;
  {
    f32x2 z[N3];
    const RowSrc src(a, a.row0 + rrel);
    float2 v[NZA];
    if (!src.gather) {
#pragma unroll
      for (int n3 = 0; n3 < NZA; ++n3) {
        const int n = tid + 256 * n3;
        v[n3] = n < a.nchan ? __ldg(src.base + n) : make_float2(0.f, 0.f);
      }
    } else {
      src.template load_strided<NZA>(tid, 256, a.nchan, v);
    }
#pragma unroll
    for (int n3 = 0; n3 < NZA; ++n3) { e += cnorm(v[n3]); z[n3] = c2_from(v[n3]); }
    FftDif2<N3, NZA, 0, N3>::run(z);
    // W_nf^{n' k3}: one coalesced table read (k3 = 1), the other powers as products (strided reads of the
    // table were 90 % of this kernel's L1 traffic, and L1 its limit)
    f32x2 w3[8];
    w3[0] = pk(1.f, 0.f); w3[1] = c2_from(__ldg(a.twf + tid));
    w3[2] = c2_mul(w3[1], w3[1]); w3[3] = c2_mul(w3[2], w3[1]); w3[4] = c2_mul(w3[2], w3[2]);
    w3[5] = c2_mul(w3[4], w3[1]); w3[6] = c2_mul(w3[4], w3[2]); w3[7] = c2_mul(w3[4], w3[3]);
#pragma unroll
    for (int i = 0; i < N3; ++i) {
      const int k3 = brev<N3>(i);
      V[k3 * 256 + tid] = k3 ? c2_mul(z[i], w3[k3]) : z[i];
    }
  }
#pragma unroll
  for (int o = 16; o >= 1; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
  if ((tid & 31) == 0) ered[tid >> 5] = e;
  __syncthreads();
  if (tid == 0) {
    float s = 0.f;
    for (int i = 0; i < 8; ++i) s += ered[i];
    const long long ei = e_index(a, a.row0 + rrel);
    if (ei >= 0) a.E[ei] = s;
  }
  // ---- step 2: groups of 16 lanes, group g <-> k3 (N3 <= 16 groups of the 16 available) ----
  const int g = tid >> 4, l = tid & 15;
  if (g < N3) {
    f32x2 z[16];
#pragma unroll
    for (int n2 = 0; n2 < 16; ++n2) z[n2] = V[g * 256 + l + 16 * n2];
    FftDif2<16, 16, 0, 16>::run(z);
    f32x2 *E = Ex + g * (16 * EP);
    f32x2 w2[16];
    c2_powers16(a.twf, l * N3, w2);                        // W_256^{n1 m} = twf[n1 m N3]
#pragma unroll
    for (int i = 0; i < 16; ++i) {
      const int k2 = brev<16>(i);
      E[l * EP + k2] = k2 ? c2_mul(z[i], w2[k2]) : z[i];   // W_256^{n1 k2}
    }
  }
  __syncthreads();                                       // every group is done with V; E complete
  float *img = (float *)V;                               // row image, pair-interleaved floats
  if (g < N3) {
    const f32x2 *E = Ex + g * (16 * EP);
    f32x2 v[16];
#pragma unroll
    for (int n1 = 0; n1 < 16; ++n1) v[n1] = E[n1 * EP + l];
    FftDif2<16, 16, 0, 16>::run(v);
#pragma unroll
    for (int i = 0; i < 16; ++i) {
      const int col = N3 * (16 * brev<16>(i) + l) + g;
      // float4 slot of the column pair, XOR-swizzled by bits 3..5 so that the 16 lanes (column stride N3)
      // spread over the banks instead of hitting two of them
      const int q = col >> 1, qs = q ^ ((q >> 3) & 7);
      float *p = img + (qs << 2) + (col & 1);
      p[0] = lo32(v[i]); p[2] = hi32(v[i]);
    }
  }
  __syncthreads();
  // ---- step 3 ----
  u64 key = 0;
  float4 *dst = (float4 *)(a.Y + rrel * (long long)a.pitch);
  for (int c = tid; c < NF / 2; c += 256) {
    float4 q = ((const float4 *)img)[c ^ ((c >> 3) & 7)];
    if (!delay_ok(2 * c, a.dlo, a.dhi)) { q.x = 0.f; q.z = 0.f; }
    if (!delay_ok(2 * c + 1, a.dlo, a.dhi)) { q.y = 0.f; q.w = 0.f; }
    dst[c] = q;
    if (a.keys1) {   // uniform: the w = 1 peaks
      const u64 k0 = make_key(fmaf(q.x, q.x, q.z * q.z), (uint32_t)(2 * c)), k1 = make_key(fmaf(q.y, q.y, q.w * q.w), (uint32_t)(2 * c + 1));
      key = k0 > key ? k0 : key;
      key = k1 > key ? k1 : key;
    }
  }
  if (a.keys1) {   // uniform branch
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) {
      const u64 other = __shfl_xor_sync(0xffffffffu, key, o);
      key = other > key ? other : key;
    }
    if ((tid & 31) == 0) kred[tid >> 5] = key;
    __syncthreads();
    if (tid == 0) {
      for (int i = 0; i < 8; ++i) key = kred[i] > key ? kred[i] : key;
      const long long row = a.row0 + rrel;
      const long long pair = row / a.nap;
      const int t = (int)(row - pair * a.nap);
      const int j = t / a.stride1;
      if (j * a.stride1 == t && j < a.nwin1) a.keys1[pair * a.per_pair + j] = key;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Row (delay) FFT for large nf = 4096, 8192 (the band transforms of the all-IF search): radix-16 Stockham
// passes with the 16-point butterflies in registers (packed FFT), ONE shared buffer of nf complex used in
// place (every thread reads its 16 inputs, barrier, writes its 16 outputs, barrier), a final radix-2 /
// radix-1 pass... nf = 16^a * R with R in {1, 2, 4, 8}:  4096 = 16^3, 8192 = 16^3 * 2.
// The buffer is padded by one element per 16 (index p -> p + p/16, RBI): the first pass stores 16
// consecutive elements per thread, which would otherwise be a 16-way bank conflict.
// One row per CTA of nf/16 threads.  Pass with Ns = product of the earlier radices, radix R, butterfly j
// (k = j mod Ns):  v[m] = in[j + m nf/R] W_{Ns R}^{k m};  out[(j - k) R + k + m' Ns] = DFT_R(v)[m'].
// ------------------------------------------------------------------------------------------------
#define RBI(p) ((p) + ((p) >> 4))
template <int NZ, bool TW>
__device__ __forceinline__ void rowbig_pass(f32x2 (&v)[16], const RowArgs &a, int j, int Ns, int nf) {
  // twiddles W_{16 Ns}^{k m} = W_nf^{k m nf/(16 Ns)} (m < 16; none in the first pass, k = 0), then the
  // 16-point transform; output bit-reversed.  Only m = 1 and 4 come from the table (lanes read it with a
  // stride of m entries: 15 loads per thread were 60 % of this kernel's L1 traffic); the others are products
  // of at most four of them.
  if constexpr (TW) {
    static_assert(NZ == 16, "later passes are dense");
    f32x2 w[16];
    c2_powers16(a.twf, (j & (Ns - 1)) * (nf / (Ns * 16)), w);
#pragma unroll
    for (int m = 1; m < 16; ++m) v[m] = c2_mul(v[m], w[m]);
  }
  FftDif2<16, NZ, 0, 16>::run(v);
}

template <int NF, int NZ>
__global__ void __launch_bounds__(NF / 16, 2) k_rowbig(RowArgs a) {
  constexpr int T = NF / 16;                     // threads = radix-16 butterflies per pass
  constexpr int RL = NF == 8192 ? 2 : 1;         // last radix (8192 = 16^3 * 2)
  extern __shared__ f32x2 rb[];                  // [NF + NF/16]
  __shared__ u64 kred[16];
  __shared__ float ered[16];
  const int tid = threadIdx.x;
  const long long rrel = blockIdx.x;
  const RowSrc src(a, a.row0 + rrel);
  f32x2 v[16];
  float e = 0.f;
  // ---- pass 1 (Ns = 1): inputs straight from the slab, element tid + m T; only the first NZ of the 16 are non-zero
  {
    float2 x[NZ];
    src.template load_strided<NZ>(tid, T, a.nchan, x);
#pragma unroll
    for (int m = 0; m < NZ; ++m) { e += cnorm(x[m]); v[m] = c2_from(x[m]); }
  }
  rowbig_pass<NZ, false>(v, a, tid, 1, NF);
#pragma unroll
  for (int i = 0; i < 16; ++i) rb[RBI(tid * 16 + brev<16>(i))] = v[i];     // (j - k) R + k + m' Ns with Ns = 1, k = 0
#pragma unroll
  for (int o = 16; o >= 1; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
  if ((tid & 31) == 0) ered[tid >> 5] = e;
  __syncthreads();
  if (tid == 0) {
    float s = 0.f;
    for (int i = 0; i < T / 32; ++i) s += ered[i];
    const long long ei = e_index(a, a.row0 + rrel);
    if (ei >= 0) a.E[ei] = s;
  }
  // ---- passes 2, 3 (Ns = 16, 256): radix 16 in place
#pragma unroll
  for (int Ns = 16; Ns <= 256; Ns *= 16) {
#pragma unroll
    for (int m = 0; m < 16; ++m) v[m] = rb[RBI(tid + m * T)];
    __syncthreads();
    rowbig_pass<16, true>(v, a, tid, Ns, NF);
    const int k = tid & (Ns - 1), j0 = (tid - k) * 16 + k;
#pragma unroll
    for (int i = 0; i < 16; ++i) rb[RBI(j0 + brev<16>(i) * Ns)] = v[i];
    __syncthreads();
  }
  // ---- store: pair-interleaved float4 rows, the w = 1 peak
  u64 key = 0;
  float4 *dst = (float4 *)(a.Y + rrel * (long long)a.pitch);
  const int psub = a.psub, srho = src.rho;
  auto emit = [&](int c, f32x2 z0, f32x2 z1) {   // columns 2c, 2c + 1 (true delay bin of column d': psub d' + rho)
    float4 q = make_float4(lo32(z0), lo32(z1), hi32(z0), hi32(z1));
    if (!delay_ok(2 * c * psub + srho, a.dlo, a.dhi)) { q.x = 0.f; q.z = 0.f; }
    if (!delay_ok((2 * c + 1) * psub + srho, a.dlo, a.dhi)) { q.y = 0.f; q.w = 0.f; }
    dst[c] = q;
    if (a.keys1) {   // uniform
      const u64 k0 = make_key(fmaf(q.x, q.x, q.z * q.z), (uint32_t)(2 * c)), k1 = make_key(fmaf(q.y, q.y, q.w * q.w), (uint32_t)(2 * c + 1));
      key = k0 > key ? k0 : key;
      key = k1 > key ? k1 : key;
    }
  };
  if constexpr (RL == 2) {
    // last pass (Ns = 4096, radix 2) for nf = 8192, fused with the store: out[j] = lo[j] + W_8192^j hi[j],
    // out[j + 4096] = lo[j] - W_8192^j hi[j].  Thread: column pairs c = tid + 512 q (q < 4), j = 2c, 2c + 1;
    // W^{2c} = W^{2 tid} W_8^q: two table reads per thread, the W_8^q are compile-time constants.
    const f32x2 wa = c2_from(__ldg(a.twf + 2 * tid)), wb = c2_from(__ldg(a.twf + 2 * tid + 1));
    auto last = [&](auto qc) {
      constexpr int q = decltype(qc)::value;
      const int c = tid + q * T;
      const f32x2 lo0 = rb[RBI(2 * c)], lo1 = rb[RBI(2 * c + 1)];
      const f32x2 h0 = c2_mul(rb[RBI(2 * c + NF / 2)], c2_mul_w<q, 8>(wa));
      const f32x2 h1 = c2_mul(rb[RBI(2 * c + 1 + NF / 2)], c2_mul_w<q, 8>(wb));
      emit(c, add2(lo0, h0), add2(lo1, h1));
      emit(c + NF / 4, sub2(lo0, h0), sub2(lo1, h1));
    };
    last(std::integral_constant<int, 0>{}); last(std::integral_constant<int, 1>{});
    last(std::integral_constant<int, 2>{}); last(std::integral_constant<int, 3>{});
  } else {
    for (int c = tid; c < NF / 2; c += T) emit(c, rb[RBI(2 * c)], rb[RBI(2 * c + 1)]);
  }
  if (a.keys1) {   // uniform branch
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) {
      const u64 other = __shfl_xor_sync(0xffffffffu, key, o);
      key = other > key ? other : key;
    }
    if ((tid & 31) == 0) kred[tid >> 5] = key;
    __syncthreads();
    if (tid == 0) {
      for (int i = 0; i < T / 32; ++i) key = kred[i] > key ? kred[i] : key;
      const long long row = a.row0 + rrel;
      const long long pair = row / a.nap;
      const int t = (int)(row - pair * a.nap);
      const int jw = t / a.stride1;
      if (jw * a.stride1 == t && jw < a.nwin1) a.keys1[pair * a.per_pair + jw] = key;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Column (rate) transform + power + argmax, generic.
// Thread task id (d fastest): ((pair_local * nwin + j) * M + rho) * nf + d.
// ------------------------------------------------------------------------------------------------
struct ColArgs {
  const float2 *Y;      // [npairs_chunk][nap][pitch]
  u64 *keys;            // canonical window keys
  const float2 *twt;    // [nt] exp(-2 pi i k/nt)
  long long total;      // number of thread tasks
  long long per_pair;   // windows per (bl, ifq) pair over all widths
  long long offc;       // canonical offset of this width inside a pair
  long long pair0;      // first pair of the chunk
  int nap, nf, log2nf, w, stride, nt, log2m, nwin, pitch, paired;
};

template <int L>
__global__ void __launch_bounds__(256) k_col(ColArgs a) {
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const bool live = gid < a.total;
  const int M = 1 << a.log2m;
  u64 key = 0;
  long long c = 0;
  if (live) {
    const int d = (int)(gid & (a.nf - 1));
    long long rest = gid >> a.log2nf;
    const int rho = (int)(rest & (M - 1));
    rest >>= a.log2m;
    const int j = (int)(rest % a.nwin);
    const long long pl = rest / a.nwin;
    c = (a.pair0 + pl) * a.per_pair + a.offc + j;
    const int t0 = j * a.stride;
    const size_t row0 = (size_t)(pl * a.nap + t0) * a.pitch;
    float2 acc[L];
#pragma unroll
    for (int i = 0; i < L; ++i) acc[i] = make_float2(0.f, 0.f);
    const int ntm = a.nt - 1;
    for (int tb = 0; tb < a.w; tb += L) {
#pragma unroll
      for (int t2 = 0; t2 < L; ++t2) {
        const int t = tb + t2;
        if (t < a.w) {
          const float2 y = ld_y(a.Y, row0 + (size_t)t * a.pitch, d, a.paired);
          const float2 tw = __ldg(a.twt + ((rho * t) & ntm));
          cmac(acc[t2], y, tw);
        }
      }
    }
    FftDif<L, 0, L>::run(acc);
    float best = -1.f;
    int bs = 0;
#pragma unroll
    for (int s = 0; s < L; ++s) {
      const float p = cnorm(acc[brev<L>(s)]);
      if (p > best) { best = p; bs = s; }
    }
    const uint32_t r = (uint32_t)(rho + (bs << a.log2m));
    key = make_key(best, r * (uint32_t)a.nf + (uint32_t)d);
  }
  if ((long long)a.nf << a.log2m >= 32) {
    // all 32 lanes belong to one window (tasks per window is a multiple of 32)
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) {
      const u64 other = __shfl_xor_sync(0xffffffffu, key, o);
      key = other > key ? other : key;
    }
    if (live && (threadIdx.x & 31) == 0) atomicMax(a.keys + c, key);
  } else if (live) {
    atomicMax(a.keys + c, key);
  }
}

// ------------------------------------------------------------------------------------------------
// Finalize: SNR, threshold, dense peaks, ordered compaction (count -> scan -> scatter).
// ------------------------------------------------------------------------------------------------
struct Sched {   // the window schedule (device copy lives in the plan)
  int nwidths, nbl, nif, nap, nf, log2nf;
  int allif;              // f2: one delay across all IFs (pairs = baselines; records carry ifq = -1)
  int ngs;                // f2: partial noise sums per window (k_allif's gsplit), 1 otherwise
  float snr_thresh;
  int dlo, dhi, dfirst;   // restricted delay range (dlo < 0: none); dfirst = the lowest searched delay bin
  long long per_pair, nwin_total;
  int width[16], stride[16], nt[16];
  long long nwin[16];     // windows per pair
  long long offc[16];     // canonical offset inside a pair
  long long offd[16];     // dense-layout offset: npair * sum_{q'<q} nwin
};

struct WinStat { float power, snr; int rate_idx, delay_idx, q, j, t0; long long pair; };

// the CTA's shared copy of the schedule, word by word by all threads (one thread copying 640 bytes was a quarter of
// k_finalize on a candidates-only search, where the rest of the kernel is a scan of the keys); caller synchronises
__device__ __forceinline__ void sched_load(Sched &dst, const Sched *src) {
  static_assert(sizeof(Sched) % 4 == 0, "copied as 32-bit words");
  for (int i = threadIdx.x; i < (int)(sizeof(Sched) / 4); i += blockDim.x) ((uint32_t *)&dst)[i] = ((const uint32_t *)src)[i];
}

// Selection statistic: the in-plane amplitude snr (a7), or - when `zst` is given (f4, the other reading
// of PAPER.md:196) - the peak power normalised ACROSS the windows of its (pair, width) series:
// z = (P1 - mean) * inv_std with zst[pair * nwidths + q] = (mean, 1/std) (inv_std = 0 when std = 0).
// In that mode the z-score is what the record's `snr` field carries.
// `noise` (f2): the per-window noise written by k_allif (mean of P over the delay axis) replaces the
// Parseval sum of per-AP energies, which still decides whether the window is identically zero.
__device__ __forceinline__ WinStat window_stat(const Sched &s, const u64 *keys, const float *E, long long c,
                                               const double2 *zst = nullptr, const float *noise = nullptr) {
  WinStat o;
  o.pair = c / s.per_pair;
  long long rem = c - o.pair * s.per_pair;
  int q = 0;
  while (q + 1 < s.nwidths && rem >= s.nwin[q]) { rem -= s.nwin[q]; ++q; }
  o.q = q; o.j = (int)rem; o.t0 = o.j * s.stride[q];
  const u64 k = keys[c];
  o.power = key_power(k);
  if (o.power == 0.f) {
    // a zero key: an all-zero window, or one the candidates-only mode did not evaluate (pruned, skipped): power 0 at
    // the first searched bin, snr 0 - the window energy is not needed (most windows of a pruned search end here)
    o.rate_idx = 0; o.delay_idx = s.dfirst; o.snr = 0.f;
    if (zst) { const double2 ms = zst[o.pair * s.nwidths + q]; o.snr = (float)((0.0 - ms.x) * ms.y); }
    return o;
  }
  const uint32_t idx = key_index(k);
  o.rate_idx = (int)(idx >> s.log2nf);
  o.delay_idx = (int)(idx & (uint32_t)(s.nf - 1));
  // noise = mean |F|^2 over the padded plane = sum over the window of |V|^2 (Parseval)
  const float *e = E + o.pair * s.nap + o.t0;
  float es = 0.f;
  for (int t = 0; t < s.width[q]; ++t) es += e[t];
  float nz = es;
  // (a w = 1 window's peak comes from the row kernel; its mean of P over the delay axis IS the AP's energy)
  if (noise && s.width[q] > 1) { nz = 0.f; for (int g = 0; g < s.ngs; ++g) nz += noise[c * s.ngs + g]; }
  o.snr = (es > 0.f && nz > 0.f) ? sqrtf(o.power / nz) : 0.f;
  // an all-zero window (flagged data, the zero fill of dedispersion) has an identically zero plane:
  // P1 = 0 at (0, 0) by the tie rule.  The sliding sum would leave rounding residue of earlier samples
  // here, so the exact statement is made from the energy (es == 0 iff every sample is zero).
  // (with a restricted delay range the first searched bin is (0, dfirst); a plane whose searched bins are all zero
  //  reports it too)
  if (es == 0.f || o.power == 0.f) { o.power = 0.f; o.rate_idx = 0; o.delay_idx = s.dfirst; }
  if (zst) {
    const double2 ms = zst[o.pair * s.nwidths + q];
    o.snr = (float)(((double)o.power - ms.x) * ms.y);
  }
  return o;
}

// f4: mean and 1/std (population) of the peak-power series of one (pair, width); one CTA per series,
// double accumulation in a fixed order (deterministic).
__global__ void __launch_bounds__(256) k_zstat(const Sched *sp, const u64 *keys, const float *E, double2 *zst,
                                               const float *noise) {
  __shared__ Sched s;
  __shared__ double sh1[256], sh2[256];
  if (threadIdx.x == 0) s = *sp;
  __syncthreads();
  const long long pair = blockIdx.x / s.nwidths;
  const int q = blockIdx.x % s.nwidths;
  const long long c0 = pair * s.per_pair + s.offc[q];
  double a = 0.0, b = 0.0;
  for (long long j = threadIdx.x; j < s.nwin[q]; j += 256) {
    const double p = (double)window_stat(s, keys, E, c0 + j, nullptr, noise).power;
    a += p; b += p * p;
  }
  sh1[threadIdx.x] = a; sh2[threadIdx.x] = b;
  __syncthreads();
  for (int o = 128; o >= 1; o >>= 1) {
    if (threadIdx.x < o) { sh1[threadIdx.x] += sh1[threadIdx.x + o]; sh2[threadIdx.x] += sh2[threadIdx.x + o]; }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    const double n = (double)s.nwin[q];
    const double mean = n > 0 ? sh1[0] / n : 0.0;
    double var = n > 0 ? sh2[0] / n - mean * mean : 0.0;
    // two-pass refinement is not needed at 1e-4: powers are O(1e2..1e8) and n <= 2^31, double keeps > 9 digits
    if (var < 0) var = 0;
    zst[blockIdx.x] = make_double2(mean, var > 0 ? 1.0 / sqrt(var) : 0.0);
  }
}

constexpr int FIN_THREADS = 256, FIN_TILES = 8;   // 2048 windows per CTA

__global__ void __launch_bounds__(FIN_THREADS) k_finalize(const Sched *sp, const u64 *keys, const float *E,
                                                          float4 *peaks, uint32_t *blockcount,
                                                          const double2 *zst, float zth, const float *noise) {
  __shared__ Sched s;
  __shared__ uint32_t wsum[FIN_THREADS / 32];
  sched_load(s, sp);
  __syncthreads();
  uint32_t mine = 0;
  const long long base = (long long)blockIdx.x * (FIN_THREADS * FIN_TILES);
  // a zero key is a window with power 0 and snr 0 (window_stat): with a non-negative threshold and neither dense peaks nor
  // the z-score asked for it is no candidate and nothing is written - no index arithmetic for it (a candidates-only search
  // leaves most keys zero: the pass is then a scan of the key array)
  const bool skip_zero = !peaks && !zst && s.snr_thresh >= 0.f;
  for (int tile = 0; tile < FIN_TILES; ++tile) {
    const long long c = base + tile * FIN_THREADS + threadIdx.x;
    if (c < s.nwin_total) {
      if (skip_zero && (keys[c] >> 32) == 0ull) continue;
      const WinStat o = window_stat(s, keys, E, c, zst, noise);
      if (peaks) {
        const long long di = s.offd[o.q] + o.pair * s.nwin[o.q] + o.j;
        peaks[di] = make_float4(o.power, o.snr, __int_as_float(o.rate_idx), __int_as_float(o.delay_idx));
      }
      mine += o.snr > (zst ? zth : s.snr_thresh) ? 1u : 0u;
    }
  }
  for (int o = 16; o >= 1; o >>= 1) mine += __shfl_xor_sync(0xffffffffu, mine, o);
  if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = mine;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t t = 0;
    for (int i = 0; i < FIN_THREADS / 32; ++i) t += wsum[i];
    blockcount[blockIdx.x] = t;
  }
}

// single CTA: exclusive scan of blockcount[n] in place, total -> *ncand
__global__ void __launch_bounds__(1024) k_scan(uint32_t *blockcount, long long n, uint32_t *ncand) {
  __shared__ uint32_t part[1024];
  const long long per = (n + 1023) / 1024;
  const long long lo = threadIdx.x * per, hi = lo + per < n ? lo + per : n;
  uint32_t s = 0;
  for (long long i = lo; i < hi; ++i) s += blockcount[i];
  part[threadIdx.x] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t run = 0;
    for (int i = 0; i < 1024; ++i) { const uint32_t v = part[i]; part[i] = run; run += v; }
    *ncand = run;
  }
  __syncthreads();
  uint32_t run = part[threadIdx.x];
  for (long long i = lo; i < hi; ++i) { const uint32_t v = blockcount[i]; blockcount[i] = run; run += v; }
}

struct CandOut { int bl, ifq, wid, win, t0, rate_idx, delay_idx; float power, snr; };

__global__ void __launch_bounds__(FIN_THREADS) k_scatter(const Sched *sp, const u64 *keys, const float *E,
                                                         const uint32_t *blockoff, CandOut *cands,
                                                         uint32_t capacity, const double2 *zst, float zth, const float *noise,
                                                         const uint32_t *total) {
  __shared__ Sched s;
  __shared__ uint32_t wsum[FIN_THREADS / 32];
  __shared__ uint32_t running;
  // a block without candidates (k_finalize counted them; `total` is k_scan's sum) has nothing to write
  if ((blockIdx.x + 1 < gridDim.x ? blockoff[blockIdx.x + 1] : *total) == blockoff[blockIdx.x]) return;
  sched_load(s, sp);
  if (threadIdx.x == 0) running = blockoff[blockIdx.x];
  __syncthreads();
  const bool skip_zero = !zst && s.snr_thresh >= 0.f;
  const long long base = (long long)blockIdx.x * (FIN_THREADS * FIN_TILES);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int tile = 0; tile < FIN_TILES; ++tile) {
    const long long c = base + tile * FIN_THREADS + threadIdx.x;
    WinStat o;
    bool flag = false;
    if (c < s.nwin_total && !(skip_zero && (keys[c] >> 32) == 0ull)) {
      o = window_stat(s, keys, E, c, zst, noise);
      flag = o.snr > (zst ? zth : s.snr_thresh);
    }
    const uint32_t bal = __ballot_sync(0xffffffffu, flag);
    if (lane == 0) wsum[wid] = __popc(bal);
    __syncthreads();
    uint32_t before = running;
    for (int i = 0; i < wid; ++i) before += wsum[i];
    if (flag) {
      const uint32_t pos = before + __popc(bal & ((1u << lane) - 1u));
      if (pos < capacity) {
        CandOut r;
        r.bl = (int)(o.pair / s.nif); r.ifq = s.allif ? -1 : (int)(o.pair % s.nif); r.wid = o.q; r.win = o.j; r.t0 = o.t0;
        r.rate_idx = o.rate_idx; r.delay_idx = o.delay_idx; r.power = o.power; r.snr = o.snr;
        cands[pos] = r;
      }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      uint32_t t = 0;
      for (int i = 0; i < FIN_THREADS / 32; ++i) t += wsum[i];
      running += t;
    }
    __syncthreads();
  }
}

}  // namespace volks
