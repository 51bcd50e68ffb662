// kernels_slide.cuh - stride-1 rate transform by a sliding sum (widths with stride == 1, Nt == 2w).
//
//   k_slide<L>   a4+a5+a6 for every window of one width: per (window, delay column) the zero-padded
//                rate DFT, |.|^2 and the per-window argmax, WITHOUT recomputing
//                the transform of each window from scratch.
//
// With the absolute-time phase reference  A_t0[r] = sum_{t0 <= t < t0+w} y[t] W^{r t},  W = e^{-2 pi i/Nt},
// |A_t0[r]|^2 = |F_t0[r]|^2 (F is the window-relative transform of include/volks.h; the two differ by
// the unit factor W^{r t0}), and consecutive windows differ by one sample in and one sample out:
//   A_{t0+1}[r] = A_t0[r] + W^{r t0} ((-1)^r y[t0+w] - y[t0])          (Nt = 2w  =>  W^{r w} = (-1)^r)
// One complex multiply-add per bin per step instead of a 5 log2 Nt flop FFT butterfly chain.  The
// sum is purely additive (no rotating accumulator), so rounding error grows like sqrt(steps); every
// segment of SEG windows restarts from an exactly computed transform (fold + L-point FFT), which
// bounds the growth.
//
// Work split: a warp owns 32 adjacent delay columns (lane = column) and one residue rho of the rate
// index: its thread keeps the L bins r = rho + M s (s < L, M = Nt/L) of its column in registers.
//   W_Nt^{r t} = W_Nt^{rho t} * W_L^{s t}:  the first factor is one warp-uniform table value per
// step, the second depends only on (s, t mod L) and is a compile-time constant once L steps are
// unrolled - most are trivial (+-1, +-i, (+-1 +- i)/sqrt 2).
// Warps never synchronise with each other; the per-window maximum is combined across warps with a
// 64-bit atomicMax on the same total-order key the generic kernel uses.
#pragma once
#include "common.cuh"

namespace volks {

constexpr int SLIDE_WARPS = 8;   // warps per CTA
#ifndef SLIDE_MIN_CTAS
#define SLIDE_MIN_CTAS 2        // register cap 128 (no spills); measured: 2 and 4 within 3 %, 3 slower
#endif

struct SlideArgs {
  const float2 *Y;      // [npairs_chunk][nap][nf] delay spectra
  u64 *keys;            // canonical window keys
  const float2 *twt;    // [nt] exp(-2 pi i k/nt)
  long long ntasks;     // warp tasks = npairs * nseg * (nf/32) * M
  long long per_pair;   // windows per (bl, ifq) pair over all widths
  long long offc;       // canonical offset of this width inside a pair
  long long pair0;      // first pair of the chunk
  int nap, nf, w, nt, log2m, nwin, seg, nseg;
  uint32_t keymask;     // 0xFFFFFFF0, passed as data so that (p & mask) | id is ONE LOP3 (register mask)
};

// acc += exp(-2 pi i K16/16) * g, K16 a compile-time constant.  exp(-i th) g = (c gx + s gy, c gy - s gx).
template <int K16>
__device__ __forceinline__ void cmac_w16(float2 &a, const float2 g) {
  constexpr float C1 = 0.92387953251128674f, S1 = 0.38268343236508977f, H = 0.70710678118654752f;
  constexpr int k = K16 & 15;
  if constexpr (k == 0) { a.x += g.x; a.y += g.y; }
  else if constexpr (k == 8) { a.x -= g.x; a.y -= g.y; }
  else if constexpr (k == 4) { a.x += g.y; a.y -= g.x; }
  else if constexpr (k == 12) { a.x -= g.y; a.y += g.x; }
  else if constexpr ((k & 1) == 0) {
    const float P = H * (g.x + g.y), Q = H * (g.y - g.x);   // shared by every such bin of the step (CSE)
    if constexpr (k == 2) { a.x += P; a.y += Q; }
    else if constexpr (k == 6) { a.x += Q; a.y -= P; }
    else if constexpr (k == 10) { a.x -= P; a.y -= Q; }
    else { a.x -= Q; a.y += P; }   // 14
  } else {
    constexpr float c = (k == 1 || k == 15) ? C1 : (k == 3 || k == 13) ? S1 : (k == 5 || k == 11) ? -S1 : -C1;
    constexpr float s = (k == 1 || k == 7) ? S1 : (k == 3 || k == 5) ? C1 : (k == 9 || k == 15) ? -S1 : -C1;
    a.x = fmaf(c, g.x, fmaf(s, g.y, a.x));
    a.y = fmaf(c, g.y, fmaf(-s, g.x, a.y));
  }
}

// One warp's state while it walks a segment of consecutive windows.
template <int L>
struct SlideState {
  float2 A[L];           // bins r = rho + M s of this lane's column, absolute-phase form
  float2 yin, yout, tw;  // prefetched operands of the NEXT update (loaded one step ahead)
  const char *pout;      // this lane's column of the pair's delay spectra, row 0
  const char *pin;       // the same column, row w
  const char *twt;
  u64 *keyp;             // canonical key of window t0 = keyp[t0]
  uint32_t rowb;         // bytes per Y row
  uint32_t nf, ntmask, rho, log2m, d, keymask;
  float sgn;             // (-1)^rho (used when M is even: every bin of the thread has rho's parity)
};

// Per-thread peak key of the L bins: power with its 4 low mantissa bits replaced by (15 - s), so one
// unsigned max orders by (power descending, s ascending).  Relative power error <= 2^-19.
template <int L>
__device__ __forceinline__ uint32_t slide_local_key(const SlideState<L> &S) {
  uint32_t best = 0;
#pragma unroll
  for (int s = 0; s < L; ++s) {
    const float p = cnorm(S.A[s]);
    const uint32_t k = (__float_as_uint(p) & S.keymask) | (uint32_t)(15 - s);
    best = k > best ? k : best;
  }
  return best;
}

// emit the window's contribution: warp max of the local keys, winner lane(s) update the 64-bit key
template <int L>
__device__ __forceinline__ void slide_emit(const SlideState<L> &S, uint32_t t0) {
  const uint32_t best = slide_local_key<L>(S);
  const uint32_t km = __reduce_max_sync(0xffffffffu, best);
  if (best == km) {
    const uint32_t s = 15u - (km & 15u);
    const uint32_t r = S.rho + (s << S.log2m);
    atomicMax(S.keyp + t0, make_key(__uint_as_float(km & 0xFFFFFFF0u), r * S.nf + S.d));
  }
}

// acc[s] += W_L^{(s B) mod L} * g for every bin s of the thread (s, B compile time).  ge / go: the
// delta of even / odd rate bins (the same value when every bin of the thread has one parity).
template <int L, int B, int S_>
struct SlideBins {
  static __device__ __forceinline__ void run(float2 (&A)[L], const float2 ge, const float2 go) {
    if constexpr (S_ < L) {
      constexpr int K16 = ((S_ * B) % L) * (16 / L);
      cmac_w16<K16>(A[S_], (S_ & 1) ? go : ge);
      SlideBins<L, B, S_ + 1>::run(A, ge, go);
    }
  }
};

// load the operands of the update t -> t+1 (rows t and t+w, warp-uniform twiddle W_Nt^{rho t})
template <int L, bool MODD>
__device__ __forceinline__ void slide_prefetch(SlideState<L> &S, uint32_t t) {
  const uint32_t off = t * S.rowb;
  S.yin = __ldg((const float2 *)(S.pin + off));
  S.yout = __ldg((const float2 *)(S.pout + off));
  if constexpr (!MODD) S.tw = __ldg((const float2 *)(S.twt + (((S.rho * t) & S.ntmask) << 3)));
}

// advance window t0 -> t0+1;  B = t0 mod L (compile time).  Uses the operands prefetched one step
// ago and prefetches those of t0+1 (row t0+1+w <= nap: the Y buffer carries one padding row).
template <int L, int B, bool MODD>
__device__ __forceinline__ void slide_update(SlideState<L> &S, uint32_t t0) {
  const float2 yin = S.yin, yout = S.yout, tw = S.tw;
  slide_prefetch<L, MODD>(S, t0 + 1);
  if constexpr (MODD) {
    // M == 1, rho == 0: the thread holds every rate bin, both parities; W_Nt = W_L
    const float2 ge = make_float2(yin.x - yout.x, yin.y - yout.y);
    const float2 go = make_float2(-yin.x - yout.x, -yin.y - yout.y);
    SlideBins<L, B, 0>::run(S.A, ge, go);
  } else {
    // M even: every bin has rho's parity; g = W_Nt^{rho t0} ((-1)^rho y_in - y_out)
    const float2 dl = make_float2(fmaf(S.sgn, yin.x, -yout.x), fmaf(S.sgn, yin.y, -yout.y));
    const float2 g = cmul(dl, tw);
    SlideBins<L, B, 0>::run(S.A, g, g);
  }
}

// L consecutive steps starting at t0 (t0 mod L == 0).  GUARD: only windows < tend exist.
template <int L, int B, bool MODD, bool GUARD>
struct SlideSteps {
  static __device__ __forceinline__ void run(SlideState<L> &S, uint32_t t0, uint32_t tend) {
    if constexpr (B < L) {
      if (!GUARD || t0 + B < tend) {
        slide_emit<L>(S, t0 + B);
        if (!GUARD || t0 + B + 1 < tend) slide_update<L, B, MODD>(S, t0 + B);
      }
      SlideSteps<L, B + 1, MODD, GUARD>::run(S, t0, tend);
    }
  }
};

// L = min(16, Nt) bins per thread;  MODD <=> M == 1 (Nt <= 16).
template <int L, bool MODD>
__global__ void __launch_bounds__(SLIDE_WARPS * 32, SLIDE_MIN_CTAS) k_slide(SlideArgs a) {
  long long wt = (long long)blockIdx.x * SLIDE_WARPS + (threadIdx.x >> 5);
  if (wt >= a.ntasks) return;                     // whole warps only: no divergence inside a warp
  const uint32_t lane = threadIdx.x & 31u;
  const int M = 1 << a.log2m;
  const int ndt = a.nf >> 5;
  SlideState<L> S;
  S.rho = (uint32_t)(wt & (M - 1)); wt >>= a.log2m;
  const int dt = (int)(wt % ndt); wt /= ndt;
  const int sg = (int)(wt % a.nseg);
  const long long pl = wt / a.nseg;
  S.nf = (uint32_t)a.nf; S.ntmask = (uint32_t)(a.nt - 1); S.log2m = (uint32_t)a.log2m;
  S.d = (uint32_t)(dt * 32) + lane;
  S.sgn = (S.rho & 1u) ? -1.f : 1.f;
  S.keymask = a.keymask;
  S.rowb = (uint32_t)a.nf * 8u;
  S.pout = (const char *)(a.Y + (size_t)pl * a.nap * a.nf + S.d);
  S.pin = S.pout + (size_t)a.w * S.rowb;
  S.twt = (const char *)a.twt;
  S.keyp = a.keys + ((a.pair0 + pl) * a.per_pair + a.offc);
  const uint32_t T0 = (uint32_t)sg * (uint32_t)a.seg;                 // multiple of Nt and of L
  const uint32_t tend = min((uint32_t)a.nwin, T0 + (uint32_t)a.seg);  // windows [T0, tend)
  slide_prefetch<L, MODD>(S, T0);

  // exact start: A[rho + M s] = sum_{t2<L} W_L^{s t2} f[t2],  f[t2] = sum_{t1} y[T0+t2+L t1] W_Nt^{rho (t2+L t1)}
  // (T0 = 0 mod Nt, so absolute and window-relative phases coincide here)
  {
    float2 f[L];
#pragma unroll
    for (int i = 0; i < L; ++i) f[i] = make_float2(0.f, 0.f);
    for (uint32_t tb = 0; tb < (uint32_t)a.w; tb += L) {
#pragma unroll
      for (int t2 = 0; t2 < L; ++t2) {
        const uint32_t t = tb + t2;
        if (t < (uint32_t)a.w) {
          const float2 y = __ldg((const float2 *)(S.pout + (T0 + t) * S.rowb));
          if constexpr (MODD) { f[t2].x += y.x; f[t2].y += y.y; }
          else cmac(f[t2], y, __ldg((const float2 *)(S.twt + (((S.rho * t) & S.ntmask) << 3))));
        }
      }
    }
    FftDif<L, 0, L>::run(f);
#pragma unroll
    for (int s = 0; s < L; ++s) S.A[s] = f[brev<L>(s)];
  }

  uint32_t t0 = T0;
  for (; t0 + L < tend; t0 += L) SlideSteps<L, 0, MODD, false>::run(S, t0, tend);
  SlideSteps<L, 0, MODD, true>::run(S, t0, tend);
}

}  // namespace volks
