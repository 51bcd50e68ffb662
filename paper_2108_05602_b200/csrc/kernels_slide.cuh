// kernels_slide.cuh - stride-1 rate transform by a sliding sum (widths with stride == 1, Nt == 2w).
//
//   k_slide<L, MODD, RING>   a4+a5+a6 for every window of one width: per (window, delay column) the zero-padded
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
// Work split: a warp owns 64 adjacent delay columns (lane = column pair) and one residue rho of the
// rate index: its thread keeps the L bins r = rho + M s (s < L, M = Nt/L) of its two columns in registers.
//   W_Nt^{r t} = W_Nt^{rho t} * W_L^{s t}:  the first factor is one warp-uniform table value per
// step, the second depends only on (s, t mod L) and is a compile-time constant once L steps are
// unrolled - most are trivial (+-1, +-i, (+-1 +- i)/sqrt 2).
// The per-window maximum is combined across the warps of a CTA through shared slots (one barrier per
// 16 windows) and across CTAs with a 64-bit atomicMax on the total-order key the generic kernel uses.
//
// Arithmetic layout (sm_100a packed FP32): a thread works on TWO adjacent delay columns (2c, 2c+1)
// and keeps every quantity as a 64-bit register pair (column a, column b): X[s] = (Re A_a[s], Re A_b[s]),
// Y[s] = (Im ...).  The delay spectra are stored pair-interleaved (common.cuh ld_y), so one 128-bit
// load yields the (re_a, re_b), (im_a, im_b) pairs directly; the warp-uniform twiddle comes from a
// pre-broadcast table (c, c, s, s); the compile-time W_L twiddles are broadcast immediates.  Every
// arithmetic instruction is then an FFMA2 / FADD2 / FMUL2 (fma.rn.f32x2 ...) with no register moves.
// Measured on B200: FFMA2 runs at half the warp-instruction rate of FFMA
// (same flops) but leaves the issue port free for the half-rate ALU-pipe instructions (LOP3 key
// tags), which overlap with it almost perfectly; scalar FFMA + LOP3 do not.
#pragma once
#include "common.cuh"

namespace volks {

constexpr int SLIDE_WARPS = 8;   // warps per CTA (at most)
#ifndef SLIDE_PF
#define SLIDE_PF 8              // L1 prefetch distance in steps (rows)
#endif
#ifndef SLIDE_MIN_CTAS
#define SLIDE_MIN_CTAS 2        // register cap 128
#endif

struct SlideArgs {
  const float2 *Y;      // [npairs_chunk][nap][pitch] delay spectra, pair-interleaved rows
  u64 *keys;            // canonical window keys
  const float2 *twt;    // [nt] exp(-2 pi i k/nt)
  const float4 *tw4;    // [nt] the same, pre-broadcast: (re, re, im, im)
  long long ntasks;     // warp tasks = npairs * nseg * (nf/64) * M
  long long per_pair;   // windows per (bl, ifq) pair over all widths
  long long offc;       // canonical offset of this width inside a pair
  long long pair0;      // first pair of the chunk
  int nap, nf, w, nt, log2m, nwin, seg, nseg, pitch;
  uint32_t keymask;     // 0xFFFFFFF0, passed as data so that (p & mask) | id is ONE LOP3 (register mask)
  // restricted delay range: only the 64-column groups that hold searched bins are worked on.  ndt groups in two
  // pieces: group i < dt_na is column group dt_a0 + i, the others dt_b0 + (i - dt_na) (whole axis: ndt = nf / 64)
  int ndt, dt_na, dt_a0, dt_b0;
  // FOLD mode (kernels_sfold.cuh): pre-thresholds (float bits), chunk-relative thr[pl * per_pair + offc + t0], and
  // the hit masks [pairs of the chunk][nblk][ndt][M] it writes (bit B of a word = window 16 blk + B)
  const uint32_t *thr;
  unsigned short *hits;
  int nblk;
  // pruned widths (kernels_prune.cuh): flags[pl * flag_stride + segment] == 0 means no window of the segment can be
  // a candidate - the CTA returns at once; nullptr = every segment is evaluated
  const unsigned char *flags;
  int flag_stride;
};

// The per-step operand of one parity class, both columns: g = (GX, GY) and the (1 -+ i)/sqrt 2
// products of the even twiddles (dead code in steps that have no such bin).
struct SlideG { f32x2 GX, GY, PP, QQ; };

__device__ __forceinline__ SlideG slide_make_g(f32x2 gx, f32x2 gy) {
  constexpr float H = 0.70710678118654752f;
  SlideG G;
  G.GX = gx; G.GY = gy;
  G.PP = mul2(add2(gx, gy), pk(H, H));   // H (gx + gy)
  G.QQ = mul2(sub2(gy, gx), pk(H, H));   // H (gy - gx)
  return G;
}

// (X, Y) += exp(-2 pi i K16/16) * g, both columns;  exp(-i th) g = (c gx + s gy, c gy - s gx).
template <int K16>
__device__ __forceinline__ void cmac2_w16(f32x2 &X, f32x2 &Y, const SlideG &G) {
  constexpr float C1 = 0.92387953251128674f, S1 = 0.38268343236508977f;
  constexpr int k = K16 & 15;
  if constexpr (k == 0) { X = add2(X, G.GX); Y = add2(Y, G.GY); }
  else if constexpr (k == 8) { X = sub2(X, G.GX); Y = sub2(Y, G.GY); }
  else if constexpr (k == 4) { X = add2(X, G.GY); Y = sub2(Y, G.GX); }
  else if constexpr (k == 12) { X = sub2(X, G.GY); Y = add2(Y, G.GX); }
  else if constexpr (k == 2) { X = add2(X, G.PP); Y = add2(Y, G.QQ); }
  else if constexpr (k == 6) { X = add2(X, G.QQ); Y = sub2(Y, G.PP); }
  else if constexpr (k == 10) { X = sub2(X, G.PP); Y = sub2(Y, G.QQ); }
  else if constexpr (k == 14) { X = sub2(X, G.QQ); Y = add2(Y, G.PP); }
  else {
    constexpr float c = (k == 1 || k == 15) ? C1 : (k == 3 || k == 13) ? S1 : (k == 5 || k == 11) ? -S1 : -C1;
    constexpr float s = (k == 1 || k == 7) ? S1 : (k == 3 || k == 5) ? C1 : (k == 9 || k == 15) ? -S1 : -C1;
    X = fma2(G.GX, pk(c, c), fma2(G.GY, pk(s, s), X));
    Y = fma2(G.GY, pk(c, c), fma2(G.GX, pk(-s, -s), Y));
  }
}

// FOLD mode: an upper bound of |z| for both columns of a packed complex value without a square root:
//   |z| <= max(|x|, |y|) + (sqrt 2 - 1) min(|x|, |y|)   (the chord of the convex sqrt(1 + r^2) on r in [0, 1]; within 8 %)
__device__ __forceinline__ f32x2 fold_oct(f32x2 X, f32x2 Y) {
  const float xa = fabsf(lo32(X)), ya = fabsf(lo32(Y)), xb = fabsf(hi32(X)), yb = fabsf(hi32(Y));
  return pk(fmaf(0.41421357f, fminf(xa, ya), fmaxf(xa, ya)), fmaf(0.41421357f, fminf(xb, yb), fmaxf(xb, yb)));
}

// One warp's state while it walks a segment of consecutive windows.
template <int L>
struct SlideState {
  f32x2 X[L], Y[L];             // bins r = rho + M s of columns (a, b), absolute-phase form
  f32x2 xin, yin, xout, yout;   // prefetched operands of the NEXT update (loaded one step ahead)
  f32x2 twx, twy;               // ... and its warp-uniform twiddle, pre-broadcast
  f32x2 sgn2;                   // ((-1)^rho, (-1)^rho)  (M even: every bin of the thread has rho's parity)
  const char *pout;             // this lane's column pair, row 0 of the pair's delay spectra
  const char *pin;              // the same columns, row w
  const char *tw4;
  u64 *keyp;                    // canonical key of window t0 = keyp[t0]
  uint32_t rowb;                // bytes per Y row
  uint32_t ntmask, rho, idx0, idxs, keymask, lane;   // plane index of bin s, column a: idx0 + s * idxs
  uint32_t tilekey;             // 0xFFFFFFFF - (2^31 | idx0), slide_emit_u
  // RING variant: shared-memory addresses of this lane's entry in the ring rows of the current block's
  // first leaving row (sm_out) and first entering row (sm_in); ring geometry in bytes
  uint32_t sm_out, sm_in, ring_lo, ring_hi, rrowb;
  uint32_t twp, tw_lo, tw_hi;   // RING: this warp's twiddle row W_Nt^{rho t}, t = 0..Nt (shared memory), entry of the current block
  // FOLD mode: X / Y hold the folded sums f[k] (k = t mod 16) instead of the bins; e = sum_k fold_oct(f[k]) >= sum_k |f[k]|
  // of both columns; the AMPLITUDE pre-thresholds of the block's 16 windows (lowered by 1e-3 for the rounding of e) sit in
  // shared memory - every warp of the CTA works on the same windows
  f32x2 e;
  uint32_t mask;                // this LANE's hit bits (OR-reduced over the warp at the end of the block)
  uint32_t thrs;                // shared address of the current block's 16 amplitude thresholds (CTA-wide: one segment)
};

// emit the window's contribution: per column the max of (power with its 4 low mantissa bits replaced
// by 15 - s): one unsigned max orders by (power descending, s ascending), relative power error
// <= 2^-19 (R1).  Then the better column (ties: the lower one), the warp max, and the
// winning lane (lowest among equal keys) parks the 64-bit key in the CTA's slot [step][warp].
template <int L>
__device__ __forceinline__ void slide_emit(const SlideState<L> &S, u64 *slot) {
  uint32_t ba = 0, bb = 0;
#pragma unroll
  for (int s = 0; s < L; ++s) {
    const f32x2 pw = fma2(S.Y[s], S.Y[s], mul2(S.X[s], S.X[s]));
    ba = max(ba, (__float_as_uint(lo32(pw)) & S.keymask) | (uint32_t)(15 - s));
    bb = max(bb, (__float_as_uint(hi32(pw)) & S.keymask) | (uint32_t)(15 - s));
  }
  const bool colb = bb > ba;
  const uint32_t best = colb ? bb : ba;
  const uint32_t km = __reduce_max_sync(0xffffffffu, best);
  const uint32_t tied = __ballot_sync(0xffffffffu, best == km);
  if (S.lane == (uint32_t)__ffs(tied) - 1u) {
    const uint32_t s = 15u - (km & 15u);
    *slot = make_key(__uint_as_float(km & 0xFFFFFFF0u), S.idx0 + s * S.idxs + (colb ? 1u : 0u));
  }
}

// Untagged emit (the kernels with M >= 2, i.e. w >= 16): the maximum power and the delay COLUMN it sits in - one
// 3-input max per bin instead of two LOP3 + the max.  The slot carries (exact power bits, 2^31 | plane index of the
// column's first bin rho * nf + d): which of the column's 16 rate bins r = rho + M s holds the maximum is found
// afterwards, for the windows that need it, by k_recover (an exact re-evaluation of that one column: 16 bins from
// w samples); DESIGN.md section 6.  Ties between columns: the lower one.
template <int L>
__device__ __forceinline__ void slide_emit_u(const SlideState<L> &S, u64 *slot) {
  uint32_t ba = 0, bb = 0;
#pragma unroll
  for (int s = 0; s < L; ++s) {
    const f32x2 pw = fma2(S.Y[s], S.Y[s], mul2(S.X[s], S.X[s]));
    ba = max(ba, __float_as_uint(lo32(pw)));
    bb = max(bb, __float_as_uint(hi32(pw)));
  }
  const uint32_t best = max(ba, bb);
  const uint32_t km = __reduce_max_sync(0xffffffffu, best);
  const uint32_t tied = __ballot_sync(0xffffffffu, best == km);
  if (S.lane == (uint32_t)__ffs(tied) - 1u)
    *slot = ((u64)km << 32) | (u64)(S.tilekey - (bb > ba ? 1u : 0u));
}

// after a block of nsteps (<= 16) windows starting at t0: threads 0..nsteps-1 reduce the warps'
// slots of their window and update the canonical key.  Slots are double-buffered, so one
// __syncthreads per block orders both the reads here and the next writes.
__device__ __forceinline__ void slide_flush(u64 *keyp, const u64 *slots, uint32_t t0, uint32_t nsteps, int nwarps) {
  __syncthreads();
  if (threadIdx.x < nsteps) {
    const u64 *p = slots + threadIdx.x * SLIDE_WARPS;
    u64 k = p[0];
    for (int i = 1; i < nwarps; ++i) k = p[i] > k ? p[i] : k;
    atomicMax(keyp + t0 + threadIdx.x, k);
  }
}

// bins s = S_ .. L-1:  (X[s], Y[s]) += W_L^{(s B) mod L} * g.   Ge / Go: operand of the even / odd
// rate bins (identical when every bin of the thread has one parity).
template <int L, int B, int S_>
struct SlideBins {
  static __device__ __forceinline__ void run(SlideState<L> &S, const SlideG &Ge, const SlideG &Go) {
    if constexpr (S_ < L) {
      constexpr int K16 = ((S_ * B) % L) * (16 / L);
      cmac2_w16<K16>(S.X[S_], S.Y[S_], (S_ & 1) ? Go : Ge);
      SlideBins<L, B, S_ + 1>::run(S, Ge, Go);
    }
  }
};

// 128-bit shared-memory load as two register pairs
__device__ __forceinline__ void lds2(uint32_t addr, f32x2 &a, f32x2 &b) {
  asm volatile("ld.shared.v2.b64 {%0,%1}, [%2];" : "=l"(a), "=l"(b) : "r"(addr));
}

// load the operands of the update t -> t+1 (rows t and t+w of both columns, warp-uniform twiddle).
// BN = t - (first window of the current 16-step block), 0..16 (compile time; RING only).
// RR: bytes per ring row when known at compile time (0: S.rrowb) - the row offsets become immediates
template <int L, bool MODD, bool RING, int BN, int RR>
__device__ __forceinline__ void slide_prefetch(SlideState<L> &S, uint32_t t) {
  if constexpr (RING) {
    const uint32_t rrowb = RR ? (uint32_t)RR : S.rrowb;
    uint32_t ao = S.sm_out + BN * rrowb, ai = S.sm_in + BN * rrowb;
    if constexpr (BN == 16) {   // first row of the next block: the ring may wrap here (and only here)
      ao = ao >= S.ring_hi ? ao - (S.ring_hi - S.ring_lo) : ao;
      ai = ai >= S.ring_hi ? ai - (S.ring_hi - S.ring_lo) : ai;
    }
    lds2(ai, S.xin, S.yin);
    lds2(ao, S.xout, S.yout);
  } else {
    const uint32_t off = t * S.rowb;
    // row t+w is new to this SM: pull the row SLIDE_PF steps ahead into L1 now, so that the register
    // load one step ahead is an L1 hit (the Y buffer carries SLIDE_PF + 2 padding rows)
    asm volatile("prefetch.global.L1 [%0];" ::"l"(S.pin + off + SLIDE_PF * S.rowb));
    ldg2(S.pin + off, S.xin, S.yin);
    ldg2(S.pout + off, S.xout, S.yout);
  }
  if constexpr (RING) lds2(S.twp + BN * 16u, S.twx, S.twy);   // the warp's own row: consecutive entries, no index arithmetic
  else if constexpr (!MODD) ldg2(S.tw4 + (((S.rho * t) & S.ntmask) << 4), S.twx, S.twy);
}

// advance window t0 -> t0+1;  B = t0 mod L (compile time).  Uses the operands prefetched one step
// ago and prefetches those of t0+1.
template <int L, int B, bool MODD, bool RING, int RR, bool FOLD = false>
__device__ __forceinline__ void slide_update(SlideState<L> &S, uint32_t t0) {
  const f32x2 xin = S.xin, yin = S.yin, xout = S.xout, yout = S.yout, twx = S.twx, twy = S.twy;
  slide_prefetch<L, MODD, RING, B + 1, RR>(S, t0 + 1);
  if constexpr (MODD) {
    // M == 1, rho == 0: the thread holds every rate bin, both parities; W_Nt = W_L
    const SlideG Ge = slide_make_g(sub2(xin, xout), sub2(yin, yout));
    const SlideG Go = slide_make_g(sub2(neg2(xin), xout), sub2(neg2(yin), yout));
    SlideBins<L, B, 0>::run(S, Ge, Go);
  } else {
    // M even: every bin has rho's parity; g = W_Nt^{rho t0} ((-1)^rho y_in - y_out)
    const f32x2 dx = fma2(xin, S.sgn2, neg2(xout)), dy = fma2(yin, S.sgn2, neg2(yout));
    const f32x2 gx = fma2(dx, twx, mul2(dy, neg2(twy)));
    const f32x2 gy = fma2(dx, twy, mul2(dy, twx));
    if constexpr (FOLD) {
      // the leaving and the entering sample share the class B = t0 mod 16 (w is a multiple of 16): ONE sum changes
      const f32x2 eo = fold_oct(S.X[B], S.Y[B]);
      S.X[B] = add2(S.X[B], gx); S.Y[B] = add2(S.Y[B], gy);
      S.e = add2(sub2(S.e, eo), fold_oct(S.X[B], S.Y[B]));
    } else {
      const SlideG G = slide_make_g(gx, gy);
      SlideBins<L, B, 0>::run(S, G, G);
    }
  }
}

// L consecutive steps starting at t0 (t0 mod L == 0).  GUARD: only windows < tend exist.
template <int L, int B, bool MODD, bool GUARD, bool RING, int RR, bool FOLD = false>
struct SlideSteps {
  static __device__ __forceinline__ void run(SlideState<L> &S, uint32_t t0, uint32_t tend, u64 *slot) {
    if constexpr (B < L) {
      if (!GUARD || t0 + B < tend) {
        if constexpr (FOLD) {
          // every bin of (rho, column) obeys |A| <= sum_k |f[k]| <= e (kernels_sfold.cuh): one bit per window and lane, no branch
          float thrB;                               // a broadcast shared-memory load: no warp collective in the steps
          asm volatile("ld.shared.f32 %0, [%1];" : "=f"(thrB) : "r"(S.thrs + 4u * B));
          if (fmaxf(lo32(S.e), hi32(S.e)) > thrB) S.mask |= 1u << B;
        }
        // M == 1 (w <= 8): tagged keys, exact index at once; M >= 2: power + tile id, index by k_recover
        else if constexpr (MODD) slide_emit<L>(S, slot + B * SLIDE_WARPS);
        else slide_emit_u<L>(S, slot + B * SLIDE_WARPS);
        if (!GUARD || t0 + B + 1 < tend) slide_update<L, B, MODD, RING, RR, FOLD>(S, t0 + B);
      }
      SlideSteps<L, B + 1, MODD, GUARD, RING, RR, FOLD>::run(S, t0, tend, slot);
    }
  }
};

// exact transform of window T0 for ONE column (col = 0/1 of the pair):
//   A[rho + M s] = sum_{t2<L} W_L^{s t2} f[t2],  f[t2] = sum_{t1} y[T0+t2+L t1] W_Nt^{rho (t2+L t1)}
// (T0 = 0 mod Nt, so absolute and window-relative phases coincide).  Result in natural s order.
template <int L, bool MODD, bool FOLD = false>
__device__ __forceinline__ void slide_start_column(float2 (&A)[L], const char *pout, uint32_t rowb, uint32_t T0,
                                                   uint32_t w, const float2 *twt, uint32_t rho, uint32_t ntmask, int col) {
  float2 f[L];
#pragma unroll
  for (int i = 0; i < L; ++i) f[i] = make_float2(0.f, 0.f);
  for (uint32_t tb = 0; tb < w; tb += L) {
#pragma unroll
    for (int t2 = 0; t2 < L; ++t2) {
      const uint32_t t = tb + t2;
      if (t < w) {
        const float *p = (const float *)(pout + (T0 + t) * rowb) + col;
        const float2 y = make_float2(__ldg(p), __ldg(p + 2));
        if constexpr (MODD) { f[t2].x += y.x; f[t2].y += y.y; }
        else cmac(f[t2], y, __ldg(twt + ((rho * t) & ntmask)));
      }
    }
  }
  if constexpr (FOLD) {      // the folded sums themselves (class t2 = t mod L)
#pragma unroll
    for (int s = 0; s < L; ++s) A[s] = f[s];
    return;
  }
  FftDif<L, 0, L>::run(f);
#pragma unroll
  for (int s = 0; s < L; ++s) A[s] = f[brev<L>(s)];
}

// RING variant: the CTA's rows of delay spectra travel through a shared-memory ring of R = w + 48 rows
// (its 64 * DT columns), filled 16 rows per block with cp.async one block ahead.  rel = row index
// relative to the segment start T0; ring slot = rel mod R; R is a multiple of 16 and block starts are
// multiples of 16, so the 16 rows of a block never wrap.
struct SlideRing {
  uint32_t base;      // shared address of the ring
  uint32_t rrowb;     // bytes per ring row = 512 * DT
  uint32_t R;         // rows
  const char *gsrc;   // global address of (pair row 0, first column of the CTA)
  uint32_t rowb;      // bytes per Y row
  uint32_t T0, nap;
};

// all threads of the CTA: copy rows rel in [r0, r0 + n) into the ring (source row clamped to the padding row)
__device__ __forceinline__ void slide_ring_fill(const SlideRing &G, uint32_t r0, uint32_t n) {
  const uint32_t cpr = G.rrowb >> 4;                       // 16-byte chunks per ring row
  for (uint32_t i = threadIdx.x; i < n * cpr; i += blockDim.x) {
    const uint32_t r = i / cpr, c = i - r * cpr, rel = r0 + r;
    const uint32_t grow = min(G.T0 + rel, G.nap);
    const uint32_t dst = G.base + (rel % G.R) * G.rrowb + (c << 4);
    const char *src = G.gsrc + (size_t)grow * G.rowb + (c << 4);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src));
  }
}

// the same for the 16 new rows of a block, rel in [r0, r0 + 16), whose first row sits in ring slot `slot` (kept by the
// caller: no modulo); RR = bytes per ring row at compile time (a power of two: shifts for the row / chunk split), or 0
template <int RR>
__device__ __forceinline__ void slide_ring_fill_block(const SlideRing &G, uint32_t r0, uint32_t slot) {
  const uint32_t cpr = RR ? (uint32_t)RR >> 4 : G.rrowb >> 4;
  for (uint32_t i = threadIdx.x; i < 16u * cpr; i += blockDim.x) {
    const uint32_t r = i / cpr, c = i - r * cpr;
    uint32_t sl = slot + r;
    sl = sl >= G.R ? sl - G.R : sl;
    const uint32_t grow = min(G.T0 + r0 + r, G.nap);
    const uint32_t dst = G.base + sl * (RR ? (uint32_t)RR : G.rrowb) + (c << 4);
    const char *src = G.gsrc + (size_t)grow * G.rowb + (c << 4);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src));
  }
}

// L = min(16, Nt) bins per thread;  MODD <=> M == 1 (Nt <= 16);  RING (M >= 4 only): rows through shared memory.
// FOLD (M >= 4, candidates-only mode): the folded-sum form of kernels_sfold.cuh - no bins, no keys, one hit bit per window
template <int L, bool MODD, bool RING, int RR = 0, bool FOLD = false>
__global__ void __launch_bounds__(SLIDE_WARPS * 32, SLIDE_MIN_CTAS) k_slide(SlideArgs a) {
  // blockDim.x = 32 * min(SLIDE_WARPS, ndt * M): every warp of a CTA works on the same (pair, segment)
  __shared__ u64 slots[2][16 * SLIDE_WARPS];
  [[maybe_unused]] __shared__ float fthr[2][16];   // FOLD: amplitude pre-thresholds of the current / the next block
  extern __shared__ float4 slide_ring[];
  const int nwarps = blockDim.x >> 5, warp = threadIdx.x >> 5;
  long long wt = (long long)blockIdx.x * nwarps + warp;
  const uint32_t lane = threadIdx.x & 31u;
  const int M = 1 << a.log2m;
  const int ndt = a.ndt;                          // 64 columns per warp; the groups with searched delay bins
  SlideState<L> S;
  S.lane = lane;
  S.rho = (uint32_t)(wt & (M - 1)); wt >>= a.log2m;
  const int dti = (int)(wt % ndt); wt /= ndt;
  const int dt = dti < a.dt_na ? a.dt_a0 + dti : a.dt_b0 + (dti - a.dt_na);
  const int sg = (int)(wt % a.nseg);
  const long long pl = wt / a.nseg;
  if (a.flags && !a.flags[pl * a.flag_stride + sg]) return;   // the whole CTA shares (pair, segment)
  const uint32_t c = (uint32_t)(dt * 32) + lane;  // column pair (2c, 2c+1)
  S.ntmask = (uint32_t)(a.nt - 1);
  S.idx0 = S.rho * (uint32_t)a.nf + 2u * c;       // plane index r * nf + d of bin s: r = rho + M s
  S.idxs = (uint32_t)a.nf << a.log2m;
  S.tilekey = 0xFFFFFFFFu - (0x80000000u | S.idx0);   // bit 31: a column (its bin s = 0), not yet a bin
  const float sg1 = (S.rho & 1u) ? -1.f : 1.f;
  S.sgn2 = pk(sg1, sg1);
  S.keymask = a.keymask;
  S.rowb = (uint32_t)a.pitch * 8u;
  S.pout = (const char *)(a.Y + (size_t)pl * a.nap * a.pitch) + (size_t)c * 16u;
  S.pin = S.pout + (size_t)a.w * S.rowb;
  S.tw4 = (const char *)a.tw4;
  S.keyp = a.keys + ((a.pair0 + pl) * a.per_pair + a.offc);
  const uint32_t T0 = (uint32_t)sg * (uint32_t)a.seg;                 // multiple of Nt and of L
  const uint32_t tend = min((uint32_t)a.nwin, T0 + (uint32_t)a.seg);  // windows [T0, tend)
  [[maybe_unused]] const uint32_t *thrp = nullptr;
  [[maybe_unused]] unsigned short *hp = nullptr;
  [[maybe_unused]] uint32_t thr_next = 0x7f000000u;   // float bits: 1.7e38
  if constexpr (FOLD) {
    thrp = a.thr + (pl * a.per_pair + a.offc);
    hp = a.hits + (((size_t)pl * a.nblk) * ndt + dti) * M + S.rho;      // + blk * ndt * M
    if (threadIdx.x < 16) {   // threads 0..15 keep the thresholds two blocks ahead: raw in a register, converted a block later
      fthr[0][threadIdx.x] = T0 + threadIdx.x < tend ? 0.999f * sqrtf(__uint_as_float(__ldg(thrp + T0 + threadIdx.x))) : 3.0e38f;
      thr_next = T0 + 16u + threadIdx.x < tend ? __ldg(thrp + T0 + 16u + threadIdx.x) : 0x7f000000u;
    }
  }
  SlideRing G;
  if constexpr (RING) {
    // the CTA's warps are (rho fastest, then dt): its first warp's dt is the first column group
    const long long wt0 = ((long long)blockIdx.x * nwarps) >> a.log2m;
    const int dti0 = (int)(wt0 % ndt);              // (the pieces are multiples of the CTA's groups: contiguous columns)
    const int dt0 = dti0 < a.dt_na ? a.dt_a0 + dti0 : a.dt_b0 + (dti0 - a.dt_na);
    const int dtc = nwarps >> a.log2m > 0 ? nwarps >> a.log2m : 1;    // column groups per CTA
    G.base = (uint32_t)__cvta_generic_to_shared(slide_ring);
    G.rrowb = 512u * (uint32_t)dtc;
    G.R = (uint32_t)a.w + 48u;
    G.rowb = S.rowb;
    G.gsrc = (const char *)(a.Y + (size_t)pl * a.nap * a.pitch) + (size_t)dt0 * 512u;
    G.T0 = T0; G.nap = (uint32_t)a.nap;
    S.rrowb = G.rrowb;
    S.ring_lo = G.base + (uint32_t)(dt - dt0) * 512u + lane * 16u;    // this lane's entry of ring row 0
    S.ring_hi = S.ring_lo + G.R * G.rrowb;
    S.sm_out = S.ring_lo;                                             // rel 0
    S.sm_in = S.ring_lo + (uint32_t)a.w * G.rrowb;                    // rel w
    // twiddle rows behind the ring: [warp][Nt + 1] float4, entry t = W_Nt^{rho t} pre-broadcast (entry Nt = entry 0)
    S.tw_lo = G.base + G.R * G.rrowb + (uint32_t)warp * (uint32_t)(a.nt + 1) * 16u;
    S.tw_hi = S.tw_lo + (uint32_t)a.nt * 16u;
    S.twp = S.tw_lo;                                                  // T0 = 0 mod Nt
    for (uint32_t i = lane; i <= (uint32_t)a.nt; i += 32u) {
      const float4 v = __ldg(a.tw4 + ((S.rho * i) & S.ntmask));
      asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(S.tw_lo + i * 16u), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
    }
    slide_ring_fill(G, 0u, (uint32_t)a.w + 17u);                      // rows of block 0 (and the start window)
    asm volatile("cp.async.wait_all;" ::: "memory");
    __syncthreads();
  }
  if constexpr (FOLD && !RING) __syncthreads();                         // fthr[0]
  slide_prefetch<L, MODD, RING, 0, RR>(S, T0);
  if constexpr (FOLD && RING) {
    // the first window's samples are rows 0 .. w - 1 of the ring, their twiddles W_Nt^{rho t} entries 0 .. w - 1 of the
    // warp's row (T0 = 0 mod Nt): both columns at once, packed
#pragma unroll
    for (int k = 0; k < L; ++k) { S.X[k] = pk(0.f, 0.f); S.Y[k] = pk(0.f, 0.f); }
    for (uint32_t tb = 0; tb < (uint32_t)a.w; tb += L) {
#pragma unroll
      for (int k = 0; k < L; ++k) {
        f32x2 yx, yy, twx, twy;
        lds2(S.ring_lo + (tb + k) * S.rrowb, yx, yy);
        lds2(S.tw_lo + (tb + k) * 16u, twx, twy);
        S.X[k] = fma2(yx, twx, fma2(yy, neg2(twy), S.X[k]));
        S.Y[k] = fma2(yx, twy, fma2(yy, twx, S.Y[k]));
      }
    }
  } else {
    float2 Aa[L], Ab[L];
    slide_start_column<L, MODD, FOLD>(Aa, S.pout, S.rowb, T0, (uint32_t)a.w, a.twt, S.rho, S.ntmask, 0);
    slide_start_column<L, MODD, FOLD>(Ab, S.pout, S.rowb, T0, (uint32_t)a.w, a.twt, S.rho, S.ntmask, 1);
#pragma unroll
    for (int s = 0; s < L; ++s) { S.X[s] = pk(Aa[s].x, Ab[s].x); S.Y[s] = pk(Aa[s].y, Ab[s].y); }
  }

  [[maybe_unused]] uint32_t fslot = (uint32_t)a.w + 17u;   // RING: slot of the next row to fill (R = w + 48 > w + 17)
  uint32_t t0 = T0, buf = 0;
  for (;; t0 += L, buf ^= 1u) {
    const bool full = t0 + L < tend;
    if constexpr (RING) {                        // the next block's new rows
      slide_ring_fill_block<RR>(G, t0 - T0 + (uint32_t)a.w + 17u, fslot);
      fslot += 16u; fslot = fslot >= G.R ? fslot - G.R : fslot;
    }
    if constexpr (FOLD) {
      if (full && threadIdx.x < 16) {            // the next block's thresholds; visible after this block's barrier
        fthr[buf ^ 1u][threadIdx.x] = 0.999f * sqrtf(__uint_as_float(thr_next));
        thr_next = t0 + 32u + threadIdx.x < tend ? __ldg(thrp + t0 + 32u + threadIdx.x) : 0x7f000000u;
      }
      S.thrs = (uint32_t)__cvta_generic_to_shared(&fthr[buf][0]);
      if ((((t0 - T0) >> 4) & 3u) == 0u) {       // summed afresh every 64 steps (the updates in between drift by ~1e-5)
        S.e = pk(0.f, 0.f);
#pragma unroll
        for (int k = 0; k < L; ++k) S.e = add2(S.e, fold_oct(S.X[k], S.Y[k]));
      }
      S.mask = 0;
    }
    if (full) SlideSteps<L, 0, MODD, false, RING, RR, FOLD>::run(S, t0, tend, &slots[buf][warp]);
    else SlideSteps<L, 0, MODD, true, RING, RR, FOLD>::run(S, t0, tend, &slots[buf][warp]);
    if constexpr (RING) asm volatile("cp.async.wait_all;" ::: "memory");
    if constexpr (FOLD) {
      const uint32_t hit = __reduce_or_sync(0xffffffffu, S.mask);
      if (lane == 0) hp[(size_t)(t0 >> 4) * (size_t)(ndt * M)] = (unsigned short)hit;
      __syncthreads();                           // the next block's thresholds (and ring rows) are complete and visible
    } else {
      slide_flush(S.keyp, slots[buf], t0, full ? (uint32_t)L : tend - t0, nwarps);
    }
    if (!full) break;
    if constexpr (RING) {   // advance the block base by 16 rows (wraps only at a block boundary)
      S.sm_out += 16u * S.rrowb; S.sm_out = S.sm_out >= S.ring_hi ? S.sm_out - (S.ring_hi - S.ring_lo) : S.sm_out;
      S.sm_in += 16u * S.rrowb;  S.sm_in = S.sm_in >= S.ring_hi ? S.sm_in - (S.ring_hi - S.ring_lo) : S.sm_in;
      S.twp += 16u * 16u;        S.twp = S.twp >= S.tw_hi ? S.twp - (S.tw_hi - S.tw_lo) : S.twp;
    }
  }
}

// Pre-thresholds of the candidates-only mode: one thread per (pair of the chunk, sliding width, window):
//   thr = SLIDE_PRE * snr_thresh^2 * sum_{t<w} E[t0 + t]   (the window energy = the noise of a7, summed in the
// order k_finalize uses), stored as float bits.  A window is a candidate iff P1 > snr_thresh^2 * energy, so every
// candidate lies above thr: k_recover finds the index of exactly those windows, k_bound keeps their segments.
#ifndef SLIDE_PRE
#define SLIDE_PRE 0.98f
#endif
struct WinThrArgs {
  const float *E;        // [npair][nap] per-AP energies
  uint32_t *thr;         // [pairs of the chunk][per_pair]
  long long per_pair, pair0, total;   // total = pairs of the chunk * windows of the sliding widths per pair
  float thr2;            // snr_thresh^2
  int nap, nq;
  int w[16], stride[16], nwin[16];
  long long offc[16], cum[17];        // cum: prefix sums of nwin over the listed widths
};

__global__ void __launch_bounds__(256) k_winthr(WinThrArgs a) {
  const long long gid = (long long)blockIdx.x * 256 + threadIdx.x;
  if (gid >= a.total) return;
  const long long per = a.cum[a.nq];
  const long long pl = gid / per;
  long long r = gid - pl * per;
  int i = 0;
  while (r >= a.cum[i + 1]) ++i;
  const int j = (int)(r - a.cum[i]);
  const float *e = a.E + (a.pair0 + pl) * a.nap + (long long)j * a.stride[i];   // t0 = j * stride
  float es = 0.f;
  for (int t = 0; t < a.w[i]; ++t) es += e[t];
  a.thr[pl * a.per_pair + a.offc[i] + j] = __float_as_uint(SLIDE_PRE * a.thr2 * es);
}

}  // namespace volks
