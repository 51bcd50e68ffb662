// kernels_sfold.cuh - the stride-1 rate transform in the candidates-only mode for the wide widths (Nt >= 64):
// the sliding sum kept in FOLDED form, the transform done only where a candidate is possible.
//
// With the absolute-phase sum of kernels_slide.cuh, A[rho + M s] = sum_{t in window} y[t] W_Nt^{rho t} W_16^{s (t mod 16)}
// (M = Nt / 16), the 16 rate bins of one (rate residue rho, delay column) are the 16-point DFT of the folded sums
//   f[k] = sum_{t in window, t = k mod 16} y[t] W_Nt^{rho t},      A[rho + M s] = sum_{k < 16} W_16^{s k} f[k].
// The window width is a multiple of 16, so sliding the window by one AP removes a sample from and adds a sample to the
// SAME class k = t0 mod 16: ONE complex multiply-add per step,  f[k] += W_Nt^{rho t0} ((-1)^rho y[t0 + w] - y[t0]),
// instead of the sixteen of k_slide.  The bins themselves are needed only where one of them can reach the window's
// pre-threshold (k_winthr: 0.98 of the power a candidate needs), and every bin obeys the triangle inequality
//   |A[rho + M s]| <= sum_k |f[k]| <= sum_k ( max(|x_k|, |y_k|) + (sqrt 2 - 1) min(|x_k|, |y_k|) ) =: e      (f[k] = x_k + i y_k),
// the second step being an upper bound of |z| without a square root (the chord of sqrt(1 + r^2) on [0, 1]; within 8 %).
// For noise e is a sum of 16 near-Rayleigh terms: mean 29.6, deviation 3.8 in units of sqrt(nchan) sigma sqrt(w / 64) x ...;
// at snr_thresh 6 the amplitude pre-threshold (47.5 in the same units) lies 4.7 deviations above the mean at any width
// with a near-Gaussian tail: about 1e-6 per column, 1e-4 of the (window, rho, 64-column tile) triples pass on noise.
// (The Cauchy-Schwarz form 16 sum |f|^2 - a Gamma(16) tail - let 0.7 % pass and was measured at 3.5 % on configs[2].)
//   k_slide<.., FOLD>  (kernels_slide.cuh) the fold is a MODE of the sliding kernel and inherits its operand path (the
//                 cp.async shared-memory ring, twiddle rows at immediate offsets, loads one step ahead): warp = (pair,
//                 segment, rho, 64-column tile), lane = column pair, state f[16] of both columns (packed FP32) and e.
//                 Per step: k_slide's operand g, one packed complex add into f[t0 mod 16], e updated by the change of
//                 that term (summed afresh every 16 steps), and ONE BIT: does e of either column of any lane exceed
//                 the window's amplitude pre-threshold.  No branch, no key: per 16 windows the warp stores a 16-bit hit mask.
//   k_sfold_density   per (pair, segment): more than 1/8 of the segment's hit bits set (interference: a tone raises |Y| in
//                 every delay column) -> `dense`: the ordinary sliding kernel evaluates that segment (it costs 141 warp
//                 instructions per 1024 bins of a window; an evaluation from the samples several times that).
//   k_sfold_compact, k_sfold_eval  the other segments: their non-zero mask words go into a list; a fixed grid of warps
//                 takes one word at a time: the first flagged window of the (rho, tile) is folded from its w samples, the
//                 following ones by sliding; at every flagged window the 16-point transform of a copy, |.|^2, the first
//                 maximum in plane order: exact keys (power, plane index), atomicMax per window.
// A candidate has a bin above the pre-threshold, so its (rho, tile) is flagged and evaluated exactly; a window without a
// flagged tile keeps the zero key (not a candidate - all the candidates-only mode promises, R6).
#pragma once
#include "common.cuh"
#include "kernels_colfft2.cuh"   // FftDifS: split-format 16-point DIF

namespace volks {

#ifndef SFOLD_SEGMUL
#define SFOLD_SEGMUL 4            // segment of k_slide<FOLD> = this many segments of the sliding kernel
#endif

// Dynamic range.  The fold kernel's running sums keep about 2^-23 x 2 x 64 steps of relative rounding of the LARGEST value
// they held; when a row of overwhelming energy leaves the window, that residue stays behind at its absolute size and can
// exceed the 1e-3 margin of the amplitude threshold.  nf * E[t] bounds |Y[t][d]|^2 of every column of row t: where it
// exceeds FOLD_BIG x the power pre-threshold of the window starting there (amplitude ratio 64), k_sfold_guard flags every
// window from that block to the end of the fold segment (evaluated exactly from their samples by k_sfold_eval, which for
// its part re-folds after such a row instead of sliding across it).
#ifndef FOLD_BIG
#define FOLD_BIG 4096.0f
#endif

constexpr int SFOLD_EVAL_WARPS = 148 * 8;   // k_sfold_eval's grid: one-warp CTAs, 8 resident per SM at 248 registers

struct SfoldArgs {
  const float2 *Y;       // [pairs of the chunk][nap][pitch] pair-interleaved delay spectra
  const float4 *tw4;     // [nt] rate twiddles exp(-2 pi i k/nt), pre-broadcast (re, re, im, im)
  const unsigned short *hits;   // [pairs of the chunk][nblk][ndt][M] hit masks of k_slide<FOLD>: bit B = window 16 blk + B
  unsigned short *hits_rw;      // the same array for k_sfold_guard
  unsigned short *big16;        // [pairs of the chunk][nblk]: bit i = row 16 blk + i has overwhelming energy (k_sfold_guard)
  unsigned char *dense;  // [pairs of the chunk][nseg]
  uint32_t *list;        // [0] = number of entries, then the indices of the non-zero mask words of the sparse segments
  const uint32_t *thr;   // pre-thresholds (float bits), chunk-relative: thr[pl * per_pair + offc + t0]
  const float *E;        // per-AP energies of the chunk's pairs: E[pl * nap + t] (FOLD_BIG, kernels_slide.cuh)
  u64 *keys;             // canonical window keys
  long long ntasks;      // k_sfold_eval: warps = pairs * nblk * ndt * M;  k_sfold_density: CTAs = pairs * nseg
  long long per_pair, offc, pair0;
  int nap, nf, w, nt, log2m, nwin, seg, nseg, pitch, nblk;
  int ndt, dt_na, dt_a0, dt_b0;   // the 64-column groups worked on (restricted delay range), as in SlideArgs
};

__global__ void __launch_bounds__(128) k_sfold_density(SfoldArgs a) {
  __shared__ int part[4];
  const long long pl = blockIdx.x / a.nseg;
  const int sg = (int)(blockIdx.x % a.nseg);
  const int wps = (a.ndt << a.log2m);                       // words per block of 16 windows
  const int blk0 = sg * (a.seg >> 4), blk1 = min(a.nblk, blk0 + (a.seg >> 4));
  const unsigned short *h = a.hits + ((size_t)pl * a.nblk + blk0) * wps;
  const int nwords = (blk1 - blk0) * wps;
  int n = 0;
  for (int i = threadIdx.x; i < nwords; i += 128) n += __popc((unsigned)h[i]);
#pragma unroll
  for (int o = 16; o >= 1; o >>= 1) n += __shfl_xor_sync(0xffffffffu, n, o);
  if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = n;
  __syncthreads();
  if (threadIdx.x == 0) a.dense[pl * a.nseg + sg] = (unsigned char)((part[0] + part[1] + part[2] + part[3]) * 8 > nwords * 16 ? 1 : 0);
  if (blockIdx.x == 0 && threadIdx.x == 0) a.list[0] = 0;   // (k_sfold_compact follows on the same stream)
}

// one CTA per (pair, fold segment of `fseg` windows): the first block of 16 windows in which a row of overwhelming energy
// leaves; from there to the end of the segment every mask word becomes "all windows" (rare: most CTAs only read)
__global__ void __launch_bounds__(128) k_sfold_guard(SfoldArgs a, int fseg) {
  __shared__ int firstblk;
  const int nfseg = (a.nwin + fseg - 1) / fseg;
  const long long pl = blockIdx.x / nfseg;
  const int fs = (int)(blockIdx.x % nfseg);
  const int t0 = fs * fseg, t1 = min(a.nwin, t0 + fseg);
  if (threadIdx.x == 0) firstblk = 0x7fffffff;
  __syncthreads();
  const uint32_t *thrp = a.thr + (pl * a.per_pair + a.offc);
  const float *ep = a.E + pl * a.nap;
  int mine = 0x7fffffff;
  for (int tb = t0; tb < t1; tb += 128) {                   // (t0 is a multiple of 16: a warp covers two blocks of 16 rows)
    const int t = tb + (int)threadIdx.x;
    const bool big = t < t1 && (float)a.nf * __ldg(ep + t) > FOLD_BIG * __uint_as_float(__ldg(thrp + t));
    if (big) mine = min(mine, t >> 4);
    const uint32_t m = __ballot_sync(0xffffffffu, big);     // one 16-bit word per block for k_sfold_eval: bit i = row 16 blk + i
    if ((threadIdx.x & 15) == 0 && t < t1) a.big16[(size_t)pl * a.nblk + (t >> 4)] = (unsigned short)((m >> (threadIdx.x & 16)) & 0xFFFFu);
  }
  if (mine != 0x7fffffff) atomicMin(&firstblk, mine);
  __syncthreads();
  const int fb = firstblk;
  if (fb == 0x7fffffff) return;
  const int wps = a.ndt << a.log2m;                         // words per block of 16 windows
  const int b1 = (t1 + 15) >> 4;
  unsigned short *h = a.hits_rw + ((size_t)pl * a.nblk) * wps;
  for (int i = threadIdx.x; i < (b1 - fb) * wps; i += 128) {
    const int blk = fb + i / wps;
    const int nvalid = min(16, a.nwin - blk * 16);
    h[(size_t)blk * wps + i % wps] = (unsigned short)((1u << nvalid) - 1u);
  }
}

// the non-zero mask words of the segments the sliding kernel does not take, as a list (order: whatever the atomics give -
// the evaluation ends in atomicMax over a total order, so the result does not depend on it).  The flagged words cluster
// around the pulses: with one warp per 32 consecutive words the busy warps decided the kernel's length (61 % of the SMs'
// cycles active); from the list every warp takes one word at a time.
__global__ void __launch_bounds__(256) k_sfold_compact(SfoldArgs a) {
  const long long w0 = (long long)blockIdx.x * 256 + threadIdx.x;      // hit word (pair, block, tile, rho)
  bool take = false;
  if (w0 < a.ntasks && a.hits[w0] != 0) {
    const long long q = (w0 >> a.log2m) / a.ndt;                       // pair * nblk + block
    take = !a.dense[(q / a.nblk) * a.nseg + (int)((q % a.nblk) / (a.seg >> 4))];
  }
  const uint32_t m = __ballot_sync(0xffffffffu, take);
  if (m == 0) return;
  const uint32_t lane = threadIdx.x & 31u;
  uint32_t base = 0;
  if (lane == (uint32_t)(__ffs(m) - 1)) base = atomicAdd(a.list, (uint32_t)__popc(m));
  base = __shfl_sync(0xffffffffu, base, __ffs(m) - 1);
  if (take) a.list[1 + base + __popc(m & ((1u << lane) - 1u))] = (uint32_t)w0;
}

// ONE warp per CTA (a CTA's registers are released only when all its warps are done); a fixed grid of warps walks the
// list of k_sfold_compact, one mask word (16 windows of one (pair, rate residue, 64-column tile)) at a time.
__global__ void __launch_bounds__(32) k_sfold_eval(SfoldArgs a) {
  const uint32_t lane = threadIdx.x & 31u;
  const int M = 1 << a.log2m;
  const uint32_t nlist = a.list[0];
  for (uint32_t li = blockIdx.x; li < nlist; li += gridDim.x) {
  long long wt = (long long)a.list[1 + li];
  const uint32_t mask = a.hits[wt];
  const uint32_t bigmask = a.big16[((wt >> a.log2m) / a.ndt)];         // (pair * nblk + block): rows of overwhelming energy
  const uint32_t rho = (uint32_t)(wt & (M - 1)); wt >>= a.log2m;
  const int dti = (int)(wt % a.ndt); wt /= a.ndt;
  const int dt = dti < a.dt_na ? a.dt_a0 + dti : a.dt_b0 + (dti - a.dt_na);
  const uint32_t blk = (uint32_t)(wt % a.nblk);
  const long long pl = wt / a.nblk;
  const uint32_t c = (uint32_t)dt * 32u + lane;                        // column pair (2c, 2c + 1): one 128-bit load per row
  const char *ybase = (const char *)(a.Y + (size_t)pl * a.nap * a.pitch) + (size_t)c * 16u;
  const size_t rowb = (size_t)a.pitch * 8u;
  const char *tw4 = (const char *)a.tw4;
  u64 *keyp = a.keys + ((a.pair0 + pl) * a.per_pair + a.offc);
  const uint32_t ntm = (uint32_t)(a.nt - 1);
  // from the first to the last flagged window of the word: fold the first from its samples (absolute phase: f[k] is the
  // class (t + k) mod 16 of window t), then slide window by window - ONE sum changes per step, kept at index 0 by rotating
  // f; a rotation multiplies every bin of the 16-point transform by a unit phase, so the powers do not notice it
  const int first = __ffs(mask) - 1, last = 31 - __clz(mask);
  const float sg1 = (rho & 1u) ? -1.f : 1.f;
  const f32x2 sgn2 = pk(sg1, sg1);
  f32x2 X[16], Yv[16];
  auto fold_at = [&](uint32_t t0) {                                    // the folded sums of window t0 from its w samples
#pragma unroll
    for (int k = 0; k < 16; ++k) { X[k] = pk(0.f, 0.f); Yv[k] = pk(0.f, 0.f); }
    for (uint32_t tb = 0; tb < (uint32_t)a.w; tb += 16) {
#pragma unroll
      for (int k = 0; k < 16; ++k) {
        f32x2 yx, yy, twx, twy;
        ldg2(ybase + (size_t)(t0 + tb + k) * rowb, yx, yy);
        ldg2(tw4 + (((rho * (t0 + tb + k)) & ntm) << 4), twx, twy);
        X[k] = fma2(yx, twx, fma2(yy, neg2(twy), X[k]));
        Yv[k] = fma2(yx, twy, fma2(yy, twx, Yv[k]));
      }
    }
  };
  // (ONE fold site: the first flagged window, and again at the next flagged window behind a row of overwhelming energy,
  // whose rounding residue would sit in the slid sums)
  bool stale = true;
  for (int b = first;; ++b) {
    const uint32_t t = blk * 16u + (uint32_t)b;
    if ((mask >> b) & 1u) {
      if (stale) { fold_at(t); stale = false; }
      f32x2 GX[16], GY[16];
#pragma unroll
      for (int k = 0; k < 16; ++k) { GX[k] = X[k]; GY[k] = Yv[k]; }
      FftDifS<16, 16, 0, 16>::run(GX, GY);
      u64 key = 0;
#pragma unroll
      for (int s = 0; s < 16; ++s) {                                   // plane order: bins r = rho + M s, then the column
        const int o = brev<16>(s);                                     // output o holds bin s
        const f32x2 pw = fma2(GY[o], GY[o], mul2(GX[o], GX[o]));
        const uint32_t idx = (rho + ((uint32_t)s << a.log2m)) * (uint32_t)a.nf + 2u * c;
        const u64 ka = make_key(lo32(pw), idx), kb = make_key(hi32(pw), idx + 1u);
        key = ka > key ? ka : key;
        key = kb > key ? kb : key;
      }
#pragma unroll
      for (int o = 16; o >= 1; o >>= 1) {
        const u64 other = __shfl_xor_sync(0xffffffffu, key, o);
        key = other > key ? other : key;
      }
      if (lane == 0) atomicMax(keyp + t, key);
    }
    if (b == last) break;
    // window t -> t + 1: sample t leaves, sample t + w enters, both of the class now at index 0
    stale = stale || ((bigmask >> b) & 1u);                            // (warp-uniform)
    if (stale) continue;                                               // nothing worth sliding
    f32x2 xin, yin, xout, yout, twx, twy;
    ldg2(ybase + (size_t)(t + a.w) * rowb, xin, yin);
    ldg2(ybase + (size_t)t * rowb, xout, yout);
    ldg2(tw4 + (((rho * t) & ntm) << 4), twx, twy);
    const f32x2 dx = fma2(xin, sgn2, neg2(xout)), dy = fma2(yin, sgn2, neg2(yout));
    const f32x2 nx = add2(X[0], fma2(dx, twx, mul2(dy, neg2(twy))));
    const f32x2 ny = add2(Yv[0], fma2(dx, twy, mul2(dy, twx)));
#pragma unroll
    for (int k = 0; k < 15; ++k) { X[k] = X[k + 1]; Yv[k] = Yv[k + 1]; }
    X[15] = nx; Yv[15] = ny;
  }
  }
}

}  // namespace volks
