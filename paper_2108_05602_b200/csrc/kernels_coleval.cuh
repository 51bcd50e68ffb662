// kernels_coleval.cuh - column-level pruning of one stride-1 width (candidates of a width whose amplitude-sum bound
// (kernels_prune.cuh) is too weak to rule out whole segments, but rules out most (window, delay column) pairs).
//
// For noise the bound of a w = 32 window exceeds the pre-threshold in about 2 % of the delay columns (snr_thresh 6):
// every segment has such columns, so k_bound's segment flags prune nothing - but a candidate can only sit in one of
// them.  k_bound writes one bit per (window, column); here every set bit is evaluated by the definition:
//   k_coleval   CTA = (pair, 128 consecutive windows).  The tile's bits are compacted into a shared-memory list (128
//               columns at a time, a fixed order); every thread takes entries in turn: it loads the window's w <= 32
//               samples of the column ONCE into registers and, for every rate residue rho < M, folds them with
//               W_Nt^{rho t} into 16 sums and runs the 16-point transform - all Nt rate bins of the column, exactly
//               (the code of k_recover, for every residue) - keeping the first maximum in plane order.  A residue
//               whose folded sums cannot reach the window's pre-threshold (sum_k |f[k]| bounds its 16 bins) skips the
//               transform: nearly all of them, the amplitude-sum bound of k_bound being much the weaker one.  The window's
//               key becomes the maximum over its entries (a shared-memory atomicMax per tile) and REPLACES what the
//               window held, if it exceeds the window's pre-threshold.
// A candidate has P1 > snr_thresh^2 noise > pre-threshold and P1 <= bound^2 of its column, so its column is listed and
// the key is the exact P1 with its exact first argmax (the unlisted columns lie below the pre-threshold).  A window
// whose listed maximum stays below the pre-threshold is no candidate and keeps the key it had (its true peak may sit
// in an unlisted column).  Tiles in which more than 1/8 of the bits are set (an interference-ridden baseline) are left
// to the sliding kernel, which costs about a seventh per (window, column) - k_bound marks them `dense`.  In the
// candidates-only mode the sliding kernel of this width runs on the dense tiles only; when every window is indexed it
// runs everywhere as before and this kernel then replaces the keys of the possible candidates of the other tiles, so
// that both index modes report identical candidates.
#pragma once
#include "common.cuh"

namespace volks {

constexpr int CE_TILE = 128;       // windows per CTA
constexpr int CE_CHUNK = 128;      // columns compacted at a time
constexpr int CE_THREADS = 256;
constexpr int CE_WMAX = 32;        // samples held in registers

struct ColEvalArgs {
  const float2 *Y;        // [pairs of the chunk][nap][pitch] pair-interleaved delay spectra
  u64 *keys;
  const uint32_t *mask;   // k_bound's bits: mask[(pl * nwords + window / 32) * nf + column]
  const uint32_t *thr;    // pre-thresholds (float bits), chunk-relative: thr[pl * per_pair + offc + t0]
  const unsigned char *dense;   // k_bound: dense[pl * dstride + tile] = 1: the sliding kernel evaluates this tile, not this kernel
  const unsigned char *empty;   // ... empty[pl * dstride + tile] = 1: no bit of the tile is set (nothing to list: most tiles)
  const float2 *twt;      // [nt] rate twiddles exp(-2 pi i k/nt)
  long long per_pair, offc, pair0;
  int nap, nf, pitch, w, nt, log2m, nwin, nwords, dstride;   // dstride: tiles per pair in `dense` (k_bound's count)
  int only_above;         // 1 (every window already holds a key from the sliding kernel + k_recover): evaluate only the
                          // windows whose key exceeds the pre-threshold (the possible candidates); 0: every listed window
};

__global__ void __launch_bounds__(CE_THREADS, 2) k_coleval(ColEvalArgs a) {
  __shared__ u64 wkey[CE_TILE];
  __shared__ unsigned short list[CE_TILE * CE_CHUNK];   // entry = (word slot 2 bits | column 7 bits) << 5 | bit
  __shared__ float2 tws[2 * CE_WMAX];                   // the width's Nt <= 64 twiddles
  __shared__ int wcount[CE_THREADS / 32 + 1];
  __shared__ unsigned char need[CE_TILE];
  __shared__ float wthr[CE_TILE];                       // the windows' pre-thresholds (powers), lowered for the bound below
  __shared__ int total_sm;
  const int ntile = (a.nwin + CE_TILE - 1) / CE_TILE;
  const long long pl = blockIdx.x / ntile;
  const int tile = (int)(blockIdx.x % ntile);
  if (a.dense[pl * a.dstride + tile] || a.empty[pl * a.dstride + tile]) return;
  const int J0 = tile * CE_TILE;
  const int M = 1 << a.log2m, ntm = a.nt - 1;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x < CE_TILE) {
    wkey[threadIdx.x] = 0ull;
    bool nd = J0 + threadIdx.x < a.nwin;
    if (nd && a.only_above) {
      const long long rel = pl * a.per_pair + a.offc + J0 + threadIdx.x;
      nd = (uint32_t)(a.keys[a.pair0 * a.per_pair + rel] >> 32) > __ldg(a.thr + rel);
    }
    need[threadIdx.x] = nd ? 1 : 0;
    wthr[threadIdx.x] = J0 + threadIdx.x < a.nwin ? 0.998f * __uint_as_float(__ldg(a.thr + pl * a.per_pair + a.offc + J0 + threadIdx.x)) : 3.0e38f;
  }
  if (threadIdx.x < a.nt) tws[threadIdx.x] = __ldg(a.twt + threadIdx.x);
  const float *ybase = (const float *)(a.Y + (size_t)pl * a.nap * a.pitch);
  const size_t rowf = (size_t)a.pitch * 2u;
  for (int c0 = 0; c0 < a.nf; c0 += CE_CHUNK) {
    // ---- compaction of the (4 words) x (CE_CHUNK columns) bits of this column chunk into `list` (deterministic order)
    __syncthreads();
    int base = 0;
    for (int i0 = 0; i0 < 4 * CE_CHUNK; i0 += CE_THREADS) {
      const int i = i0 + threadIdx.x;
      const int slot = i / CE_CHUNK, col = i % CE_CHUNK;
      uint32_t bits = 0;
      if (c0 + col < a.nf && (J0 >> 5) + slot < a.nwords)
        bits = __ldg(a.mask + ((size_t)pl * a.nwords + (J0 >> 5) + slot) * a.nf + c0 + col);
      const int n = __popc(bits);
      int incl = n;                                       // warp inclusive scan
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
      if (lane == 31) wcount[warp] = incl;
      __syncthreads();
      int off = base;
      for (int k = 0; k < warp; ++k) off += wcount[k];
      int pos = off + incl - n;
      for (uint32_t b = bits; b; b &= b - 1) list[pos++] = (unsigned short)(((slot << 7 | col) << 5) | (__ffs(b) - 1));
      if (threadIdx.x == CE_THREADS - 1) total_sm = off + incl;
      __syncthreads();
      base = total_sm;
    }
    const int total = base;
    // ---- evaluation: one thread per entry
    for (int e = threadIdx.x; e < total; e += CE_THREADS) {
      const int ent = list[e];
      const int j = ((ent >> 12) << 5) | (ent & 31), d = c0 + ((ent >> 5) & 127);
      const int t0 = J0 + j;                              // stride 1
      if (!need[j]) continue;
      // a pair-interleaved row holds (re[2c], re[2c+1], im[2c], im[2c+1]) per column pair: ONE 128-bit load per sample
      // (the lanes' addresses are scattered: the load count, not the byte count, is what this kernel pays for)
      const float4 *p = (const float4 *)(ybase + (size_t)t0 * rowf) + (d >> 1);
      const bool odd = d & 1;
      float2 y[CE_WMAX];
#pragma unroll
      for (int t = 0; t < CE_WMAX; ++t) {
        if (t < a.w) {
          const float4 q = __ldg((const float4 *)((const float *)p + (size_t)t * rowf));
          y[t] = odd ? make_float2(q.y, q.w) : make_float2(q.x, q.z);
        } else y[t] = make_float2(0.f, 0.f);
      }
      float best = -1.f;
      uint32_t bidx = 0;
      const float thrw = wthr[j];
      for (int rho = 0; rho < M; ++rho) {
        float2 f[16];
#pragma unroll
        for (int t2 = 0; t2 < 16; ++t2) {
          f[t2] = cmul(y[t2], tws[(rho * t2) & ntm]);
          cmac(f[t2], y[t2 + 16], tws[(rho * (t2 + 16)) & ntm]);
        }
        // the 16 bins of this residue obey |A| <= sum_k |f[k]| <= e (the octagonal bound of kernels_sfold.cuh, 4.7 noise
        // deviations below the pre-threshold at snr_thresh 6): a residue that cannot reach the window's pre-threshold
        // cannot change the outcome (the key is replaced only by a power above it) and skips its transform
        float e = 0.f;
#pragma unroll
        for (int t2 = 0; t2 < 16; ++t2) {
          const float ax = fabsf(f[t2].x), ay = fabsf(f[t2].y);
          e += fmaxf(ax, ay) + 0.41421357f * fminf(ax, ay);
        }
        if (e * e <= thrw) continue;
        FftDif<16, 0, 16>::run(f);
#pragma unroll
        for (int s = 0; s < 16; ++s) {                    // plane order within the column: rho + M s ascending in s
          const float pw = cnorm(f[brev<16>(s)]);
          const uint32_t idx = (uint32_t)(rho + (s << a.log2m)) * (uint32_t)a.nf + (uint32_t)d;
          if (pw > best || (pw == best && idx < bidx)) { best = pw; bidx = idx; }
        }
      }
      if (best >= 0.f) atomicMax(&wkey[j], make_key(best, bidx));
    }
  }
  __syncthreads();
  if (threadIdx.x < CE_TILE && J0 + threadIdx.x < a.nwin) {
    const u64 k = wkey[threadIdx.x];
    const long long rel = pl * a.per_pair + a.offc + J0 + threadIdx.x;
    if (k && (uint32_t)(k >> 32) > __ldg(a.thr + rel)) a.keys[a.pair0 * a.per_pair + rel] = k;
  }
}

}  // namespace volks
