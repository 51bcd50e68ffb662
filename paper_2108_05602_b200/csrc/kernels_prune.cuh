// kernels_prune.cuh - exact pruning of the narrow stride-1 widths in the candidates-only index mode.
//
// A window can only be a candidate if its peak power exceeds snr_thresh^2 times its noise (a7).  For one delay
// column d the rate transform of a window is a sum of w unit-modulus multiples of its samples, so by the
// triangle inequality, for EVERY rate bin r,
//     |F[r][d]|  <=  sum_{t0 <= t < t0+w} |Y[t][d]|         (Y = the per-AP delay spectra)
// and the right-hand side slides along t0 at one add and one subtract per window and column - no transform.
// For noise the bound stays far below the threshold when w is small (|Y| is Rayleigh distributed: the sum of w
// amplitudes has mean 0.886 w sigma and deviation 0.46 sqrt(w) sigma, the threshold sits at snr_thresh sqrt(w)
// sigma: 7.4 / 5.2 deviations above the mean for w = 8 / 16 at snr_thresh 6), so the rate transform, |.|^2 and
// the peak search of a whole segment of windows are needed only where some window of it comes near the threshold
// in some column: around pulses and interference.
//   k_bound   one pass over the chunk's delay spectra: CTA = (pair, tile of 2 segments of window starts),
//             thread = column pair, the last 32 amplitudes of its columns in a shared-memory ring, one running
//             sum per pruned width; flags[pair][width][segment] = 1 iff some (window, column) of the segment has
//             bound^2 > pre-threshold of that window (k_winthr: 0.98 snr_thresh^2 noise - the 2 % cover every
//             rounding on both sides).  The sliding kernels return at once for a segment whose flag is 0; its
//             windows keep the zero key (power 0, snr 0: not candidates - which is all the mode promises).
// Exactness: a candidate has P1 > snr_thresh^2 noise > pre-threshold >= ... so its segment is flagged and is then
// evaluated completely by the same kernels as without pruning: candidates are bit-identical (tested).
#pragma once
#include "common.cuh"

namespace volks {

constexpr int PRUNE_MAXQ = 8;      // pruned widths per plan
constexpr int PRUNE_RING = 32;     // most rows of amplitude history: pruned widths are <= 32 APs
constexpr int PRUNE_THREADS = 128;

struct PruneArgs {
  const float2 *Y;        // [pairs of the chunk][nap][pitch] pair-interleaved delay spectra
  const uint32_t *thr;    // pre-thresholds as float bits: thr[pl * per_pair + offc + t0]
  unsigned char *flags;   // [pairs of the chunk][nq][nseg]
  long long per_pair;
  int nap, nf, pitch, nq, seg, nseg, wmax, ring;
  int w[PRUNE_MAXQ], nwin[PRUNE_MAXQ];
  long long offc[PRUNE_MAXQ];
};

__global__ void __launch_bounds__(PRUNE_THREADS) k_bound(PruneArgs a) {
  extern __shared__ float prune_sm[];
  // shared: thr[nq][2 seg] floats, then the ring [a.ring][blockDim.x] of packed amplitude pairs
  const int T = 2 * a.seg;
  float *thr_sm = prune_sm;
  f32x2 *ring = (f32x2 *)(prune_sm + ((a.nq * T + 3) & ~3));
  __shared__ int any[PRUNE_MAXQ][2];
  const int ntile = (a.nseg + 1) / 2;
  const long long pl = blockIdx.x / ntile;
  const int tile = (int)(blockIdx.x % ntile);
  const int R0 = tile * T;                                   // first window start (= first row) of the tile
  const int nthr = blockDim.x, rmask = a.ring - 1;
  for (int i = threadIdx.x; i < a.nq * T; i += nthr) {
    const int q = i / T, j = i - q * T;
    thr_sm[i] = R0 + j < a.nwin[q] ? __uint_as_float(__ldg(a.thr + pl * a.per_pair + a.offc[q] + R0 + j)) : 3.0e38f;
  }
  if (threadIdx.x < PRUNE_MAXQ * 2) any[threadIdx.x >> 1][threadIdx.x & 1] = 0;
  __syncthreads();
  const int nrows = min(T + a.wmax - 1, a.nap - R0);         // rows R0 .. R0 + nrows - 1 exist
  const char *ybase = (const char *)(a.Y + (size_t)pl * a.nap * a.pitch);
  const size_t rowb = (size_t)a.pitch * 8u;
  f32x2 *myring = ring + threadIdx.x;
  unsigned hit = 0;                                          // bit 2 q + half
  for (int c = threadIdx.x; c < (a.nf >> 1); c += nthr) {
    f32x2 S[PRUNE_MAXQ];
#pragma unroll
    for (int q = 0; q < PRUNE_MAXQ; ++q) S[q] = pk(0.f, 0.f);
    const char *p = ybase + (size_t)R0 * rowb + (size_t)c * 16u;
    f32x2 bx[4], by[4];                                      // four rows in flight
#pragma unroll
    for (int u = 0; u < 4; ++u) { bx[u] = by[u] = pk(0.f, 0.f); if (u < nrows) ldg2(p + (size_t)u * rowb, bx[u], by[u]); }
    for (int r0 = 0; r0 < nrows; r0 += 4) {
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int r = r0 + u;
        const f32x2 x = bx[u], y = by[u];
        if (r + 4 < nrows) ldg2(p + (size_t)(r + 4) * rowb, bx[u], by[u]);
        if (r < nrows) {
          const f32x2 e = fma2(y, y, mul2(x, x));
          float aa, ab;
          asm("sqrt.approx.f32 %0, %1;" : "=f"(aa) : "f"(lo32(e)));
          asm("sqrt.approx.f32 %0, %1;" : "=f"(ab) : "f"(hi32(e)));
          const f32x2 amp = pk(aa, ab);
          // (the leaving amplitudes are read BEFORE the new one is stored: for w == ring they share a slot)
#pragma unroll
          for (int q = 0; q < PRUNE_MAXQ; ++q) {
            if (q < a.nq) {                                  // uniform
              const int wq = a.w[q];
              S[q] = add2(S[q], amp);
              if (r >= wq) S[q] = sub2(S[q], myring[((r - wq) & rmask) * nthr]);
            }
          }
          myring[(r & rmask) * nthr] = amp;
#pragma unroll
          for (int q = 0; q < PRUNE_MAXQ; ++q) {
            if (q < a.nq) {
              const int j = r - a.w[q] + 1;                  // window start relative to the tile
              if (j >= 0 && j < T) {
                const float th = thr_sm[q * T + j];
                const float sa = lo32(S[q]), sb = hi32(S[q]);
                if (sa * sa > th || sb * sb > th) hit |= 1u << (2 * q + (j >= a.seg ? 1 : 0));
              }
            }
          }
        }
      }
    }
  }
  for (int q = 0; q < a.nq; ++q)
    for (int h = 0; h < 2; ++h)
      if (__ballot_sync(0xffffffffu, (hit >> (2 * q + h)) & 1u) && (threadIdx.x & 31) == 0) any[q][h] = 1;
  __syncthreads();
  if (threadIdx.x < a.nq * 2) {
    const int q = threadIdx.x >> 1, h = threadIdx.x & 1, sg = 2 * tile + h;
    if (sg < a.nseg) a.flags[(pl * a.nq + q) * a.nseg + sg] = (unsigned char)any[q][h];
  }
}

}  // namespace volks
