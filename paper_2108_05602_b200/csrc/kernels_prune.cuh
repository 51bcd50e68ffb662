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
//             thread = column pair, the running amplitude sums of its columns in a shared-memory ring (a window's
//             bound is the difference of two of them); flags[pair][width][segment] = 1 iff some (window, column) of the segment has
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
  int ncp, cp_na, cp_a0, cp_b0;   // column pairs to look at (restricted delay range): pair i < cp_na is cp_a0 + i, else cp_b0 + i - cp_na
  int w[PRUNE_MAXQ], nwin[PRUNE_MAXQ];
  long long offc[PRUNE_MAXQ];
  // column-level width (NCW = 1: the LAST listed width): besides its segment flags, one bit per (window, delay column):
  // cwmask[(pl * cw_nwords + window / 32) * nf + column], zeroed before the launch (k_coleval, kernels_coleval.cuh)
  uint32_t *cwmask;
  int cw_nwords;
  // ... and one byte per (pair, tile): 1 = more than 1/8 of the tile's (window, column) bits are set (interference,
  // a strong source): the sliding kernel evaluates that tile (it is cheaper there), k_coleval skips it
  unsigned char *cwdense;
};

template <int NQ, int NCW>
__global__ void __launch_bounds__(PRUNE_THREADS) k_bound(PruneArgs a) {
  extern __shared__ float prune_sm[];
  // shared: thr[NQ][TP] floats (TP = 2 seg + 64: 32 entries of +inf before and after the tile's windows, so that
  // window starts outside the tile need no branch), then the ring [a.ring][blockDim.x] of packed running sums
  const int T = 2 * a.seg, TP = T + 64;
  float *thr_sm = prune_sm;
  __shared__ int any[PRUNE_MAXQ][2];
  __shared__ int cwtotal;
  const int ntile = (a.nseg + 1) / 2;
  const long long pl = blockIdx.x / ntile;
  const int tile = (int)(blockIdx.x % ntile);
  const int R0 = tile * T;                                   // first window start (= first row) of the tile
  const int nthr = blockDim.x;                               // a power of two (nf / 2 or 128)
  for (int i = threadIdx.x; i < NQ * TP; i += nthr) {
    const int q = i / TP, j = i - q * TP - 32;
    thr_sm[i] = (j >= 0 && j < T && R0 + j < a.nwin[q]) ? __uint_as_float(__ldg(a.thr + pl * a.per_pair + a.offc[q] + R0 + j)) : 3.0e38f;
  }
  if (threadIdx.x < PRUNE_MAXQ * 2) any[threadIdx.x >> 1][threadIdx.x & 1] = 0;
  if (threadIdx.x == 0) cwtotal = 0;
  int cwcount = 0;
  const int nrows = min(T + a.wmax - 1, a.nap - R0);         // rows R0 .. R0 + nrows - 1 exist
  const char *ybase = (const char *)(a.Y + (size_t)pl * a.nap * a.pitch);
  const size_t rowb = (size_t)a.pitch * 8u;
  // ring of running sums C[r] = sum_{r' <= r} |Y[r']| of the thread's two columns: the bound of the window of width w
  // ending at row r is C[r] - C[r - w] (C = 0 before the tile: the ring starts zeroed).  Byte offsets wrap with one AND.
  char *ring = (char *)(prune_sm + ((NQ * TP + 3) & ~3)) + threadIdx.x * 8u;
  const uint32_t rstride = (uint32_t)nthr * 8u, rmask = (uint32_t)a.ring * rstride - 1u;
  // per width: byte offset of the leaving sum relative to the entering one, the threshold row, the first row of the
  // tile's second segment, the two flag bits
  uint32_t back[NQ], rhalf[NQ];
  const float *thq[NQ];
#pragma unroll
  for (int q = 0; q < NQ; ++q) {
    back[q] = (uint32_t)a.w[q] * rstride;
    thq[q] = thr_sm + q * TP + 33 - a.w[q];                  // thq[q][r] = pre-threshold of the window ending at row r
    rhalf[q] = (uint32_t)(a.seg + a.w[q] - 1);
  }
  __syncthreads();
  unsigned hit = 0;                                          // bit 2 q + half
  for (int ci = threadIdx.x; ci < a.ncp; ci += nthr) {
    const int c = ci < a.cp_na ? a.cp_a0 + ci : a.cp_b0 + (ci - a.cp_na);
    for (int k = 0; k < a.ring; ++k) *(f32x2 *)(ring + (uint32_t)k * rstride) = pk(0.f, 0.f);
    const char *p = ybase + (size_t)R0 * rowb + (size_t)c * 16u;
    f32x2 bx[4], by[4];                                      // four rows in flight
#pragma unroll
    for (int u = 0; u < 4; ++u) { bx[u] = by[u] = pk(0.f, 0.f); if (u < nrows) ldg2(p + (size_t)u * rowb, bx[u], by[u]); }
    f32x2 C = pk(0.f, 0.f);
    uint32_t roff = 0, cwa = 0, cwb = 0;
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
          C = add2(C, pk(aa, ab));
          f32x2 old[NQ];
          float th[NQ];
#pragma unroll
          for (int q = 0; q < NQ; ++q) {                     // (read before this row's store: for w == ring they share a slot)
            old[q] = *(const f32x2 *)(ring + ((roff - back[q]) & rmask));
            th[q] = thq[q][r];
          }
#pragma unroll
          for (int q = 0; q < NQ; ++q) {
            const f32x2 S = sub2(C, old[q]);
            const float m = fmaxf(lo32(S), hi32(S));
            const bool h = m * m > th[q];
            if (h) hit |= (uint32_t)r >= rhalf[q] ? 2u << (2 * q) : 1u << (2 * q);
            if constexpr (NCW == 1) {
              if (q == NQ - 1) {                             // the column-level width: a bit per (window, column pair)
                const int j = r - a.w[q] + 1;
                if (j >= 0 && j < T) {
                  cwa |= (lo32(S) * lo32(S) > th[q] ? 1u : 0u) << (j & 31);
                  cwb |= (hi32(S) * hi32(S) > th[q] ? 1u : 0u) << (j & 31);
                  if ((j & 31) == 31 || r == nrows - 1) {
                    cwcount += __popc(cwa) + __popc(cwb);
                    if (cwa | cwb)
                      *(uint2 *)(a.cwmask + ((size_t)pl * a.cw_nwords + ((R0 + j) >> 5)) * (size_t)a.nf + 2 * c) = make_uint2(cwa, cwb);
                    cwa = 0; cwb = 0;
                  }
                }
              }
            }
          }
          *(f32x2 *)(ring + (roff & rmask)) = C;
          roff += rstride;
        }
      }
    }
  }
#pragma unroll
  for (int q = 0; q < NQ; ++q)
#pragma unroll
    for (int h = 0; h < 2; ++h)
      if (__ballot_sync(0xffffffffu, (hit >> (2 * q + h)) & 1u) && (threadIdx.x & 31) == 0) any[q][h] = 1;
  if constexpr (NCW == 1) {
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) cwcount += __shfl_xor_sync(0xffffffffu, cwcount, o);
    if ((threadIdx.x & 31) == 0 && cwcount) atomicAdd(&cwtotal, cwcount);
  }
  __syncthreads();
  if (NCW == 1 && threadIdx.x == 0)
    a.cwdense[pl * ntile + tile] = (unsigned char)((long long)cwtotal * 8 > (long long)T * 2 * a.ncp ? 1 : 0);
  if (threadIdx.x < NQ * 2) {
    const int q = threadIdx.x >> 1, h = threadIdx.x & 1, sg = 2 * tile + h;
    if (sg < a.nseg) a.flags[(pl * NQ + q) * a.nseg + sg] = (unsigned char)any[q][h];
  }
}

}  // namespace volks
