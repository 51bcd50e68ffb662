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
  unsigned char *cwempty; // ... and 1 = no bit of the tile is set: k_coleval has nothing to list there
};

constexpr int PRUNE_MIRROR = 4;    // ring rows 0..3 are stored a second time behind the last: 4 consecutive rows never wrap

// dynamic shared memory of k_bound<NQ, NCW, NTHR>: thresholds + the ring of running sums (8 B per thread and row);
// NTHR = 64 or 128 threads (the ring's row stride is a compile-time constant)
__host__ __device__ inline size_t prune_smem_bytes(int nq, int seg, int ring, int nthr) {
  return (size_t)((nq * (2 * seg + 64) + 3) & ~3) * sizeof(float) + (size_t)(ring + PRUNE_MIRROR) * nthr * 8;
}

// Per row and thread: one 128-bit load issued EIGHT rows ahead (with four ncu read long-scoreboard 2.1 - 3.6 of 4 warps and
// half the DRAM bandwidth), the two amplitudes, one running sum; per width ONE shared-memory load (the running sum w rows
// back), a subtract, the larger column, d = bound^2 - pre-threshold, and a running maximum of d - no compare, no branch.
// The sign of the maximum is looked at three times per tile: the rows are split where the windows' segment changes (rows
// below rA belong to the tile's first segment for every width, rows from rB on to the second; the few rows in between
// flag both - a flag too many costs an evaluation, never a candidate).
// What bounds it (ncu, profiles/r02_ncu_kernels.md): the shared-memory data path (one 64-bit ring load per width and row,
// the ring store) and DRAM at 60 - 70 % of its peak; staging the rows through shared memory with cp.async 12 rows ahead
// removed the long-scoreboard stalls but added 8 wavefronts per warp-row to that path and came out even.
template <int NQ, int NCW, int NTHR>
__global__ void __launch_bounds__(NTHR) k_bound(PruneArgs a) {
  constexpr int PRUNE_RSTRIDE = NTHR * 8;    // bytes per ring row
  extern __shared__ float4 prune_sm4[];
  // shared: thr[NQ][TP] floats (TP = 2 seg + 64), indexed by the window's LAST row relative to the tile: entry r of width q
  // = pre-threshold of the window starting at row r - w[q] + 1 (+inf where the tile has no such window: no branch), then
  // the ring [a.ring + 4][NTHR] of packed running sums
  const int T = 2 * a.seg, TP = T + 64;
  float *thr_sm = (float *)prune_sm4;
  __shared__ int any[PRUNE_MAXQ][2];
  __shared__ int cwtotal;
  const int ntile = (a.nseg + 1) / 2;
  const long long pl = blockIdx.x / ntile;
  const int tile = (int)(blockIdx.x % ntile);
  const int R0 = tile * T;                                   // first window start (= first row) of the tile
  const int nthr = blockDim.x;                               // a power of two <= NTHR (nf / 2 or 128)
  for (int i = threadIdx.x; i < NQ * TP; i += nthr) {
    const int q = i / TP, j = i - q * TP - a.w[q] + 1;
    thr_sm[i] = (j >= 0 && j < T && R0 + j < a.nwin[q]) ? __uint_as_float(__ldg(a.thr + pl * a.per_pair + a.offc[q] + R0 + j)) : 3.0e38f;
  }
  if (threadIdx.x < PRUNE_MAXQ * 2) any[threadIdx.x >> 1][threadIdx.x & 1] = 0;
  if (threadIdx.x == 0) cwtotal = 0;
  int cwcount = 0;
  const int nrows = min(T + a.wmax - 1, a.nap - R0);         // rows R0 .. R0 + nrows - 1 exist
  const char *ybase = (const char *)(a.Y + (size_t)pl * a.nap * a.pitch);
  const size_t rowb = (size_t)a.pitch * 8u;
  // ring of running sums C[r] = sum_{r' <= r} |Y[r']| of the thread's two columns: the bound of the window of width w
  // ending at row r is C[r] - C[r - w] (C = 0 before the tile: the ring starts zeroed)
  char *ring = (char *)(thr_sm + ((NQ * TP + 3) & ~3)) + threadIdx.x * 8u;
  const uint32_t rmask = (uint32_t)a.ring * PRUNE_RSTRIDE - 1u;
  uint32_t back[NQ];
  int wmin = a.w[0];
#pragma unroll
  for (int q = 0; q < NQ; ++q) { back[q] = (uint32_t)a.w[q] * PRUNE_RSTRIDE; wmin = min(wmin, a.w[q]); }
  const int rA = (a.seg + wmin - 1) & ~3, rB = (a.seg + a.wmax - 1 + 3) & ~3;   // (multiples of 4: looked at per 4 rows)
  [[maybe_unused]] const int wcw = a.w[NQ - 1];
  __syncthreads();
  unsigned hit = 0;                                          // bit 2 q + half
  for (int ci = threadIdx.x; ci < a.ncp; ci += nthr) {
    const int c = ci < a.cp_na ? a.cp_a0 + ci : a.cp_b0 + (ci - a.cp_na);
    for (int k = 0; k < a.ring + PRUNE_MIRROR; ++k) *(f32x2 *)(ring + (uint32_t)k * PRUNE_RSTRIDE) = pk(0.f, 0.f);
    const char *p = ybase + (size_t)R0 * rowb + (size_t)c * 16u;
    f32x2 bx[8], by[8];                                      // eight rows in flight
#pragma unroll
    for (int u = 0; u < 8; ++u) { bx[u] = by[u] = pk(0.f, 0.f); if (u < nrows) ldg2(p + (size_t)u * rowb, bx[u], by[u]); }
    f32x2 C = pk(0.f, 0.f);
    float mx[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) mx[q] = -3.0e38f;
    uint32_t roff = 0, cwa = 0, cwb = 0, halves = 1u;        // halves: the segments (bit 0 / 1) the current rows can belong to
    // the column-level width: rows until its next word of 32 windows is complete; the word's address
    [[maybe_unused]] int cwn = wcw + 31;
    [[maybe_unused]] uint32_t *cwp = NCW == 1 ? a.cwmask + ((size_t)pl * a.cw_nwords + (R0 >> 5)) * (size_t)a.nf + 2 * c : nullptr;
    for (int r8 = 0; r8 < nrows; r8 += 8) {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int r0 = r8 + 4 * h;
      if (r0 >= nrows) break;
      if (r0 == rA || r0 == rB) {                            // (uniform) the rows' segment changes: note the sign, start afresh
#pragma unroll
        for (int q = 0; q < NQ; ++q) { if (mx[q] > 0.f) hit |= halves << (2 * q); mx[q] = -3.0e38f; }
        halves = r0 == rB ? 2u : 3u;
      }
      const char *ob[NQ];                                    // ring slot of row r0 - w[q]: this and the next 3 slots never wrap
      float4 th4[NQ];
#pragma unroll
      for (int q = 0; q < NQ; ++q) {
        ob[q] = ring + ((roff - back[q]) & rmask);
        th4[q] = *(const float4 *)(thr_sm + q * TP + r0);
      }
      const bool mir = roff == 0;
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int r = r0 + u;
        const f32x2 x = bx[4 * h + u], y = by[4 * h + u];
        if (r + 8 < nrows) ldg2(p + (size_t)(r + 8) * rowb, bx[4 * h + u], by[4 * h + u]);
        if (r < nrows) {
          const f32x2 e = fma2(y, y, mul2(x, x));
          float aa, ab;
          asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(aa) : "f"(lo32(e)));
          asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(ab) : "f"(hi32(e)));
          C = add2(C, pk(aa, ab));
#pragma unroll
          for (int q = 0; q < NQ; ++q) {                     // (read before this row's store: for w == ring they share a slot)
            const f32x2 S = sub2(C, *(const f32x2 *)(ob[q] + u * PRUNE_RSTRIDE));
            const float th = u == 0 ? th4[q].x : u == 1 ? th4[q].y : u == 2 ? th4[q].z : th4[q].w;
            const float m = fmaxf(lo32(S), hi32(S));
            mx[q] = fmaxf(mx[q], fmaf(m, m, -th));
            if constexpr (NCW == 1) {
              if (q == NQ - 1) {                             // the column-level width: a bit per (window, column)
                // th - S^2 is negative iff the column's bound exceeds the pre-threshold: its sign bit enters a shift
                // register (the latest window in bit 0: reversed when the word of 32 windows is complete)
                cwa = __funnelshift_l(__float_as_uint(fmaf(-lo32(S), lo32(S), th)), cwa, 1);
                cwb = __funnelshift_l(__float_as_uint(fmaf(-hi32(S), hi32(S), th)), cwb, 1);
                if (--cwn == 0) {                            // the window starting at this row - wcw + 1 completes a word
                  const uint32_t wa = __brev(cwa), wb = __brev(cwb);
                  cwcount += __popc(wa) + __popc(wb);
                  if (wa | wb) *(uint2 *)cwp = make_uint2(wa, wb);
                  cwp += a.nf;
                  cwn = 32;
                }
              }
            }
          }
          *(f32x2 *)(ring + roff + u * PRUNE_RSTRIDE) = C;
          if (mir) *(f32x2 *)(ring + (a.ring + u) * PRUNE_RSTRIDE) = C;
        }
      }
      roff = (roff + 4u * PRUNE_RSTRIDE) & rmask;
    }
    }
#pragma unroll
    for (int q = 0; q < NQ; ++q) if (mx[q] > 0.f) hit |= halves << (2 * q);
    if constexpr (NCW == 1) {
      if (cwn < 32) {                                        // the last, incomplete word: 32 - cwn windows, the first in bit 0
        const uint32_t wa = __brev(cwa) >> cwn, wb = __brev(cwb) >> cwn;
        cwcount += __popc(wa) + __popc(wb);
        if (wa | wb) *(uint2 *)cwp = make_uint2(wa, wb);
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
  if (NCW == 1 && threadIdx.x == 0) {
    a.cwdense[pl * ntile + tile] = (unsigned char)((long long)cwtotal * 8 > (long long)T * 2 * a.ncp ? 1 : 0);
    a.cwempty[pl * ntile + tile] = (unsigned char)(cwtotal == 0 ? 1 : 0);
  }
  if (threadIdx.x < NQ * 2) {
    const int q = threadIdx.x >> 1, h = threadIdx.x & 1, sg = 2 * tile + h;
    if (sg < a.nseg) a.flags[(pl * NQ + q) * a.nseg + sg] = (unsigned char)any[q][h];
  }
}

// ---------------------------------------------------------------------------------------------------------------
// k_pairfold - the column bits of the column-level width when it is w = 32 at Nt = 64 (M = 4 rate residues): the folded
// bound of kernels_sfold.cuh instead of the amplitude sum, in one streaming pass.
// The 16 bins r = rho + 4 s of residue rho are the 16-point DFT of f_rho[k] = y[t0 + k] W_64^{rho k} + y[t0 + k + 16]
// W_64^{rho (k + 16)}, and |f_rho[k]| = |y[t0 + k] + (-i)^rho y[t0 + k + 16]| =: A_rho[t0 + k] - no multiply, and a function of
// the ABSOLUTE row t = t0 + k alone.  So  max_s |F[rho + 4 s][d]| <= e_rho(t0) = sum_{t0 <= t < t0 + 16} A_rho[t]:  four sliding
// sums of width 16 per column.  For noise e_rho has mean 3.55 sqrt(P0), deviation 0.46 sqrt(P0) against the amplitude
// pre-threshold 5.94 sqrt(P0) (P0 = the mean bin power): 5.2 deviations, where the plain amplitude sum of k_bound has 2.0 and
// lets 2 - 3 % of the (window, column) pairs through to k_coleval.  A candidate's bin exceeds the pre-threshold, so its
// column's bit is set (exactness as for k_bound); the bits and the per-tile density bytes have k_bound's format.
//   CTA = (pair, 512 window starts), thread = column pair; per row: one 128-bit load (eight rows in flight), the row 16
//   back from registers (the loop is unrolled 16 times), four packed complex add/subtracts, four packed |.|^2, eight square roots, the four
//   amplitudes 16 rows back from a shared-memory ring, e_rho += A_new - A_old, the largest e per column, its square against the
//   window's pre-threshold by a sign-bit shift register (as in k_bound).
constexpr int PF_T = 512;          // window starts per CTA (four tiles of k_coleval: 31 halo rows per 512)
constexpr int PF_W = 32;           // the width this kernel is for (Nt = 64)
constexpr int PF_THREADS = 128;

struct PairFoldArgs {
  const float2 *Y;        // [pairs of the chunk][nap][pitch] pair-interleaved delay spectra
  const uint32_t *thr;    // pre-thresholds (float bits): thr[pl * per_pair + offc + t0]
  uint32_t *cwmask;       // [(pl * cw_nwords + window / 32) * nf + column], zeroed before the launch
  unsigned char *cwdense; // [pl * ntile128 + tile of 128 windows]
  unsigned char *cwempty; // same index: 1 = no bit of the tile is set
  long long per_pair, offc;
  int nap, nf, pitch, nwin, cw_nwords, ntile128;
  int ncp, cp_na, cp_a0, cp_b0;   // column pairs to look at (restricted delay range), as in PruneArgs
};

__host__ __device__ inline size_t pairfold_smem_bytes() {
  return (size_t)(PF_T + 64) * sizeof(float) + (size_t)4 * 16 * PF_THREADS * 8;
}

__global__ void __launch_bounds__(PF_THREADS) k_pairfold(PairFoldArgs a) {
  extern __shared__ float4 pf_sm4[];
  float *thr_sm = (float *)pf_sm4;                             // [PF_T + 64]: entry r = pre-threshold of the window ENDING at row r
  constexpr int NT128 = PF_T / 128;                            // k_coleval tiles per CTA
  __shared__ int cwtotal[NT128];
  const int ntile = (a.nwin + PF_T - 1) / PF_T;
  const long long pl = blockIdx.x / ntile;
  const int tile = (int)(blockIdx.x % ntile);
  const int R0 = tile * PF_T;
  for (int i = threadIdx.x; i < PF_T + 64; i += PF_THREADS) {
    const int j = i - PF_W + 1;
    thr_sm[i] = (j >= 0 && j < PF_T && R0 + j < a.nwin) ? __uint_as_float(__ldg(a.thr + pl * a.per_pair + a.offc + R0 + j)) : 3.0e38f;
  }
  if (threadIdx.x < NT128) cwtotal[threadIdx.x] = 0;
  const int nrows = min(PF_T + PF_W - 1, a.nap - R0);
  const char *ybase = (const char *)(a.Y + (size_t)pl * a.nap * a.pitch);
  const size_t rowb = (size_t)a.pitch * 8u;
  // ring (slot = row & 15) of the amplitudes [4][16][PF_THREADS] f32x2
  char *amp = (char *)(thr_sm + PF_T + 64) + threadIdx.x * 8u;
  constexpr uint32_t AMPROW = PF_THREADS * 8, AMPRHO = 16 * AMPROW;
  __syncthreads();
  int cnt[NT128];                                              // set bits per tile of 128 windows
#pragma unroll
  for (int i = 0; i < NT128; ++i) cnt[i] = 0;
  for (int ci = threadIdx.x; ci < a.ncp; ci += PF_THREADS) {
    const int c = ci < a.cp_na ? a.cp_a0 + ci : a.cp_b0 + (ci - a.cp_na);
    for (int k = 0; k < 64; ++k) *(f32x2 *)(amp + (uint32_t)k * AMPROW) = pk(0.f, 0.f);
    const char *p = ybase + (size_t)R0 * rowb + (size_t)c * 16u;
    f32x2 bx[8], by[8];                                        // eight rows in flight
    f32x2 px[16], py[16];                                      // the sixteen rows before the current one (registers, not a ring)
#pragma unroll
    for (int u = 0; u < 8; ++u) { bx[u] = by[u] = pk(0.f, 0.f); if (u < nrows) ldg2(p + (size_t)u * rowb, bx[u], by[u]); }
#pragma unroll
    for (int u = 0; u < 16; ++u) px[u] = py[u] = pk(0.f, 0.f);
    f32x2 e0 = pk(0.f, 0.f), e1 = e0, e2 = e0, e3 = e0;
    uint32_t cwa = 0, cwb = 0;
    int cwn = PF_W + 31;                                       // rows until the next word of 32 windows is complete
    uint32_t *cwp = a.cwmask + ((size_t)pl * a.cw_nwords + (R0 >> 5)) * (size_t)a.nf + 2 * c;
    int nword = 0;
    for (int r16 = 0; r16 < nrows; r16 += 16) {
#pragma unroll
      for (int u = 0; u < 16; ++u) {
        const int r = r16 + u;
        const f32x2 x = bx[u & 7], y = by[u & 7];
        if (r + 8 < nrows) ldg2(p + (size_t)(r + 8) * rowb, bx[u & 7], by[u & 7]);
        if (r < nrows) {
          const uint32_t slot = (uint32_t)u;                   // = r & 15: after unrolling the ring offsets are immediates
          const f32x2 xo = px[u], yo = py[u];                  // the row 16 back: the class's first sample
          px[u] = x; py[u] = y;
          if (r16 > 0) {
            // f_rho = y[t] + (-i)^rho y[t + 16]:  rho 0: (xo + x, yo + y), 1: (xo + y, yo - x), 2: (xo - x, yo - y), 3: (xo - y, yo + x)
            const f32x2 ax0 = add2(xo, x), ay0 = add2(yo, y), ax2 = sub2(xo, x), ay2 = sub2(yo, y);
            const f32x2 ax1 = add2(xo, y), ay1 = sub2(yo, x), ax3 = sub2(xo, y), ay3 = add2(yo, x);
            const f32x2 p0 = fma2(ay0, ay0, mul2(ax0, ax0)), p1 = fma2(ay1, ay1, mul2(ax1, ax1));
            const f32x2 p2 = fma2(ay2, ay2, mul2(ax2, ax2)), p3 = fma2(ay3, ay3, mul2(ax3, ax3));
            float s0a, s0b, s1a, s1b, s2a, s2b, s3a, s3b;
            asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(s0a) : "f"(lo32(p0)));
            asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(s0b) : "f"(hi32(p0)));
            asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(s1a) : "f"(lo32(p1)));
            asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(s1b) : "f"(hi32(p1)));
            asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(s2a) : "f"(lo32(p2)));
            asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(s2b) : "f"(hi32(p2)));
            asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(s3a) : "f"(lo32(p3)));
            asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(s3b) : "f"(hi32(p3)));
            const f32x2 A0 = pk(s0a, s0b), A1 = pk(s1a, s1b), A2 = pk(s2a, s2b), A3 = pk(s3a, s3b);
            char *as = amp + slot * AMPROW;                    // the amplitudes of row t - 16 leave, those of t = r - 16 enter
            e0 = add2(e0, sub2(A0, *(const f32x2 *)(as)));
            e1 = add2(e1, sub2(A1, *(const f32x2 *)(as + AMPRHO)));
            e2 = add2(e2, sub2(A2, *(const f32x2 *)(as + 2 * AMPRHO)));
            e3 = add2(e3, sub2(A3, *(const f32x2 *)(as + 3 * AMPRHO)));
            *(f32x2 *)(as) = A0; *(f32x2 *)(as + AMPRHO) = A1; *(f32x2 *)(as + 2 * AMPRHO) = A2; *(f32x2 *)(as + 3 * AMPRHO) = A3;
          }
          // the window ending at this row (start r - 31): the largest of the four bounds per column, squared, against its
          // pre-threshold; the sign bit of thr - e^2 enters the shift register (latest window in bit 0)
          const float ma = fmaxf(fmaxf(lo32(e0), lo32(e1)), fmaxf(lo32(e2), lo32(e3)));
          const float mb = fmaxf(fmaxf(hi32(e0), hi32(e1)), fmaxf(hi32(e2), hi32(e3)));
          const float th = thr_sm[r];
          cwa = __funnelshift_l(__float_as_uint(fmaf(-ma, ma, th)), cwa, 1);
          cwb = __funnelshift_l(__float_as_uint(fmaf(-mb, mb, th)), cwb, 1);
          if (--cwn == 0) {
            const uint32_t wa = __brev(cwa), wb = __brev(cwb);
            const int n = __popc(wa) + __popc(wb);
#pragma unroll
            for (int i = 0; i < NT128; ++i) cnt[i] += (nword >> 2) == i ? n : 0;
            if (wa | wb) *(uint2 *)cwp = make_uint2(wa, wb);
            cwp += a.nf; ++nword;
            cwn = 32;
          }
        }
      }
    }
    if (cwn < 32) {                                            // the last, incomplete word
      const uint32_t wa = __brev(cwa) >> cwn, wb = __brev(cwb) >> cwn;
      const int n = __popc(wa) + __popc(wb);
#pragma unroll
      for (int i = 0; i < NT128; ++i) cnt[i] += (nword >> 2) == i ? n : 0;
      if (wa | wb) *(uint2 *)cwp = make_uint2(wa, wb);
    }
  }
#pragma unroll
  for (int i = 0; i < NT128; ++i) {
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) cnt[i] += __shfl_xor_sync(0xffffffffu, cnt[i], o);
    if ((threadIdx.x & 31) == 0 && cnt[i]) atomicAdd(&cwtotal[i], cnt[i]);
  }
  __syncthreads();
  if (threadIdx.x < NT128 && NT128 * tile + (int)threadIdx.x < a.ntile128) {   // dense: more than 1/8 of the 128 x columns bits (k_bound's rule)
    a.cwdense[pl * a.ntile128 + NT128 * tile + threadIdx.x] = (unsigned char)((long long)cwtotal[threadIdx.x] * 8 > 128LL * 2 * a.ncp ? 1 : 0);
    a.cwempty[pl * a.ntile128 + NT128 * tile + threadIdx.x] = (unsigned char)(cwtotal[threadIdx.x] == 0 ? 1 : 0);
  }
}

}  // namespace volks
