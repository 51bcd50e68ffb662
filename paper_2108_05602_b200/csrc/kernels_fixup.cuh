// kernels_fixup.cuh - exact re-evaluation of the windows the sliding sum cannot resolve.
//
// k_slide adds and removes samples from a running sum, so a sample leaves a rounding residue of about
// 6e-8 of ITS size behind until the segment restarts.  A window whose peak power is far below that of
// an earlier window of its segment (the zero fill of dedispersion, the edge of flagged data, the fall
// of a strong RFI burst) would carry that residue as a relative error above the 1e-4 parity bound.
//   k_fixup   one CTA per (pair, sliding width, segment): prefix maximum of the segment's peak powers;
//             every window whose power is below SLIDE_FIX_RATIO times the maximum before it is
//             recomputed from its samples by the definition (fold + L-point FFT per (rate residue,
//             column), as kernels_generic.cuh k_col) and its key replaced.  Deterministic, no atomics.
// DESIGN.md section 7 ("Accuracy of the sliding sum").
#pragma once
#include "common.cuh"

namespace volks {

#ifndef SLIDE_FIX_RATIO
#define SLIDE_FIX_RATIO 1e-3f   // power ratio 1000 = amplitude ratio 32: residue 2 * 32 * 6e-8 * sqrt(256) = 6e-5 relative at most
#endif

struct FixArgs {
  const float2 *Y;       // [npairs_chunk][nap][pitch]
  u64 *keys;
  const float2 *tables;  // plan tables; rate twiddles of width q at tables + tw_off[q]
  long long per_pair, pair0;
  int nap, nf, log2nf, pitch, paired;
  int nq;                // sliding widths in this plan
  int q[16], w[16], nt[16], seg[16], nseg[16], nwin[16];
  long long offc[16], tw_off[16];
  int unit0[17];         // prefix sums of nseg over the sliding widths (units per pair = unit0[nq])
  // pruned widths (kernels_prune.cuh): segments whose flag is 0 were not evaluated (all keys zero): nothing to fix
  const unsigned char *flags;   // [pairs of the chunk][flag_nq][flag_nseg] or nullptr
  int flag_q[16];               // index of sliding width i among the pruned widths, or -1
  int flag_nq, flag_nseg;
  // the column-level width (kernels_coleval.cuh) in the candidates-only mode: its sliding kernel ran only on the tiles
  // k_bound marked dense: cwdense[pl * cw_ntile + segment] (its segments are those tiles); cw_i = its index here or -1
  const unsigned char *cwdense;
  int cw_i, cw_ntile;
  // a folded-sum width (kernels_sfold.cuh) in the candidates-only mode: sfdense[i][pl * nseg[i] + segment] = 1 for the
  // segments the sliding kernel evaluated; nullptr = every segment
  const unsigned char *sfdense[16];
};

// peak key of rate residue rho, column d of the window starting at row0 (already includes pair and t0)
template <int L>
__device__ __forceinline__ u64 fix_task(const FixArgs &a, const float2 *twt, size_t row0, int w, int nt, int rho, int d) {
  float2 acc[L];
#pragma unroll
  for (int i = 0; i < L; ++i) acc[i] = make_float2(0.f, 0.f);
  const int ntm = nt - 1, log2m = 31 - __clz(nt / L);
  for (int tb = 0; tb < w; tb += L) {
#pragma unroll
    for (int t2 = 0; t2 < L; ++t2) {
      const int t = tb + t2;
      if (t < w) cmac(acc[t2], ld_y(a.Y, (row0 + t) * a.pitch, d, a.paired), __ldg(twt + ((rho * t) & ntm)));
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
  return make_key(best, (uint32_t)(rho + (bs << log2m)) * (uint32_t)a.nf + (uint32_t)d);
}

constexpr int FIX_GROUP = 16;   // segments per CTA (a unit): most are skipped at once, a CTA per segment was launch-bound

__global__ void __launch_bounds__(256) k_fixup(FixArgs a) {
  __shared__ float pmax[256];
  __shared__ u64 red[8];
  __shared__ int flagged[256];
  __shared__ int nflag;
  const int upp = a.unit0[a.nq];
  const long long pl = blockIdx.x / upp;
  int u = (int)(blockIdx.x % upp), i = 0;
  while (u >= a.unit0[i + 1]) ++i;
  const int sg_lo = (u - a.unit0[i]) * FIX_GROUP, sg_hi = min(a.nseg[i], sg_lo + FIX_GROUP);
  // which of the unit's segments were evaluated at all: the 16 flag bytes in ONE round trip (thread per segment) - read
  // one after the other by the whole CTA they were most of this kernel's time on a pruned search
  __shared__ unsigned char todo[FIX_GROUP];
  if (threadIdx.x < FIX_GROUP) {
    const int sg = sg_lo + (int)threadIdx.x;
    bool run = sg < sg_hi;
    if (run && a.flags && a.flag_q[i] >= 0 && !a.flags[(pl * a.flag_nq + a.flag_q[i]) * a.flag_nseg + sg]) run = false;
    if (run && a.cwdense && i == a.cw_i && !a.cwdense[pl * a.cw_ntile + sg]) run = false;
    if (run && a.sfdense[i] && !a.sfdense[i][pl * a.nseg[i] + sg]) run = false;
    todo[threadIdx.x] = run ? 1 : 0;
  }
  __syncthreads();
  for (int sg = sg_lo; sg < sg_hi; ++sg) {
  if (!todo[sg - sg_lo]) continue;
  const int w = a.w[i], nt = a.nt[i], seg = a.seg[i];
  const int j0 = sg * seg, n = min(seg, a.nwin[i] - j0);          // windows j0 .. j0+n-1 (seg <= 256? see below)
  u64 *keyp = a.keys + ((a.pair0 + pl) * a.per_pair + a.offc[i]);
  const float2 *twt = a.tables + a.tw_off[i];
  const int L = min(16, nt), M = nt / L;
  for (int base = 0; base < n; base += 256) {                      // segments longer than 256 windows: in pieces,
    const int m = min(256, n - base);                              // the running maximum carried in `carry`
    __shared__ float carry;
    if (threadIdx.x == 0 && base == 0) carry = 0.f;
    __syncthreads();
    const float mine = threadIdx.x < m ? key_power(keyp[j0 + base + threadIdx.x]) : 0.f;
    pmax[threadIdx.x] = fmaxf(mine, carry);
    __syncthreads();
    for (int o = 1; o < 256; o <<= 1) {                            // inclusive prefix maximum
      const float v = threadIdx.x >= o ? pmax[threadIdx.x - o] : 0.f;
      __syncthreads();
      pmax[threadIdx.x] = fmaxf(pmax[threadIdx.x], v);
      __syncthreads();
    }
    if (threadIdx.x == 0) nflag = 0;
    __syncthreads();
    if (threadIdx.x < m && mine < SLIDE_FIX_RATIO * pmax[threadIdx.x]) flagged[atomicAdd(&nflag, 1)] = threadIdx.x;
    __syncthreads();
    const int nf_ = nflag;
    for (int k = 0; k < nf_; ++k) {
      // lowest flagged window first is not needed: every flagged window is recomputed independently
      const int j = j0 + base + flagged[k];
      const size_t row0 = (size_t)pl * a.nap + (size_t)j;           // stride 1: t0 = j
      u64 key = 0;
      for (int t = threadIdx.x; t < M * a.nf; t += 256) {
        const int d = t & (a.nf - 1), rho = t >> a.log2nf;
        u64 kk;
        if (L == 16) kk = fix_task<16>(a, twt, row0, w, nt, rho, d);
        else if (L == 8) kk = fix_task<8>(a, twt, row0, w, nt, rho, d);
        else kk = fix_task<4>(a, twt, row0, w, nt, rho, d);
        key = kk > key ? kk : key;
      }
#pragma unroll
      for (int o = 16; o >= 1; o >>= 1) {
        const u64 other = __shfl_xor_sync(0xffffffffu, key, o);
        key = other > key ? other : key;
      }
      if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = key;
      __syncthreads();
      if (threadIdx.x == 0) {
        for (int r = 1; r < 8; ++r) key = red[r] > key ? red[r] : key;
        keyp[j] = key;
      }
      __syncthreads();
    }
    if (threadIdx.x == 0) carry = pmax[255];
    __syncthreads();
  }
  }
}

}  // namespace volks
