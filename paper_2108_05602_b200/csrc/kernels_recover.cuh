// kernels_recover.cuh - the peak bin of the stride-1 windows whose sliding kernel ran without bin tags.
//
// k_slide (w >= 16) and k_colfft2 (Nt = 256, 512) leave per window the maximum power and the COLUMN it came from: one rate residue rho and one
// delay column d, i.e. the 16 rate bins r = rho + M s of that column.  Which of them is the peak is decided here:
//   k_recover   one thread per (pair, width, window).  The thread leaves at once unless the window needs its index:
//               every window in the full-index mode (dense peaks, volks_zscore_select), otherwise the windows whose
//               power exceeds their pre-threshold (k_winthr: 0.98 of what a candidate needs).  It folds the window's
//               w samples of column d with W_Nt^{rho t} into 16 sums and runs a 16-point transform (the definition
//               of the rate DFT for this residue, as k_col / k_fixup), takes |.|^2 and the first maximum, and the
//               window's key becomes (exact power, exact plane index).  A reported power and index therefore never
//               carry the sliding sum's rounding.
// Plane indices stay below 2^31 (plan validation), so bit 31 of a key's index marks "a column, not yet a bin".  The
// kernel runs after k_fixup, whose exact keys it leaves alone; k_fixup decides from the sliding powers, so both
// index modes re-evaluate the same windows and give bit-identical candidates.
// The column is the one that won in the sliding pass; another column whose maximum lies within the sliding sum's
// rounding (1e-6) of it could hold the true first argmax - a near-tie far inside the 1e-5 exemption of the
// comparison rule.
#pragma once
#include "common.cuh"

namespace volks {

struct RecoverArgs {
  const float2 *Y;        // [pairs of the chunk][nap][pitch] pair-interleaved delay spectra
  u64 *keys;
  const uint32_t *thr;    // pre-thresholds (float bits), chunk-relative: thr[pl * per_pair + offc + t0]; nullptr = every window
  const float2 *tables;   // plan tables; rate twiddles of width i at tables + tw_off[i]
  long long per_pair, pair0, total;   // total = pairs of the chunk * cum[nq]
  int nap, nf, log2nf, pitch, nq;
  int w[16], stride[16], nt[16], log2m[16], nwin[16];
  long long offc[16], tw_off[16], cum[17];   // cum: prefix sums of nwin (windows per pair of the listed widths)
};

__global__ void __launch_bounds__(128) k_recover(RecoverArgs a) {
  const long long gid = (long long)blockIdx.x * 128 + threadIdx.x;       // thread = (pair, width, window)
  if (gid >= a.total) return;
  const long long per = a.cum[a.nq];
  const long long pl = gid / per;
  long long r = gid - pl * per;
  int i = 0;
  while (i + 1 < a.nq && r >= a.cum[i + 1]) ++i;
  const int j = (int)(r - a.cum[i]);
  u64 *kp = a.keys + ((a.pair0 + pl) * a.per_pair + a.offc[i] + j);
  const u64 k0 = *kp;
  const uint32_t pbits = (uint32_t)(k0 >> 32);
  if (pbits == 0u) return;                                               // not evaluated (pruned) or identically zero
  const uint32_t tidx = key_index(k0);
  if (!(tidx >> 31)) return;                                             // already a bin (k_fixup re-evaluated the window)
  if (a.thr && pbits <= __ldg(a.thr + pl * a.per_pair + a.offc[i] + j)) return;
  const uint32_t idx0 = tidx & 0x7FFFFFFFu;                              // rho * nf + d
  const uint32_t rho = idx0 >> a.log2nf, d = idx0 & (uint32_t)(a.nf - 1);
  const int w = a.w[i], ntm = a.nt[i] - 1;
  const float2 *twt = a.tables + a.tw_off[i];
  // element d of a pair-interleaved row: float index 4 (d / 2) + (d & 1), imaginary part 2 floats on
  const float *p = (const float *)(a.Y + ((size_t)pl * a.nap + (size_t)j * a.stride[i]) * a.pitch) + ((d >> 1) << 2) + (d & 1);   // t0 = j * stride
  const size_t rowf = (size_t)a.pitch * 2u;
  float2 f[16];
#pragma unroll
  for (int t2 = 0; t2 < 16; ++t2) f[t2] = make_float2(0.f, 0.f);
  for (int tb = 0; tb < w; tb += 16) {
    float2 y[16];
#pragma unroll
    for (int t2 = 0; t2 < 16; ++t2) {                                    // 16 rows in flight
      const int t = tb + t2;
      y[t2] = t < w ? make_float2(__ldg(p + (size_t)t * rowf), __ldg(p + (size_t)t * rowf + 2)) : make_float2(0.f, 0.f);
    }
#pragma unroll
    for (int t2 = 0; t2 < 16; ++t2) {
      const int t = tb + t2;
      if (t < w) cmac(f[t2], y[t2], __ldg(twt + ((rho * (uint32_t)t) & (uint32_t)ntm)));
    }
  }
  FftDif<16, 0, 16>::run(f);
  float best = -1.f;
  int bs = 0;
#pragma unroll
  for (int s = 0; s < 16; ++s) {
    const float pw = cnorm(f[brev<16>(s)]);
    if (pw > best) { best = pw; bs = s; }
  }
  *kp = make_key(best, idx0 + (((uint32_t)bs << a.log2m[i]) << a.log2nf));
}

}  // namespace volks
