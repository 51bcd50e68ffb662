// volks_api.cu - C-ABI entry points (include/volks.h): plan / window scheduler, launches, host helpers.
#include "../../include/volks.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "kernels_generic.cuh"
#include "kernels_slide.cuh"
#include "kernels_colfft2.cuh"
#include "kernels_colfft.cuh"
#include "kernels_allif.cuh"
#include "kernels_fixup.cuh"
#include "kernels_probe.cuh"
#include "kernels_prune.cuh"
#include "kernels_recover.cuh"
#include "kernels_coleval.cuh"
#include "kernels_sfold.cuh"

using namespace volks;

namespace {

thread_local char g_cuda_msg[256] = "";

inline bool is_pow2(long long n) { return n >= 1 && (n & (n - 1)) == 0; }
inline int ilog2(long long n) { int l = 0; while ((1LL << l) < n) ++l; return l; }
inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

bool cuda_ok(cudaError_t e) {
  if (e == cudaSuccess) return true;
  snprintf(g_cuda_msg, sizeof g_cuda_msg, "%s", cudaGetErrorString(e));
  return false;
}

// one width's entry of the window schedule (a1)
struct WidthPlan {
  int w, s, nt, L, log2m;
  long long nwin;       // per pair
  size_t tw_off;        // offset (float2) of its rate twiddle table in d_tables
  size_t tw4_off;       // offset (float2, even) of the pre-broadcast copy (re, re, im, im) used by k_slide
  bool slide;           // stride-1 sliding-sum kernel (kernels_slide.cuh) instead of the generic one
  bool colfft;          // two-pass shared-memory column FFT (kernels_colfft.cuh): Nt = 32..512, nf % 32 == 0
  int cf_l1, cf_nz, cf_wpc, cf_nrange;
  int seg, nseg;        // sliding path: windows per exactly restarted segment, segments per pair
  bool untag;           // sliding path with M >= 2 (Nt >= 32): untagged kernel, peak bin by k_recover
  int prune;            // sliding path: index among the plan's pruned widths (kernels_prune.cuh), or -1
  bool cw;              // sliding path: the plan's column-level width (kernels_coleval.cuh)
  bool sf;              // sliding path, candidates-only mode: folded sliding sum + evaluation of the flagged tiles (kernels_sfold.cuh)
  size_t off_hits;      // ... its hit masks in the workspace
  size_t off_sfdense;   // ... its per-segment density flags
  size_t off_sflist;    // ... the list of non-zero mask words (count first)
  size_t off_sfbig;     // ... one 16-bit word per block of 16 rows: rows of overwhelming energy (k_sfold_guard)
  int nblk;             // ... blocks of 16 windows per pair
};

template <int L>
static void launch_col(const ColArgs &a, cudaStream_t st) {
  const long long blocks = (a.total + 255) / 256;
  k_col<L><<<(unsigned)blocks, 256, 0, st>>>(a);
}

inline size_t colfft_smem(int l1, int nt) { return (size_t)l1 * 16 * 32 * sizeof(float2) + (size_t)nt * sizeof(float4) + (size_t)l1 * sizeof(u64); }

template <int L1, int NZ>
static cudaError_t colfft_one(const ColFftArgs &a, unsigned blocks, cudaStream_t st, bool attr_only) {
  const size_t smem = colfft_smem(L1, a.nt);
  if constexpr (L1 >= 16) {
    // Nt = 256 / 512: two columns per thread in split format (kernels_colfft2.cuh) unless VOLKS_CF2=0
    const bool cf2 = a.split2 != 0;
    // k_colfft2: 512 twiddles + the strip S[L1][16][CP] + 16 slots
    const size_t smem8 = 512 * sizeof(float4) + (size_t)L1 * 16 * 8 * sizeof(float4) + 16 * sizeof(u64);
    const size_t smem8e = smem8 + (size_t)L1 * CF2E_RHO;   // k_colfft2e: + the energy strip
    const size_t smem4 = 512 * sizeof(float4) + (size_t)L1 * (256 * 4 + 32) + 16 * sizeof(u64);
    const size_t smem16 = 512 * sizeof(float4) + (size_t)L1 * 16 * 16 * sizeof(float4) + 16 * sizeof(u64);
    if (attr_only) {
      cudaError_t e = cudaFuncSetAttribute(k_colfft2<L1, NZ, 16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem16);
      if (e == cudaSuccess) e = cudaFuncSetAttribute(k_colfft2<L1, NZ, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem8);
      if (e == cudaSuccess) e = cudaFuncSetAttribute(k_colfft2<L1, NZ, 8, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem8);
      if (e == cudaSuccess) e = cudaFuncSetAttribute(k_colfft2e<L1, NZ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem8e);
      if (e == cudaSuccess) e = cudaFuncSetAttribute(k_colfft2<L1, NZ, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem4);
      if (e != cudaSuccess) return e;
    } else if (a.split2 == 4) {   // 8-column strips: four times the CTAs, 128 threads each
      k_colfft2<L1, NZ, 4><<<blocks * 4, 128, smem4, st>>>(a);
      return cudaSuccess;
    } else if (a.split2 == 2) {   // 16-column strips: twice the CTAs, 256 threads each
      // candidates-only mode: energies first (measured on configs[4]: w = 64 / 128 / 256 take 52.7 / 41.9 / 33.9 ms per step
      // with it, 66.4 / 42.4 / 30.4 ms with k_colfft2<SKIP>: the widest windows keep the older kernel)
      if (a.thr && a.energy_first && NZ <= 8) k_colfft2e<L1, NZ><<<blocks * 2, 256, smem8e, st>>>(a);
      else if (a.thr) k_colfft2<L1, NZ, 8, true><<<blocks * 2, 256, smem8, st>>>(a);   // ... pass 2 only where needed
      else k_colfft2<L1, NZ, 8><<<blocks * 2, 256, smem8, st>>>(a);
      return cudaSuccess;
    } else if (cf2) {
      k_colfft2<L1, NZ, 16><<<blocks, CF_WARPS * 32, smem16, st>>>(a);
      return cudaSuccess;
    }
  }
  if (attr_only) return cudaFuncSetAttribute(k_colfft<L1, NZ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  k_colfft<L1, NZ><<<blocks, CF_WARPS * 32, smem, st>>>(a);
  return cudaSuccess;
}

template <int L1>
static cudaError_t colfft_l1(const ColFftArgs &a, int nz, unsigned blocks, cudaStream_t st, bool attr_only) {
  switch (nz) {
    case 1: return colfft_one<L1, 1>(a, blocks, st, attr_only);
    case 2: return colfft_one<L1, 2>(a, blocks, st, attr_only);
    case 4: if constexpr (L1 >= 4) return colfft_one<L1, 4>(a, blocks, st, attr_only); break;
    case 8: if constexpr (L1 >= 8) return colfft_one<L1, 8>(a, blocks, st, attr_only); break;
    case 16: if constexpr (L1 >= 16) return colfft_one<L1, 16>(a, blocks, st, attr_only); break;
    case 32: if constexpr (L1 >= 32) return colfft_one<L1, 32>(a, blocks, st, attr_only); break;
  }
  return cudaErrorInvalidValue;
}

// attr_only: raise the kernel's dynamic shared memory limit (plan creation) instead of launching
static cudaError_t launch_colfft(const ColFftArgs &a, int l1, int nz, long long units, cudaStream_t st, bool attr_only) {
  const unsigned blocks = (unsigned)units;
  switch (l1) {
    case 2: return colfft_l1<2>(a, nz, blocks, st, attr_only);
    case 4: return colfft_l1<4>(a, nz, blocks, st, attr_only);
    case 8: return colfft_l1<8>(a, nz, blocks, st, attr_only);
    case 16: return colfft_l1<16>(a, nz, blocks, st, attr_only);
    case 32: return colfft_l1<32>(a, nz, blocks, st, attr_only);
  }
  return cudaErrorInvalidValue;
}

template <int N1, int N2>
static bool row2_nz(const RowArgs &a, int nza, unsigned blocks, cudaStream_t st) {
  switch (nza) {
    case 1: k_row2<N1, N2, 1><<<blocks, 256, 0, st>>>(a); return true;
    case 2: k_row2<N1, N2, 2><<<blocks, 256, 0, st>>>(a); return true;
    case 4: k_row2<N1, N2, 4><<<blocks, 256, 0, st>>>(a); return true;
    case 8: k_row2<N1, N2, 8><<<blocks, 256, 0, st>>>(a); return true;
    case 16: if constexpr (N2 >= 16) { k_row2<N1, N2, 16><<<blocks, 256, 0, st>>>(a); return true; } break;
  }
  return false;
}

template <int N3>
static bool row3_nz(const RowArgs &a, int nza, cudaStream_t st) {
  const unsigned blocks = (unsigned)a.nrows;
  switch (nza) {
    case 1: k_row3<N3, 1><<<blocks, 256, 0, st>>>(a); return true;
    case 2: k_row3<N3, 2><<<blocks, 256, 0, st>>>(a); return true;
    case 4: if constexpr (N3 >= 4) { k_row3<N3, 4><<<blocks, 256, 0, st>>>(a); return true; } break;
    case 8: if constexpr (N3 >= 8) { k_row3<N3, 8><<<blocks, 256, 0, st>>>(a); return true; } break;
  }
  return false;
}

template <int NF>
static bool rowbig_nz(const RowArgs &a, int nz, cudaStream_t st, bool attr_only) {
  const unsigned blocks = (unsigned)a.nrows;
  const size_t smem = (size_t)(NF + NF / 16) * sizeof(float2);   // padded, RBI in kernels_generic.cuh
#define VOLKS_ROWBIG(NZ_)                                                                                        \
  case NZ_:                                                                                                      \
    if (attr_only) return cudaFuncSetAttribute(k_rowbig<NF, NZ_>, cudaFuncAttributeMaxDynamicSharedMemorySize,   \
                                               (int)smem) == cudaSuccess;                                        \
    k_rowbig<NF, NZ_><<<blocks, NF / 16, smem, st>>>(a);                                                         \
    return true;
  switch (nz) { VOLKS_ROWBIG(1) VOLKS_ROWBIG(2) VOLKS_ROWBIG(4) VOLKS_ROWBIG(8) VOLKS_ROWBIG(16) }
#undef VOLKS_ROWBIG
  return false;
}

// radix-16 row FFT for nf = 4096 / 8192 (k_rowbig); attr_only: raise its dynamic shared memory limit
static bool launch_rowbig(const RowArgs &a, cudaStream_t st, bool attr_only) {
  if (!a.paired || (a.nf != 4096 && a.nf != 8192) || a.nrows >= (1LL << 31)) return false;
  int nz = 1;
  while (nz * (a.nf / 16) < a.nchan) nz *= 2;
  return a.nf == 4096 ? rowbig_nz<4096>(a, nz, st, attr_only) : rowbig_nz<8192>(a, nz, st, attr_only);
}

// register-form row FFT for nf in {64, 128, 256} (k_row2) and {512 .. 2048} (k_row3) with the paired Y
// layout; false = not applicable
static bool launch_row2(const RowArgs &a, cudaStream_t st) {
  if (!a.paired) return false;
  if (a.nf >= 512 && a.nf <= 2048 && a.nrows < (1LL << 31)) {
    int nza = 1;
    while (nza * 256 < a.nchan) nza *= 2;
    switch (a.nf / 256) {
      case 2: return row3_nz<2>(a, nza, st);
      case 4: return row3_nz<4>(a, nza, st);
      case 8: return row3_nz<8>(a, nza, st);
    }
    return false;
  }
  if (a.nf == 128) {           // 16 x 8 with eight lanes per row (k_row128)
    int nza = 1;
    while (nza * 16 < a.nchan) nza *= 2;
    const unsigned blocks = (unsigned)((a.nrows + 32 * ROW128_RB - 1) / (32 * ROW128_RB));
    switch (nza) {
      case 1: k_row128<1><<<blocks, 256, 0, st>>>(a); return true;
      case 2: k_row128<2><<<blocks, 256, 0, st>>>(a); return true;
      case 4: k_row128<4><<<blocks, 256, 0, st>>>(a); return true;
      case 8: k_row128<8><<<blocks, 256, 0, st>>>(a); return true;
    }
    return false;
  }
  int n1, n2;
  if (a.nf == 256) { n1 = 16; n2 = 16; } else if (a.nf == 128) { n1 = 8; n2 = 16; } else if (a.nf == 64) { n1 = 8; n2 = 8; } else return false;
  int nza = 1;
  while (nza * n1 < a.nchan) nza *= 2;                       // leading non-zero inputs of the N2-point transform
  const unsigned blocks = (unsigned)((a.nrows + 256 / n2 - 1) / (256 / n2));
  if (a.nf == 256) return row2_nz<16, 16>(a, nza, blocks, st);
  if (a.nf == 128) return row2_nz<8, 16>(a, nza, blocks, st);
  return row2_nz<8, 8>(a, nza, blocks, st);
}

// fold: the FOLD mode of the kernel (kernels_sfold.cuh; Nt >= 64 only: M >= 4)
static void launch_slide(const SlideArgs &a, cudaStream_t st, bool fold = false) {
  // every warp of a CTA must share its (pair, segment): warps per CTA = min(SLIDE_WARPS, ndt * M)
  const long long per_seg = (long long)a.ndt << a.log2m;
  int wpb = SLIDE_WARPS;                         // the largest power of two <= 8 that divides the warps of a segment
  while (per_seg % wpb) wpb >>= 1;
  const unsigned blocks = (unsigned)(a.ntasks / wpb);
  const int thr = wpb * 32;
  if (a.nt >= 32) {
    // M >= 4: rows travel through a shared-memory ring of (w + 48) x 512 * (column groups) bytes
    const int dtc = std::max(1, wpb >> a.log2m);
    // + the warps' twiddle rows ([wpb][Nt + 1] float4) behind the ring
    const size_t ring = (size_t)(a.w + 48) * 512 * dtc + (size_t)wpb * (a.nt + 1) * 16;
    if (a.log2m >= 2 && ring <= 100 * 1024) {
      if (fold) {
        if (dtc == 1) k_slide<16, false, true, 512, true><<<blocks, thr, ring, st>>>(a);
        else if (dtc == 2) k_slide<16, false, true, 1024, true><<<blocks, thr, ring, st>>>(a);
        else k_slide<16, false, true, 0, true><<<blocks, thr, ring, st>>>(a);
      } else {
        if (dtc == 1) k_slide<16, false, true, 512><<<blocks, thr, ring, st>>>(a);
        else if (dtc == 2) k_slide<16, false, true, 1024><<<blocks, thr, ring, st>>>(a);
        else k_slide<16, false, true><<<blocks, thr, ring, st>>>(a);
      }
    }
    else if (fold) k_slide<16, false, false, 0, true><<<blocks, thr, 0, st>>>(a);
    else k_slide<16, false, false><<<blocks, thr, 0, st>>>(a);
  }
  else if (a.nt == 16) k_slide<16, true, false><<<blocks, thr, 0, st>>>(a);
  else if (a.nt == 8) k_slide<8, true, false><<<blocks, thr, 0, st>>>(a);
  else k_slide<4, true, false><<<blocks, thr, 0, st>>>(a);
}

// the ring kernels' dynamic shared memory limit (per device, process-wide: always the maximum they can need)
static bool slide_attrs() {
  const int lim = 100 * 1024;
  return cudaFuncSetAttribute(k_slide<16, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim) == cudaSuccess &&
         cudaFuncSetAttribute(k_slide<16, false, true, 512>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim) == cudaSuccess &&
         cudaFuncSetAttribute(k_slide<16, false, true, 1024>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim) == cudaSuccess &&
         cudaFuncSetAttribute(k_slide<16, false, true, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim) == cudaSuccess &&
         cudaFuncSetAttribute(k_slide<16, false, true, 512, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim) == cudaSuccess &&
         cudaFuncSetAttribute(k_slide<16, false, true, 1024, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim) == cudaSuccess;
}

// k_bound's dynamic shared memory limit (per device, process-wide)
constexpr size_t PRUNE_SMEM_LIMIT = 96 * 1024;
template <int NQ>
static bool bound_attr() {
  return cudaFuncSetAttribute(k_bound<NQ, 0, 64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PRUNE_SMEM_LIMIT) == cudaSuccess &&
         cudaFuncSetAttribute(k_bound<NQ, 1, 64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PRUNE_SMEM_LIMIT) == cudaSuccess &&
         cudaFuncSetAttribute(k_bound<NQ, 0, 128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PRUNE_SMEM_LIMIT) == cudaSuccess &&
         cudaFuncSetAttribute(k_bound<NQ, 1, 128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PRUNE_SMEM_LIMIT) == cudaSuccess;
}
static bool bound_attrs() {
  return cudaFuncSetAttribute(k_pairfold, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pairfold_smem_bytes()) == cudaSuccess &&
         bound_attr<1>() && bound_attr<2>() && bound_attr<3>() && bound_attr<4>() && bound_attr<5>() && bound_attr<6>() &&
         bound_attr<7>() && bound_attr<8>();
}

}  // namespace

struct volks_plan {
  Sched sched;                 // host copy
  Sched *d_sched = nullptr;    // device copy
  std::vector<WidthPlan> wp;
  float2 *d_tables = nullptr;  // [nf] delay twiddles, then per width [nt] rate twiddles
  int nchan = 0, pitch = 0;
  int paired = 0;               // Y rows pair-interleaved (common.cuh ld_y)
  mutable cudaStream_t copy_stream = nullptr;      // volks_search_host: H2D copies of the slab chunks
  mutable cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_free[2] = {nullptr, nullptr};
  mutable const float2 *d_cal = nullptr;   // volks_plan_set_cal: DEVICE cf32[nbl][nif][nchan] applied in the slab load
  int nslide = 0;                // widths on the sliding-sum path (k_fixup re-evaluates their outlier windows)
  volks_options opt;             // the options the plan was created with (defaults: volks_options_init)
  int nuntag = 0;                // sliding widths with untagged kernels (their peak bins come from k_recover)
  bool cand_only = false;        // searches without d_peaks recover indices / evaluate segments for possible candidates only
  int nprune = 0, prune_nseg = 0, prune_seg = 0, prune_wmax = 0;   // pruned widths (k_bound): count, common segmentation
  int nsf = 0;                   // widths on the folded-sum path in the candidates-only mode (kernels_sfold.cuh)
  bool cw_pf = false;            // the column-level width is w = 32 at Nt = 64: its bits come from k_pairfold (folded bound), not k_bound
  int cwq = -1, cw_nwords = 0;   // the column-level width (index into wp) and the 32-window words of its bit mask per pair
  size_t off_cwmask = 0, off_cwdense = 0;
  int dt_n = 0, dt_na = 0, dt_a0 = 0, dt_b0 = 0;   // 64-column groups the sliding kernels / k_bound work on (restricted delay range)
  size_t off_flags = 0;          // their segment flags [pairs_per_chunk][nprune][prune_nseg]
  size_t off_thr = 0;            // their windows' pre-thresholds (k_winthr), chunk-relative
  mutable bool last_full_index = true;   // the most recent search left exact indices for EVERY window (volks_zscore_select)
  int device = 0;                // the CUDA device the plan was created on
  int cf_split2 = 2;             // opt.cf2: k_colfft2 (two columns per thread, split format) for Nt = 256 / 512
  int ai_psub = 1;               // f2 with nfa > 8192: nfa = ai_psub * row_nf (virtual sub-rows, kernels_generic.cuh)
  int row_nf = 0;                // size of the row transform (= sched.nf unless ai_psub > 1)
  size_t premod_off = 0;         // offset (float2) of the W_nfa table in d_tables
  int ai_nif = 0, ai_nchan = 0; // f2 all-IF plan: source nif / nchan (0 = ordinary per-IF plan)
  size_t off_noise = 0;         // f2: per-window noise written by k_allif
  bool row_generic = false;     // VOLKS_PATH=generic: the shared-memory Stockham row kernel only
  int wid1 = -1;                // a width with w == 1 whose peaks the row kernel emits itself (or -1)
  long long npair = 0;
  // workspace layout (byte offsets)
  size_t off_keys = 0, off_E = 0, off_cnt = 0, off_zst = 0, off_Y = 0, ws_bytes = 0;
  long long nfin_blocks = 0;
  long long pairs_per_chunk = 0, nchunks = 0;
  int host_split = 4;            // volks_search_host: copies (and kernel chunks) of pairs_per_chunk / host_split pairs
  // row kernel shape
  int row_tpr = 1, row_rows_per_cta = 1;
  size_t row_smem = 0;
  int launches = 0;
  // optional per-launch timing (volks_plan_profile): events recorded on the launching stream
  mutable bool prof_on = false;
  mutable std::vector<cudaEvent_t> prof_ev;      // 2 per launch (begin, end), grown on demand
  mutable std::vector<int> prof_kind, prof_wid;  // of the most recent volks_fringe_search
};

namespace {
// Brackets one kernel launch with events when profiling is enabled (no-op otherwise).
struct ProfScope {
  const volks_plan *pl; cudaStream_t st; size_t slot;
  ProfScope(const volks_plan *p, cudaStream_t s, int kind, int wid) : pl(p), st(s), slot(0) {
    if (!pl->prof_on) return;
    slot = pl->prof_kind.size();
    pl->prof_kind.push_back(kind); pl->prof_wid.push_back(wid);
    while (pl->prof_ev.size() < 2 * (slot + 1)) { cudaEvent_t e; cudaEventCreate(&e); pl->prof_ev.push_back(e); }
    cudaEventRecord(pl->prof_ev[2 * slot], st);
  }
  ~ProfScope() { if (pl->prof_on) cudaEventRecord(pl->prof_ev[2 * slot + 1], st); }
};
}  // namespace

extern "C" {

int volks_version(void) { return 100; }

const char *volks_strerror(int code) {
  switch (code) {
    case VOLKS_OK: return "ok";
    case VOLKS_EINVAL: return "invalid argument";
    case VOLKS_ECUDA: return g_cuda_msg[0] ? g_cuda_msg : "CUDA error";
    case VOLKS_ENOMEM: return "out of host memory";
    case VOLKS_EOVERFLOW: return "output capacity exceeded";
    case VOLKS_ELIMIT: return "problem larger than the static scratch of volks_search_noalloc (VOLKS_NOALLOC_SCRATCH_BYTES)";
    default: return "unknown error";
  }
}

static int plan_create_impl(const volks_params *p, const volks_options *o, volks_plan **out, int ai_nif, int ai_nchan, int psub = 1);

void volks_options_init(volks_options *o) {
  if (!o) return;
  memset(o, 0, sizeof *o);
  o->struct_bytes = (int32_t)sizeof(volks_options);
  o->slide_seg = 256; o->y_pad = 16; o->chunk_mb = 4096; o->cf_wpc = 128; o->cf2 = 2; o->ai_waves = 2; o->host_split = 4;
  o->prune_seg = 64;
  o->delay_lo = 0; o->delay_hi = -1;      // the whole delay axis
}

int volks_plan_create(const volks_params *p, volks_plan **out) { return plan_create_impl(p, nullptr, out, 0, 0); }
int volks_plan_create_opt(const volks_params *p, const volks_options *o, volks_plan **out) { return plan_create_impl(p, o, out, 0, 0); }
int volks_plan_create_allif(const volks_params *p, volks_plan **out) { return volks_plan_create_allif_opt(p, nullptr, out); }

int volks_plan_create_allif_opt(const volks_params *p, const volks_options *o, volks_plan **out) {
  if (!p || !out) return VOLKS_EINVAL;
  *out = nullptr;
  if (p->nbl < 1 || p->nif < 1 || p->nchan < 1 || p->nwidths < 1 || p->nwidths > VOLKS_MAX_WIDTHS) return VOLKS_EINVAL;
  if ((long long)p->nif * p->nchan > p->nf || p->nf < 64 || p->nf > 32768 || !is_pow2(p->nf)) return VOLKS_EINVAL;
  if ((long long)p->nif * p->nchan > 8192) return VOLKS_EINVAL;      // the band must fit one 8192-point row transform
  int32_t ones[VOLKS_MAX_WIDTHS];
  for (int q = 0; q < VOLKS_MAX_WIDTHS; ++q) ones[q] = 1;
  volks_params b = *p;          // the band of one (bl, AP) as a single "IF" of nif * nchan points; no rate axis
  b.nif = 1; b.nchan = p->nif * p->nchan; b.nt = ones;
  // nfa > 8192 (EL060: 8 IF x 1024 x pad 4 = 32768): psub interleaved 8192-point transforms per AP
  const int psub = p->nf > 8192 ? p->nf / 8192 : 1;
  b.nf = p->nf / psub;
  return plan_create_impl(&b, o, out, p->nif, p->nchan, psub);
}

static int plan_create_impl(const volks_params *p, const volks_options *o, volks_plan **out, int ai_nif, int ai_nchan, int psub) {
  if (!p || !out) return VOLKS_EINVAL;
  *out = nullptr;
  volks_options opt;
  volks_options_init(&opt);
  if (o) {
    if (o->struct_bytes != (int32_t)sizeof(volks_options)) return VOLKS_EINVAL;   // built against another header
    opt = *o;
    if (opt.slide_seg < 16 || opt.y_pad < 0 || opt.y_pad > 1024 || (opt.y_pad & 1) || opt.chunk_mb < 1 || opt.cf_wpc < 1 ||
        (opt.cf2 != 0 && opt.cf2 != 1 && opt.cf2 != 2 && opt.cf2 != 4) || opt.ai_waves < 1 || opt.host_split < 1 ||
        opt.prune_seg < 16 || opt.prune_seg > 4096 || !is_pow2(opt.prune_seg))
      return VOLKS_EINVAL;
    // a restricted delay range is given in bins of the padded delay axis the caller asked for (nf, or nfa for f2)
    if (opt.delay_hi >= 0 && (opt.delay_lo < 0 || opt.delay_lo >= p->nf * psub || opt.delay_hi >= p->nf * psub)) return VOLKS_EINVAL;
    if (opt.delay_hi < -1) return VOLKS_EINVAL;
  }
  const bool allif = ai_nif > 0;
  if (p->nbl < 1 || p->nif < 1 || p->nap < 0 || p->nchan < 1) return VOLKS_EINVAL;
  if (p->nwidths < 1 || p->nwidths > VOLKS_MAX_WIDTHS || !p->width || !p->stride || !p->nt) return VOLKS_EINVAL;
  if (!is_pow2(p->nf) || p->nf < p->nchan || p->nf > 8192) return VOLKS_EINVAL;   // row transforms up to 8192 points
  if (!(p->snr_thresh == p->snr_thresh)) return VOLKS_EINVAL;
  for (int q = 0; q < p->nwidths; ++q) {
    if (p->width[q] < 1 || p->stride[q] < 1 || !is_pow2(p->nt[q]) || (!allif && p->nt[q] < p->width[q])) return VOLKS_EINVAL;
    if ((long long)p->nt[q] * p->nf > (1LL << 31)) return VOLKS_EINVAL;   // plane index must fit 32 bits
  }
  volks_plan *pl = new (std::nothrow) volks_plan();
  if (!pl) return VOLKS_ENOMEM;
  Sched &s = pl->sched;
  memset(&s, 0, sizeof s);
  s.nwidths = p->nwidths; s.nbl = p->nbl; s.nif = p->nif; s.nap = p->nap; s.nf = p->nf * psub;
  s.log2nf = ilog2(s.nf); s.snr_thresh = p->snr_thresh;
  if (opt.delay_hi >= 0 && !(opt.delay_lo == 0 && opt.delay_hi == s.nf - 1)) {
    s.dlo = opt.delay_lo; s.dhi = opt.delay_hi;
    s.dfirst = s.dlo <= s.dhi ? s.dlo : 0;       // a wrapping range contains bin 0
  } else { s.dlo = -1; s.dhi = -1; s.dfirst = 0; }
  {
    // 64-column groups that hold searched bins, as at most two pieces (a wrapping range: the low bins, then the high
    // ones), each widened to an even group boundary so that the two-group CTAs of k_slide read contiguous columns
    const int ng = std::max(1, s.nf / 64);
    pl->dt_n = ng; pl->dt_na = ng; pl->dt_a0 = 0; pl->dt_b0 = 0;
    if (s.dlo >= 0 && ng >= 2 && !allif) {
      auto lo2 = [](int g) { return g & ~1; };
      auto hi2 = [&](int g) { return std::min(ng, (g + 2) & ~1); };     // exclusive, even
      if (s.dlo <= s.dhi) { pl->dt_a0 = lo2(s.dlo / 64); pl->dt_na = hi2(s.dhi / 64) - pl->dt_a0; pl->dt_n = pl->dt_na; }
      else {
        const int a1 = hi2(s.dhi / 64), b0 = lo2(s.dlo / 64);            // [0, a1) and [b0, ng)
        if (a1 >= b0) { pl->dt_a0 = 0; pl->dt_na = ng; pl->dt_n = ng; }
        else { pl->dt_a0 = 0; pl->dt_na = a1; pl->dt_b0 = b0; pl->dt_n = a1 + (ng - b0); }
      }
    }
  }
  pl->ai_psub = psub; pl->row_nf = p->nf;
  pl->nchan = p->nchan;
  pl->npair = (long long)p->nbl * p->nif;
  pl->ai_nif = ai_nif; pl->ai_nchan = ai_nchan; s.allif = allif ? 1 : 0;
  // k_allif: one CTA per sub-row of 8192 delay columns (CP = 4 pairs per thread, no spills); measured on config 5
  // (nfa 32768): 4096 -> 8.1 ms per width, 8192 -> 7.0, 16384 -> 7.0-7.7, one CTA (CP = 16, spills) 15-16
  s.ngs = allif ? psub : 1;
  long long per_pair = 0;
  size_t tw_total = (size_t)p->nf;
  pl->opt = opt;
  if (!cuda_ok(cudaGetDevice(&pl->device))) { delete pl; return VOLKS_ECUDA; }
  const bool force_generic = opt.force_generic != 0;
  const int seg_req = std::max(16, opt.slide_seg);
  pl->cf_split2 = opt.cf2;   // 2: 16-column strips (two 256-thread CTAs per SM), 1: 32-column strips, 0: k_colfft (nf >= 32 there: Y rows are pair-interleaved)
  for (int q = 0; q < p->nwidths; ++q) {
    WidthPlan w;
    w.w = p->width[q]; w.s = p->stride[q]; w.nt = p->nt[q];
    w.nwin = p->nap < w.w ? 0 : (long long)(p->nap - w.w) / w.s + 1;
    w.L = std::min(16, w.nt);
    w.log2m = ilog2(w.nt / w.L);
    // sliding-sum path: stride 1, pad x2 in time, whole warps of delay columns, 32-bit row offsets
    w.slide = !force_generic && w.s == 1 && w.w >= 2 && w.nt == 2 * w.w && p->nf >= 64 &&
              ((long long)p->nap + SLIDE_PF + 2) * (p->nf + 64) * 8 < (1LL << 32);
    if (allif) w.slide = false;
    w.untag = w.slide && w.nt >= 32;     // (+ the k_colfft2 widths, set below once colfft is known)
    w.colfft = !allif && !force_generic && !w.slide && w.nt >= 32 && w.nt <= 512 && p->nf >= 32 && w.nwin > 0;
    // exact pruning by the amplitude-sum bound (kernels_prune.cuh): narrow widths whose noise-only bound stays
    // >= 4.5 deviations below the threshold, (0.99 snr_thresh - 0.886 sqrt(w)) / 0.4637 (Rayleigh amplitudes)
    w.prune = -1;
    if (w.slide && !opt.full_index && !opt.no_prune && p->snr_thresh > 0.f && w.w <= PRUNE_RING &&
        pl->nprune + (pl->cwq >= 0 ? 1 : 0) < PRUNE_MAXQ &&
        p->nap >= w.w && (0.99 * p->snr_thresh - 0.886 * sqrt((double)w.w)) / 0.4637 >= 4.5 && w.nt <= opt.prune_seg)
      w.prune = pl->nprune++;
    // column-level pruning (kernels_coleval.cuh) for ONE width whose bound is too weak for whole segments but leaves
    // few delay columns per window: >= 1.5 deviations (<= 7 % of the columns pass on noise); w = 32 at snr_thresh 6
    w.cw = false;
    if (w.prune < 0 && pl->cwq < 0 && w.slide && w.nt >= 32 && !opt.full_index && !opt.no_prune && p->snr_thresh > 0.f &&
        w.w <= PRUNE_RING && pl->nprune < PRUNE_MAXQ && p->nap >= w.w && w.nt <= 2 * PRUNE_RING && opt.prune_seg == 64 &&
        (0.99 * p->snr_thresh - 0.886 * sqrt((double)w.w)) / 0.4637 >= 1.5) { w.cw = true; pl->cwq = q; }
    // folded sliding sum (kernels_sfold.cuh) for the wide stride-1 widths in the candidates-only mode: pays when noise
    // stays below the Cauchy-Schwarz bound's test, 16 x Gamma(16): (0.98 snr_thresh^2 / 16 - 1) / 0.25 >= 4 deviations
    w.sf = w.slide && w.nt >= 64 && w.prune < 0 && !w.cw && !opt.full_index && !opt.no_prune && p->snr_thresh > 0.f &&
           (0.98 * p->snr_thresh * p->snr_thresh / 16.0 - 1.0) / 0.25 >= 4.0;
    w.off_hits = 0; w.nblk = (int)((w.nwin + 15) / 16);
    w.cf_l1 = w.nt / 16;
    if (w.colfft && w.nt >= 256 && opt.cf2 != 0) w.untag = true;   // k_colfft2 keeps no bin tags either
    w.cf_nz = 1;
    while (w.cf_nz * 16 < w.w) w.cf_nz *= 2;
    // windows per CTA: up to 128 (L1 reuse of overlapping windows), fewer when the grid would not fill 148 SMs x 4
    w.cf_wpc = (int)std::min<long long>(opt.cf_wpc,
                                        std::max<long long>(8, (long long)p->nbl * p->nif * (p->nf / 32) * w.nwin / 592));
    w.cf_nrange = (int)((w.nwin + w.cf_wpc - 1) / w.cf_wpc);
    w.seg = std::max((seg_req / w.nt) * w.nt, w.nt);
    if (w.prune >= 0) w.seg = opt.prune_seg;      // one segmentation for every pruned width (a multiple of its Nt)
    if (w.cw) w.seg = CE_TILE;                    // the column-level width: segments = k_coleval's / k_bound's tiles of 128
    // f2: one CTA per (baseline, segment): segments short enough to fill 148 SMs x 2, at most seg_req windows
    if (allif) w.seg = (int)std::max<long long>(16, std::min<long long>((seg_req / 16) * 16, (w.nwin * p->nbl / 296 + 15) / 16 * 16));
    w.nseg = w.nwin > 0 ? (int)((w.nwin + w.seg - 1) / w.seg) : 0;
    w.tw_off = tw_total;
    tw_total += (size_t)w.nt;
    tw_total += tw_total & 1;          // 16-byte alignment of the float4 copy
    w.tw4_off = tw_total;
    tw_total += (size_t)2 * w.nt;
    s.width[q] = w.w; s.stride[q] = w.s; s.nt[q] = w.nt; s.nwin[q] = w.nwin; s.offc[q] = per_pair;
    per_pair += w.nwin;
    pl->wp.push_back(w);
  }
  s.per_pair = per_pair;
  s.nwin_total = per_pair * pl->npair;
  long long acc = 0;
  for (int q = 0; q < p->nwidths; ++q) { s.offd[q] = acc; acc += pl->npair * s.nwin[q]; }
  if (s.nwin_total >= (1LL << 40)) { delete pl; return VOLKS_EINVAL; }

  // row kernel shape: nf/4 threads per row (at least 1, at most 512), ~256 threads per CTA
  // one warp per row up to nf = 512 (warp barriers only); wider rows take nf/4 threads and a whole CTA
  pl->row_tpr = p->nf <= 512 ? std::max(1, std::min(32, p->nf / 4)) : std::min(512, p->nf / 4);
  pl->row_rows_per_cta = std::max(1, 256 / pl->row_tpr);
  pl->row_smem = (size_t)2 * pl->row_rows_per_cta * p->nf * sizeof(float2) + (size_t)pl->row_rows_per_cta * 16 * sizeof(u64);
  if (pl->row_smem > 200 * 1024) { delete pl; return VOLKS_EINVAL; }

  // chunking of the delay-spectrum intermediate Y over (bl, ifq) pairs: <= 4 GiB per chunk
  // Y row pitch: nf + 16 elements (one 128-byte line) when rows would otherwise sit a power of two
  // apart and fall into the same few L1 sets (kernels_slide.cuh reads w+1 rows of a column tile)
  pl->pitch = (p->nf >= 32 && psub == 1) ? p->nf + opt.y_pad : p->nf;   // sub-rows are contiguous
  pl->paired = p->nf >= 2 ? 1 : 0;
  pl->row_generic = force_generic;
  const size_t y_pair = (size_t)p->nap * psub * pl->pitch * sizeof(float2);
  // VOLKS_CHUNK_MB: bytes of delay spectra per chunk of pairs (default 4 GiB; tests use small chunks)
  const size_t budget = (size_t)opt.chunk_mb << 20;
  long long ppc = y_pair ? (long long)std::max<size_t>(1, budget / std::max<size_t>(y_pair, 1)) : pl->npair;
  ppc = std::min(ppc, pl->npair);
  pl->nchunks = (pl->npair + ppc - 1) / ppc;
  pl->pairs_per_chunk = (pl->npair + pl->nchunks - 1) / pl->nchunks;
  pl->nchunks = (pl->npair + pl->pairs_per_chunk - 1) / pl->pairs_per_chunk;
  pl->host_split = opt.host_split;
  if (allif) {
    // k_allif launches pairs_per_chunk x psub x nseg CTAs of up to 1024 threads (two per SM): size the
    // segments of windows for about VOLKS_AI_WAVES (default 2) waves of 296 CTAs (restart cost per segment: w rows;
    // measured at the paper's size: 1 wave 41.5 ms per trial, 2 waves 38.1, 4 waves 38.7, 8 waves 39.7)
    const long long waves = opt.ai_waves;
    for (auto &w : pl->wp) {
      if (w.nwin <= 0) continue;
      const long long want = std::max<long long>(1, (296 * waves + pl->pairs_per_chunk * psub - 1) / (pl->pairs_per_chunk * psub));
      long long seg = ((w.nwin + want - 1) / want + 15) / 16 * 16;
      seg = std::max<long long>(seg, 16);
      w.seg = (int)seg;
      w.nseg = (int)((w.nwin + seg - 1) / seg);
    }
  }

  pl->nfin_blocks = (s.nwin_total + FIN_THREADS * FIN_TILES - 1) / (FIN_THREADS * FIN_TILES);
  {
    // every grid of a search must fit the 2^31 - 1 limit of gridDim.x (the launches cast to unsigned)
    const long long GMAX = (1LL << 31) - 1, ppc_ = pl->pairs_per_chunk;
    bool fits = pl->nfin_blocks <= GMAX && ppc_ * p->nap * psub <= GMAX;
    for (auto &w : pl->wp) {
      if (w.nwin == 0) continue;
      const long double col_blocks = ((long double)ppc_ * w.nwin * (1 << w.log2m) * p->nf * psub + 255) / 256;
      const long double slide_blocks = (long double)ppc_ * w.nseg * std::max(1, p->nf / 64) * (1 << w.log2m);
      const long double cf_blocks = (long double)ppc_ * std::max(1, p->nf / 32) * w.cf_nrange * 4;
      const long double ai_blocks = (long double)ppc_ * w.nseg * psub;
      if ((!w.slide && !w.colfft && !allif && col_blocks > GMAX) || (w.slide && slide_blocks > GMAX) ||
          (w.colfft && cf_blocks > GMAX) || (allif && ai_blocks > GMAX)) fits = false;
    }
    for (auto &w : pl->wp)     // k_sfold_eval: one warp per (block of 16 windows, 64-column group, rate residue)
      if (w.sf && (long double)ppc_ * w.nblk * std::max(1, p->nf / 64) * (1 << w.log2m) > GMAX) fits = false;
    long long rec_warps = 0;
    for (auto &w : pl->wp) rec_warps += w.untag ? w.nwin : 0;
    if ((long double)ppc_ * rec_warps / 128 > GMAX) fits = false;    // k_recover: one thread per window
    if (!fits) { delete pl; return VOLKS_EINVAL; }
  }
  size_t off = 0;
  pl->off_keys = off; off = align_up(off + (size_t)std::max<long long>(s.nwin_total, 1) * sizeof(u64), 256);
  pl->off_E = off;    off = align_up(off + (size_t)std::max<long long>(pl->npair * p->nap, 1) * sizeof(float), 256);
  pl->off_cnt = off;  off = align_up(off + (size_t)std::max<long long>(pl->nfin_blocks, 1) * sizeof(uint32_t), 256);
  // + padding rows: the sliding kernel loads one row, and prefetches SLIDE_PF + 1 rows, past the last sample
  pl->off_noise = off; off = align_up(off + (allif ? (size_t)std::max<long long>(s.nwin_total, 1) * s.ngs * sizeof(float) : 0), 256);
  pl->off_zst = off;  off = align_up(off + (size_t)std::max<long long>(pl->npair * p->nwidths, 1) * sizeof(double2), 256);
  // candidates-only mode (volks_options.full_index = 0, a positive threshold): a search without d_peaks finds the
  // peak bin only of windows above their pre-threshold and prunes the narrow widths (kernels_prune.cuh)
  pl->cand_only = !opt.full_index && p->snr_thresh > 0.f;
  for (auto &w : pl->wp) {
    pl->nuntag += (w.untag && w.nwin > 0) ? 1 : 0;
    if (w.prune >= 0 || w.cw) {
      pl->prune_nseg = std::max(pl->prune_nseg, (int)((w.nwin + opt.prune_seg - 1) / opt.prune_seg));
      pl->prune_wmax = std::max(pl->prune_wmax, w.w);
    }
  }
  pl->prune_seg = opt.prune_seg;
  // k_bound's shared memory (thresholds of a tile of 2 prune_seg windows per width + the ring + the staged rows)
  if ((pl->nprune || pl->cwq >= 0) && prune_smem_bytes(pl->nprune + 1, opt.prune_seg, PRUNE_RING, PRUNE_THREADS) > PRUNE_SMEM_LIMIT) {
    delete pl;
    return VOLKS_EINVAL;
  }
  pl->off_thr = off;  off = align_up(off + ((pl->cand_only && (pl->nuntag || pl->nprune)) ? (size_t)pl->pairs_per_chunk * per_pair * sizeof(uint32_t) : 0), 256);
  pl->off_flags = off; off = align_up(off + (size_t)pl->pairs_per_chunk * (pl->nprune + 1) * pl->prune_nseg, 256);
  // the column-level width's bits: k_bound's tiles are 2 prune_seg windows, a multiple of 32
  pl->cw_pf = pl->cwq >= 0 && pl->wp[pl->cwq].w == PF_W && pl->wp[pl->cwq].nt == 2 * PF_W && opt.prune_seg == 64;
  pl->cw_nwords = pl->cwq >= 0 ? (int)(((pl->prune_nseg + 1) / 2) * (2 * opt.prune_seg / 32)) : 0;
  // (twice: the density bytes, then one byte per tile "no bit set" for k_coleval)
  pl->off_cwdense = off; off = align_up(off + 2 * (size_t)pl->pairs_per_chunk * ((pl->prune_nseg + 1) / 2) + 1, 256);
  pl->off_cwmask = off; off = align_up(off + (size_t)pl->pairs_per_chunk * pl->cw_nwords * p->nf * sizeof(uint32_t), 256);
  for (auto &w : pl->wp) {      // hit masks of the folded-sum widths: [pairs of the chunk][nblk][64-column groups][M] u16
    if (!w.sf || w.nwin == 0) { w.sf = false; continue; }
    pl->nsf += 1;
    w.off_hits = off;
    off = align_up(off + (size_t)pl->pairs_per_chunk * w.nblk * pl->dt_n * (1 << w.log2m) * sizeof(unsigned short), 256);
    w.off_sfdense = off;
    off = align_up(off + (size_t)pl->pairs_per_chunk * w.nseg, 256);
    w.off_sfbig = off;
    off = align_up(off + (size_t)pl->pairs_per_chunk * w.nblk * sizeof(unsigned short), 256);
    w.off_sflist = off;
    off = align_up(off + (1 + (size_t)pl->pairs_per_chunk * w.nblk * pl->dt_n * (1 << w.log2m)) * sizeof(uint32_t), 256);
  }
  pl->off_Y = off;    off = align_up(off + (size_t)pl->pairs_per_chunk * std::max<size_t>(y_pair, 8) + (size_t)(SLIDE_PF + 2) * pl->pitch * sizeof(float2), 256);
  pl->ws_bytes = off;

  int active = 0;
  for (auto &w : pl->wp) pl->nslide += (w.slide && w.nwin > 0) ? 1 : 0;
  if (!force_generic && !allif)
    for (int q = 0; q < p->nwidths && pl->wid1 < 0; ++q)
      if (pl->wp[q].w == 1 && pl->wp[q].nwin > 0) pl->wid1 = q;
  for (int q = 0; q < p->nwidths; ++q) active += (pl->wp[q].nwin > 0 && q != pl->wid1) ? 1 : 0;
  // kernels of this library per search (the key memset is a driver memset, not counted)
  // (a search without dense peaks; with them the candidates-only index mode and its k_winthr launch are off)
  pl->launches = s.nwin_total > 0 ? (int)(pl->nchunks * (1 + active + (pl->nslide > 0 ? 1 : 0) + ((pl->cand_only && (pl->nuntag || pl->nprune)) ? 1 : 0) + ((pl->nprune || (pl->cwq >= 0 && !pl->cw_pf)) ? 1 : 0) + (pl->cw_pf ? 1 : 0) + (pl->nuntag ? 1 : 0) + (pl->cwq >= 0 ? 1 : 0) + 5 * pl->nsf) + 3) : 0;

  // tables, computed in double precision on the host
  if (psub > 1) { pl->premod_off = tw_total; tw_total += (size_t)s.nf; }
  std::vector<float2> tab(tw_total);
  for (int k = 0; psub > 1 && k < s.nf; ++k) {
    const double a = -2.0 * 3.14159265358979323846264338327950288 * k / s.nf;
    tab[pl->premod_off + k] = make_float2((float)cos(a), (float)sin(a));
  }
  const double PI = 3.14159265358979323846264338327950288;
  for (int k = 0; k < p->nf; ++k) {
    const double a = -2.0 * PI * k / p->nf;
    tab[k] = make_float2((float)cos(a), (float)sin(a));
  }
  for (auto &w : pl->wp)
    for (int k = 0; k < w.nt; ++k) {
      const double a = -2.0 * PI * k / w.nt;
      tab[w.tw_off + k] = make_float2((float)cos(a), (float)sin(a));
      tab[w.tw4_off + 2 * k] = make_float2((float)cos(a), (float)cos(a));
      tab[w.tw4_off + 2 * k + 1] = make_float2((float)sin(a), (float)sin(a));
    }
  bool ok = cuda_ok(cudaMalloc(&pl->d_tables, tw_total * sizeof(float2))) &&
            cuda_ok(cudaMalloc(&pl->d_sched, sizeof(Sched))) &&
            cuda_ok(cudaMemcpy(pl->d_tables, tab.data(), tw_total * sizeof(float2), cudaMemcpyHostToDevice)) &&
            cuda_ok(cudaMemcpy(pl->d_sched, &s, sizeof(Sched), cudaMemcpyHostToDevice));
  // kernel attributes are process-wide per device: every kernel gets the MAXIMUM it can ever need (never a
  // plan-dependent value, so that a later plan cannot lower an earlier one's limit)
  ok = ok && cuda_ok(cudaFuncSetAttribute(k_row_fft, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
  for (auto &w : pl->wp)
    if (ok && w.colfft) {
      ColFftArgs ca; memset(&ca, 0, sizeof ca); ca.nt = w.nt;
      ok = cuda_ok(launch_colfft(ca, w.cf_l1, w.cf_nz, 0, nullptr, true));
    }
  if (ok && !slide_attrs()) ok = cuda_ok(cudaGetLastError()) && false;
  if (ok && !bound_attrs()) ok = cuda_ok(cudaGetLastError()) && false;
  if (ok && (p->nf == 4096 || p->nf == 8192)) {
    RowArgs ra; memset(&ra, 0, sizeof ra);
    ra.paired = pl->paired; ra.nf = p->nf; ra.nchan = p->nchan; ra.nrows = 1;
    if (!launch_rowbig(ra, nullptr, true)) { cuda_ok(cudaGetLastError()); snprintf(g_cuda_msg, sizeof g_cuda_msg, "k_rowbig: shared memory attribute refused"); ok = false; }
  }
  if (!ok) { volks_plan_destroy(pl); return VOLKS_ECUDA; }
  *out = pl;
  return VOLKS_OK;
}

int volks_plan_destroy(volks_plan *pl) {
  if (!pl) return VOLKS_EINVAL;
  if (pl->d_tables) cudaFree(pl->d_tables);
  if (pl->d_sched) cudaFree(pl->d_sched);
  for (cudaEvent_t e : pl->prof_ev) cudaEventDestroy(e);
  for (int k = 0; k < 2; ++k) { if (pl->ev_copied[k]) cudaEventDestroy(pl->ev_copied[k]); if (pl->ev_free[k]) cudaEventDestroy(pl->ev_free[k]); }
  if (pl->copy_stream) cudaStreamDestroy(pl->copy_stream);
  delete pl;
  return VOLKS_OK;
}

int volks_plan_query(const volks_plan *pl, size_t *workspace_bytes, int64_t *nwin_per_width, int64_t *nwin_total) {
  if (!pl) return VOLKS_EINVAL;
  if (workspace_bytes) *workspace_bytes = pl->ws_bytes;
  if (nwin_per_width) for (int q = 0; q < pl->sched.nwidths; ++q) nwin_per_width[q] = pl->sched.nwin[q];
  if (nwin_total) *nwin_total = pl->sched.nwin_total;
  return VOLKS_OK;
}

int volks_plan_launch_count(const volks_plan *pl) { return pl ? pl->launches : VOLKS_EINVAL; }

int volks_fringe_search(const volks_plan *pl, const void *d_vis, void *d_workspace, volks_peak *d_peaks,
                        volks_cand *d_cands, uint32_t cand_capacity, uint32_t *d_ncand, void *cuda_stream) {
  return volks_fringe_search_dd(pl, d_vis, nullptr, d_workspace, d_peaks, d_cands, cand_capacity, d_ncand, cuda_stream);
}

static int run_search(const volks_plan *pl, const void *vis, void *d_stage, const int32_t *d_shift, void *d_workspace,
                      volks_peak *d_peaks, volks_cand *d_cands, uint32_t cand_capacity, uint32_t *d_ncand,
                      void *cuda_stream);

int volks_fringe_search_dd(const volks_plan *pl, const void *d_vis, const int32_t *d_shift, void *d_workspace,
                           volks_peak *d_peaks, volks_cand *d_cands, uint32_t cand_capacity, uint32_t *d_ncand,
                           void *cuda_stream) {
  if (pl && pl->ai_nif) return VOLKS_EINVAL;     // an all-IF plan: use volks_allif_search
  return run_search(pl, d_vis, nullptr, d_shift, d_workspace, d_peaks, d_cands, cand_capacity, d_ncand, cuda_stream);
}

int volks_allif_search(const volks_plan *pl, const void *d_vis, const int32_t *d_shift, void *d_workspace,
                       volks_peak *d_peaks, volks_cand *d_cands, uint32_t cand_capacity, uint32_t *d_ncand,
                       void *cuda_stream) {
  if (!pl || !pl->ai_nif) return VOLKS_EINVAL;   // needs a plan from volks_plan_create_allif
  return run_search(pl, d_vis, nullptr, d_shift, d_workspace, d_peaks, d_cands, cand_capacity, d_ncand, cuda_stream);
}

int volks_plan_set_cal(volks_plan *pl, const void *d_cal) {
  if (!pl) return VOLKS_EINVAL;
  pl->d_cal = (const float2 *)d_cal;
  return VOLKS_OK;
}

int volks_cal_phasors(const double *delay_s, const double *phase_rad, int32_t npair, int32_t nchan, double chan_hz,
                      float *cal) {
  if (!delay_s || !phase_rad || !cal || npair < 0 || nchan < 1 || !(chan_hz > 0)) return VOLKS_EINVAL;
  const double TWO_PI = 6.28318530717958647692528676655900577;
  for (int32_t p = 0; p < npair; ++p)
    for (int32_t j = 0; j < nchan; ++j) {
      const double ph = -(TWO_PI * (j * chan_hz) * delay_s[p] + phase_rad[p]);
      cal[2 * ((size_t)p * nchan + j)] = (float)cos(ph);
      cal[2 * ((size_t)p * nchan + j) + 1] = (float)sin(ph);
    }
  return VOLKS_OK;
}

int volks_plan_query_host(const volks_plan *pl, size_t *stage_bytes) {
  if (!pl || !stage_bytes) return VOLKS_EINVAL;
  const long long ppc = std::max<long long>(1, (pl->pairs_per_chunk + pl->host_split - 1) / pl->host_split);   // run_search's host chunk
  *stage_bytes = align_up((size_t)ppc * pl->sched.nap * pl->nchan * sizeof(float2), 256);
  return VOLKS_OK;
}

int volks_search_host(const volks_plan *pl, const void *h_vis, void *d_stage, const int32_t *d_shift,
                      void *d_workspace, volks_peak *d_peaks, volks_cand *d_cands, uint32_t cand_capacity,
                      uint32_t *d_ncand, void *cuda_stream) {
  if (!pl || !h_vis || !d_stage) return VOLKS_EINVAL;
  return run_search(pl, h_vis, d_stage, d_shift, d_workspace, d_peaks, d_cands, cand_capacity, d_ncand, cuda_stream);
}

// vis: DEVICE slab (d_stage == nullptr) or HOST slab copied chunk by chunk through the two halves of
// d_stage on the plan's copy stream, overlapped with the kernels of the previous chunk.
static int run_search(const volks_plan *pl, const void *d_vis, void *d_stage, const int32_t *d_shift, void *d_workspace,
                      volks_peak *d_peaks, volks_cand *d_cands, uint32_t cand_capacity, uint32_t *d_ncand,
                      void *cuda_stream) {
  if (!pl || !d_vis || !d_workspace || !d_ncand || (!d_cands && cand_capacity > 0)) return VOLKS_EINVAL;
  const size_t pair_elems = (size_t)pl->sched.nap * pl->nchan;   // visibilities of one pair (all-IF: one baseline)
  size_t stage_bytes = 0;
  if (d_stage) {
    volks_plan_query_host(pl, &stage_bytes);
    if (!pl->copy_stream) {
      if (!cuda_ok(cudaStreamCreateWithFlags(&pl->copy_stream, cudaStreamNonBlocking))) return VOLKS_ECUDA;
      for (int k = 0; k < 2; ++k) {
        if (!cuda_ok(cudaEventCreateWithFlags(&pl->ev_copied[k], cudaEventDisableTiming)) ||
            !cuda_ok(cudaEventCreateWithFlags(&pl->ev_free[k], cudaEventDisableTiming))) return VOLKS_ECUDA;
      }
    }
  }
  {
    int dev = -1;
    if (!cuda_ok(cudaGetDevice(&dev))) return VOLKS_ECUDA;
    if (dev != pl->device) return VOLKS_EINVAL;        // the plan's tables live on the device it was created on
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const Sched &s = pl->sched;
  char *ws = (char *)d_workspace;
  // candidates-only index mode for the eligible sliding widths unless the dense peak array (every window's exact
  // index) is wanted or the plan was created with full_index
  const bool hy = pl->cand_only && (pl->nuntag > 0 || pl->nprune > 0) && d_peaks == nullptr;
  const unsigned char *flags = hy && pl->nprune ? (const unsigned char *)(ws + pl->off_flags) : nullptr;
  pl->last_full_index = !hy;
  u64 *keys = (u64 *)(ws + pl->off_keys);
  float *E = (float *)(ws + pl->off_E);
  uint32_t *cnt = (uint32_t *)(ws + pl->off_cnt);
  float2 *Y = (float2 *)(ws + pl->off_Y);
  const float *noise = pl->ai_nif ? (const float *)(ws + pl->off_noise) : nullptr;
  if (s.nwin_total == 0) {
    return cuda_ok(cudaMemsetAsync(d_ncand, 0, sizeof(uint32_t), st)) ? VOLKS_OK : VOLKS_ECUDA;
  }
  pl->prof_kind.clear(); pl->prof_wid.clear();
  if (!cuda_ok(cudaMemsetAsync(keys, 0, (size_t)s.nwin_total * sizeof(u64), st))) return VOLKS_ECUDA;
  // host slab: a quarter of the plan's chunk per copy (VOLKS_HOST_SPLIT, default 4), so that the first copy
  // and the last chunk's kernels - the two parts of the pipeline nothing overlaps - are short (config 2:
  // 211 -> 187 ms per step from pinned memory; the device-resident search keeps the large chunks, which its
  // kernels prefer: 163 against 168 ms)
  const long long ppc = d_stage ? std::max<long long>(1, (pl->pairs_per_chunk + pl->host_split - 1) / pl->host_split)
                                : pl->pairs_per_chunk;
  const long long nchunks = (pl->npair + ppc - 1) / ppc;
  for (long long ch = 0; ch < nchunks; ++ch) {
    const long long pair0 = ch * ppc;
    const long long np = std::min(ppc, pl->npair - pair0);
    RowArgs ra;
    ra.vis = (const float2 *)d_vis;
    if (d_stage) {
      const int k = (int)(ch & 1);
      char *dst = (char *)d_stage + (size_t)k * stage_bytes;
      // the stage half is free once the row kernel that last read it (chunk ch-2, or the previous call's)
      // is done: ev_free[k] is recorded right after that kernel; a never-recorded event does not block
      if (!cuda_ok(cudaStreamWaitEvent(pl->copy_stream, pl->ev_free[k], 0))) return VOLKS_ECUDA;
      if (!cuda_ok(cudaMemcpyAsync(dst, (const char *)d_vis + (size_t)pair0 * pair_elems * sizeof(float2),
                                   (size_t)np * pair_elems * sizeof(float2), cudaMemcpyHostToDevice, pl->copy_stream)) ||
          !cuda_ok(cudaEventRecord(pl->ev_copied[k], pl->copy_stream)) ||
          !cuda_ok(cudaStreamWaitEvent(st, pl->ev_copied[k], 0))) return VOLKS_ECUDA;
      ra.vis = (const float2 *)dst - (size_t)pair0 * pair_elems;   // kernels index by absolute pair
    }
    ra.Y = Y; ra.E = E; ra.twf = pl->d_tables;
    ra.row0 = pair0 * s.nap * pl->ai_psub; ra.nrows = np * s.nap * pl->ai_psub;
    ra.psub = pl->ai_psub; ra.premod = pl->ai_psub > 1 ? pl->d_tables + pl->premod_off : nullptr;
    ra.nchan = pl->nchan; ra.nf = pl->row_nf; ra.tpr = pl->row_tpr; ra.rows_per_cta = pl->row_rows_per_cta; ra.pitch = pl->pitch; ra.paired = pl->paired;
    ra.cal = pl->d_cal;
    ra.dlo = pl->ai_nif ? -1 : s.dlo; ra.dhi = pl->ai_nif ? -1 : s.dhi;   // (f2: k_allif masks its argmax; its noise needs every column)
    ra.shift = d_shift; ra.nif = s.nif; ra.allif_nif = pl->ai_nif; ra.allif_nchan = pl->ai_nchan;
    ra.keys1 = nullptr; ra.per_pair = s.per_pair; ra.nap = s.nap; ra.stride1 = 1; ra.nwin1 = 0;
    if (pl->wid1 >= 0) { ra.keys1 = keys + s.offc[pl->wid1]; ra.stride1 = s.stride[pl->wid1]; ra.nwin1 = (int)s.nwin[pl->wid1]; }
    const long long rblocks = (ra.nrows + ra.rows_per_cta - 1) / ra.rows_per_cta;
    {
      ProfScope ps(pl, st, VOLKS_K_ROW, -1);
      if (pl->row_generic || !(launch_row2(ra, st) || launch_rowbig(ra, st, false)))
        k_row_fft<<<(unsigned)rblocks, ra.tpr * ra.rows_per_cta, pl->row_smem, st>>>(ra);
      if (d_stage && !cuda_ok(cudaEventRecord(pl->ev_free[ch & 1], st))) return VOLKS_ECUDA;
    }
    const bool use_cw = pl->cwq >= 0 && pl->wp[pl->cwq].nwin > 0;   // (needs the pre-thresholds and k_bound in both index modes)
    const int cw_in_bound = use_cw && !pl->cw_pf ? 1 : 0;           // the column-level width is one of k_bound's widths
    if (hy || use_cw) {
      WinThrArgs ta;
      ta.E = E; ta.thr = (uint32_t *)(ws + pl->off_thr); ta.per_pair = s.per_pair; ta.pair0 = pair0;
      ta.thr2 = s.snr_thresh * s.snr_thresh; ta.nap = s.nap; ta.nq = 0; ta.cum[0] = 0;
      for (int q = 0; q < s.nwidths; ++q) {
        const WidthPlan &w = pl->wp[q];
        if ((!w.untag && w.prune < 0) || w.nwin == 0) continue;
        const int i = ta.nq++;
        ta.w[i] = w.w; ta.stride[i] = w.s; ta.nwin[i] = (int)w.nwin; ta.offc[i] = s.offc[q]; ta.cum[i + 1] = ta.cum[i] + w.nwin;
      }
      ta.total = np * ta.cum[ta.nq];
      {
        ProfScope ps(pl, st, VOLKS_K_WINTHR, -1);
        k_winthr<<<(unsigned)((ta.total + 255) / 256), 256, 0, st>>>(ta);
      }
      if (flags || use_cw) {
        PruneArgs pa;
        pa.Y = Y; pa.thr = ta.thr; pa.flags = (unsigned char *)(ws + pl->off_flags); pa.per_pair = s.per_pair;
        pa.nap = s.nap; pa.nf = s.nf; pa.pitch = pl->pitch; pa.seg = pl->prune_seg;
        pa.nseg = pl->prune_nseg;
        pa.ncp = pl->dt_n * 32; pa.cp_na = pl->dt_na * 32; pa.cp_a0 = pl->dt_a0 * 32; pa.cp_b0 = pl->dt_b0 * 32;
        // the pruned widths (candidates-only mode), then the column-level width as the last entry
        pa.nq = 0; pa.wmax = 1;
        for (int q = 0; q < s.nwidths && flags; ++q) {
          const WidthPlan &w = pl->wp[q];
          if (w.prune < 0) continue;
          pa.w[w.prune] = w.w; pa.nwin[w.prune] = (int)w.nwin; pa.offc[w.prune] = s.offc[q];
          pa.nq = std::max(pa.nq, w.prune + 1); pa.wmax = std::max(pa.wmax, w.w);
        }
        pa.cwmask = nullptr; pa.cw_nwords = pl->cw_nwords; pa.cwdense = (unsigned char *)(ws + pl->off_cwdense);
        pa.cwempty = pa.cwdense + (size_t)pl->pairs_per_chunk * ((pl->prune_nseg + 1) / 2);
        if (use_cw) {
          pa.cwmask = (uint32_t *)(ws + pl->off_cwmask);
          if (!cuda_ok(cudaMemsetAsync(pa.cwmask, 0, (size_t)np * pl->cw_nwords * s.nf * sizeof(uint32_t), st))) return VOLKS_ECUDA;
        }
        if (cw_in_bound) {
          const WidthPlan &w = pl->wp[pl->cwq];
          const int i = pa.nq++;
          pa.w[i] = w.w; pa.nwin[i] = (int)w.nwin; pa.offc[i] = s.offc[pl->cwq]; pa.wmax = std::max(pa.wmax, w.w);
        }
        const int thr = std::min(PRUNE_THREADS, s.nf / 2);   // (nf >= 64: a power of two >= 32)
        pa.ring = pa.wmax <= 16 ? 16 : 32;                 // rows of amplitude history (a power of two >= wmax)
        const int nthr_t = thr > 64 ? 128 : 64;            // the kernel's compile-time thread count (row strides)
        const size_t smem = prune_smem_bytes(pa.nq, pa.seg, pa.ring, nthr_t);
        const unsigned blocks = (unsigned)(np * ((pa.nseg + 1) / 2));
        ProfScope ps(pl, st, VOLKS_K_BOUND, -1);
#define VOLKS_BOUND(NQ_)                                                                   \
  case NQ_:                                                                                \
    if (cw_in_bound) { if (nthr_t == 128) k_bound<NQ_, 1, 128><<<blocks, thr, smem, st>>>(pa); else k_bound<NQ_, 1, 64><<<blocks, thr, smem, st>>>(pa); } \
    else { if (nthr_t == 128) k_bound<NQ_, 0, 128><<<blocks, thr, smem, st>>>(pa); else k_bound<NQ_, 0, 64><<<blocks, thr, smem, st>>>(pa); } \
    break;
        switch (pa.nq) { VOLKS_BOUND(1) VOLKS_BOUND(2) VOLKS_BOUND(3) VOLKS_BOUND(4) VOLKS_BOUND(5) VOLKS_BOUND(6) VOLKS_BOUND(7) VOLKS_BOUND(8) }
#undef VOLKS_BOUND
        if (use_cw && pl->cw_pf) {     // the column-level width's bits by the folded bound (same stream, same profile slot)
          const WidthPlan &w = pl->wp[pl->cwq];
          PairFoldArgs fa;
          fa.Y = Y; fa.thr = ta.thr; fa.cwmask = pa.cwmask; fa.cwdense = pa.cwdense; fa.cwempty = pa.cwempty;
          fa.per_pair = s.per_pair; fa.offc = s.offc[pl->cwq];
          fa.nap = s.nap; fa.nf = s.nf; fa.pitch = pl->pitch; fa.nwin = (int)w.nwin; fa.cw_nwords = pl->cw_nwords;
          fa.ntile128 = (pl->prune_nseg + 1) / 2;
          fa.ncp = pa.ncp; fa.cp_na = pa.cp_na; fa.cp_a0 = pa.cp_a0; fa.cp_b0 = pa.cp_b0;
          k_pairfold<<<(unsigned)(np * ((w.nwin + PF_T - 1) / PF_T)), PF_THREADS, pairfold_smem_bytes(), st>>>(fa);
        }
      }
    }
    for (int q = 0; q < s.nwidths; ++q) {
      const WidthPlan &w = pl->wp[q];
      if (w.nwin == 0 || q == pl->wid1) continue;
      ColArgs ca;
      ca.Y = Y; ca.keys = keys; ca.twt = pl->d_tables + w.tw_off;
      ca.per_pair = s.per_pair; ca.offc = s.offc[q]; ca.pair0 = pair0;
      ca.nap = s.nap; ca.nf = s.nf; ca.log2nf = s.log2nf; ca.w = w.w; ca.stride = w.s; ca.nt = w.nt;
      ca.log2m = w.log2m; ca.nwin = (int)w.nwin; ca.pitch = pl->pitch; ca.paired = pl->paired;
      ca.total = ((np * w.nwin) << w.log2m) * s.nf;
      if (pl->ai_nif) {
        AllifArgs aa;
        aa.Y = Y; aa.keys = keys; aa.noise = (float *)(ws + pl->off_noise); aa.E = E;
        aa.per_pair = s.per_pair; aa.offc = s.offc[q]; aa.pair0 = pair0;
        aa.nap = s.nap; aa.nf = s.nf; aa.w = w.w; aa.stride = w.s; aa.nwin = (int)w.nwin; aa.seg = w.seg;
        aa.nseg = w.nseg; aa.pitch = pl->pitch * pl->ai_psub;
        aa.gsplit = s.ngs; aa.dlo = s.dlo; aa.dhi = s.dhi;
        const int cols = s.nf / s.ngs;                               // columns per CTA
        const int thr = std::min(1024, cols / 2), cp = cols / 2 / thr;
        const unsigned blocks = (unsigned)(np * w.nseg * s.ngs);
        ProfScope ps(pl, st, VOLKS_K_ALLIF, q);
        if (s.ngs > 1) k_allif<4, true><<<blocks, thr, 0, st>>>(aa);   // cols = 8192
        else if (cp == 1) k_allif<1, false><<<blocks, thr, 0, st>>>(aa);
        else if (cp == 2) k_allif<2, false><<<blocks, thr, 0, st>>>(aa);
        else k_allif<4, false><<<blocks, thr, 0, st>>>(aa);
        continue;
      }
      const bool fold = w.slide && w.sf && hy;   // candidates-only mode, wide stride-1 width (kernels_sfold.cuh)
      if (w.slide) {
        SlideArgs sa;
        sa.Y = Y; sa.keys = keys; sa.twt = pl->d_tables + w.tw_off; sa.tw4 = (const float4 *)(pl->d_tables + w.tw4_off);
        sa.per_pair = s.per_pair; sa.offc = s.offc[q]; sa.pair0 = pair0;
        sa.nap = s.nap; sa.nf = s.nf; sa.w = w.w; sa.nt = w.nt; sa.log2m = w.log2m; sa.nwin = (int)w.nwin;
        sa.seg = w.seg; sa.nseg = w.nseg; sa.keymask = 0xFFFFFFF0u; sa.pitch = pl->pitch;
        sa.ndt = pl->dt_n; sa.dt_na = pl->dt_na; sa.dt_a0 = pl->dt_a0; sa.dt_b0 = pl->dt_b0;
        sa.ntasks = ((np * w.nseg * (long long)pl->dt_n) << w.log2m);
        sa.flags = flags && w.prune >= 0 ? flags + (size_t)w.prune * pl->prune_nseg : nullptr;
        sa.flag_stride = (pl->nprune + cw_in_bound) * pl->prune_nseg;
        if (hy && w.cw) { sa.flags = (const unsigned char *)(ws + pl->off_cwdense); sa.flag_stride = (pl->prune_nseg + 1) / 2; }   // dense tiles only
        sa.thr = (const uint32_t *)(ws + pl->off_thr); sa.hits = nullptr; sa.nblk = w.nblk;
        if (fold) {
          // 1. the folded sliding sum: one hit bit per (window, rate residue, 64-column tile)
          // (longer segments than the sliding kernel's: a step costs a fifth, so the start of a segment - its first window
          // folded from w samples - weighs five times as much)
          sa.hits = (unsigned short *)(ws + w.off_hits);
          sa.seg = w.seg * SFOLD_SEGMUL; sa.nseg = (int)((w.nwin + sa.seg - 1) / sa.seg);
          sa.ntasks = ((np * sa.nseg * (long long)pl->dt_n) << w.log2m);
          {
            ProfScope ps(pl, st, VOLKS_K_SFOLD, q);
            launch_slide(sa, st, true);
          }
          sa.seg = w.seg; sa.nseg = w.nseg;
          sa.ntasks = ((np * w.nseg * (long long)pl->dt_n) << w.log2m);
          // 2. segments with more than 1/8 of their bits set (interference) go to the ordinary sliding kernel
          SfoldArgs ea;
          ea.Y = Y; ea.tw4 = (const float4 *)(pl->d_tables + w.tw4_off); ea.hits = sa.hits; ea.dense = (unsigned char *)(ws + w.off_sfdense); ea.list = (uint32_t *)(ws + w.off_sflist); ea.keys = keys;
          ea.thr = sa.thr; ea.E = E + pair0 * (long long)s.nap; ea.hits_rw = (unsigned short *)(ws + w.off_hits);
          ea.big16 = (unsigned short *)(ws + w.off_sfbig);
          ea.per_pair = s.per_pair; ea.offc = s.offc[q]; ea.pair0 = pair0;
          ea.nap = s.nap; ea.nf = s.nf; ea.w = w.w; ea.nt = w.nt; ea.log2m = w.log2m; ea.nwin = (int)w.nwin;
          ea.seg = w.seg; ea.nseg = w.nseg; ea.pitch = pl->pitch; ea.nblk = w.nblk;
          ea.ndt = pl->dt_n; ea.dt_na = pl->dt_na; ea.dt_a0 = pl->dt_a0; ea.dt_b0 = pl->dt_b0;
          ea.ntasks = np * w.nseg;
          {
            ProfScope ps(pl, st, VOLKS_K_SFOLD_EVAL, q);
            {   // dynamic-range guard: windows behind a row of overwhelming energy are flagged wholesale
              const int fseg = w.seg * SFOLD_SEGMUL;
              k_sfold_guard<<<(unsigned)(np * ((w.nwin + fseg - 1) / fseg)), 128, 0, st>>>(ea, fseg);
            }
            k_sfold_density<<<(unsigned)ea.ntasks, 128, 0, st>>>(ea);
            // 3. every other flagged (window, rho, tile) exactly, from its samples
            ea.ntasks = ((np * w.nblk * (long long)pl->dt_n) << w.log2m);
            k_sfold_compact<<<(unsigned)((ea.ntasks + 255) / 256), 256, 0, st>>>(ea);
            k_sfold_eval<<<SFOLD_EVAL_WARPS, 32, 0, st>>>(ea);
          }
          sa.hits = nullptr; sa.flags = ea.dense; sa.flag_stride = w.nseg;     // 4. the dense segments, below
        }
        ProfScope ps(pl, st, VOLKS_K_SLIDE, q);
        launch_slide(sa, st);
        continue;
      }
      if (w.colfft) {
        ColFftArgs fa;
        fa.Y = Y; fa.keys = keys; fa.tw4 = (const float4 *)(pl->d_tables + w.tw4_off);
        fa.per_pair = s.per_pair; fa.offc = s.offc[q]; fa.pair0 = pair0;
        fa.nap = s.nap; fa.nf = s.nf; fa.w = w.w; fa.stride = w.s; fa.nt = w.nt; fa.nwin = (int)w.nwin;
        fa.pitch = pl->pitch; fa.paired = pl->paired; fa.split2 = pl->cf_split2; fa.wpc = w.cf_wpc; fa.nrange = w.cf_nrange; fa.keymask = 0xFFFFFFF0u;
        fa.thr = hy && w.untag ? (const uint32_t *)(ws + pl->off_thr) : nullptr;
        fa.energy_first = CF2_ENERGY_FIRST;
        ProfScope ps(pl, st, VOLKS_K_COLFFT, q);
        if (!cuda_ok(launch_colfft(fa, w.cf_l1, w.cf_nz, np * (s.nf / 32) * w.cf_nrange, st, false))) return VOLKS_ECUDA;
        continue;
      }
      ProfScope ps(pl, st, VOLKS_K_COL, q);
      switch (w.L) {
        case 1: launch_col<1>(ca, st); break;
        case 2: launch_col<2>(ca, st); break;
        case 4: launch_col<4>(ca, st); break;
        case 8: launch_col<8>(ca, st); break;
        default: launch_col<16>(ca, st); break;
      }
    }
    // exact re-evaluation of the sliding widths' windows that sit far below an earlier window of their segment
    if (pl->nslide > 0) {
      FixArgs fa;
      fa.Y = Y; fa.keys = keys; fa.tables = pl->d_tables; fa.per_pair = s.per_pair; fa.pair0 = pair0;
      fa.nap = s.nap; fa.nf = s.nf; fa.log2nf = s.log2nf; fa.pitch = pl->pitch; fa.paired = pl->paired;
      fa.nq = 0; fa.unit0[0] = 0;
      fa.cwdense = hy && use_cw ? (const unsigned char *)(ws + pl->off_cwdense) : nullptr; fa.cw_i = -1; fa.cw_ntile = (pl->prune_nseg + 1) / 2;
      fa.flags = flags; fa.flag_nq = pl->nprune + cw_in_bound; fa.flag_nseg = pl->prune_nseg;
      for (int q = 0; q < s.nwidths; ++q) {
        const WidthPlan &w = pl->wp[q];
        if (!w.slide || w.nwin == 0) continue;
        const int i = fa.nq++;
        if (hy && w.cw) fa.cw_i = i;
        // a folded-sum width: only its dense segments went through the sliding kernel (the others hold exact keys)
        fa.sfdense[i] = hy && w.sf ? (const unsigned char *)(ws + w.off_sfdense) : nullptr;
        fa.q[i] = q; fa.w[i] = w.w; fa.nt[i] = w.nt; fa.seg[i] = w.seg; fa.nseg[i] = w.nseg; fa.nwin[i] = (int)w.nwin;
        fa.offc[i] = s.offc[q]; fa.tw_off[i] = (long long)w.tw_off; fa.flag_q[i] = w.prune;
        fa.unit0[i + 1] = fa.unit0[i] + (w.nseg + FIX_GROUP - 1) / FIX_GROUP;
      }
      ProfScope ps(pl, st, VOLKS_K_FIXUP, -1);
      if (fa.unit0[fa.nq] > 0) k_fixup<<<(unsigned)(np * fa.unit0[fa.nq]), 256, 0, st>>>(fa);
    }
    // the peak bins of the untagged sliding widths: every window (full index) or the possible candidates
    if (pl->nuntag > 0) {
      RecoverArgs ra2;
      ra2.Y = Y; ra2.keys = keys; ra2.thr = hy ? (const uint32_t *)(ws + pl->off_thr) : nullptr; ra2.tables = pl->d_tables;
      ra2.per_pair = s.per_pair; ra2.pair0 = pair0; ra2.nap = s.nap; ra2.nf = s.nf; ra2.log2nf = s.log2nf; ra2.pitch = pl->pitch;
      ra2.nq = 0; ra2.cum[0] = 0;
      for (int q = 0; q < s.nwidths; ++q) {
        const WidthPlan &w = pl->wp[q];
        if (!w.untag || w.nwin == 0) continue;
        const int i = ra2.nq++;
        ra2.w[i] = w.w; ra2.stride[i] = w.s; ra2.nt[i] = w.nt; ra2.log2m[i] = w.log2m; ra2.nwin[i] = (int)w.nwin; ra2.offc[i] = s.offc[q];
        ra2.tw_off[i] = (long long)w.tw_off; ra2.cum[i + 1] = ra2.cum[i] + w.nwin;
      }
      ra2.total = np * ra2.cum[ra2.nq];
      ProfScope ps(pl, st, VOLKS_K_RECOVER, -1);
      k_recover<<<(unsigned)((ra2.total + 127) / 128), 128, 0, st>>>(ra2);
    }
    // the column-level width: every listed (window, column pair) by the definition; replaces the keys of those windows
    if (use_cw) {
      const WidthPlan &w = pl->wp[pl->cwq];
      ColEvalArgs ea;
      ea.Y = Y; ea.keys = keys; ea.mask = (const uint32_t *)(ws + pl->off_cwmask);
      ea.twt = pl->d_tables + w.tw_off; ea.thr = (const uint32_t *)(ws + pl->off_thr);
      ea.per_pair = s.per_pair; ea.offc = s.offc[pl->cwq]; ea.pair0 = pair0;
      ea.nap = s.nap; ea.nf = s.nf; ea.pitch = pl->pitch; ea.w = w.w; ea.nt = w.nt; ea.log2m = w.log2m;
      ea.nwin = (int)w.nwin; ea.nwords = pl->cw_nwords; ea.dense = (const unsigned char *)(ws + pl->off_cwdense);
      ea.empty = ea.dense + (size_t)pl->pairs_per_chunk * ((pl->prune_nseg + 1) / 2);
      ea.dstride = (pl->prune_nseg + 1) / 2; ea.only_above = hy ? 0 : 1;
      ProfScope ps(pl, st, VOLKS_K_COLEVAL, pl->cwq);
      k_coleval<<<(unsigned)(np * ((w.nwin + CE_TILE - 1) / CE_TILE)), CE_THREADS, 0, st>>>(ea);
    }
  }
  {
    ProfScope ps(pl, st, VOLKS_K_FINALIZE, -1);
    k_finalize<<<(unsigned)pl->nfin_blocks, FIN_THREADS, 0, st>>>(pl->d_sched, keys, E, (float4 *)d_peaks, cnt, nullptr, 0.f, noise);
  }
  {
    ProfScope ps(pl, st, VOLKS_K_SCAN, -1);
    k_scan<<<1, 1024, 0, st>>>(cnt, pl->nfin_blocks, d_ncand);
  }
  {
    ProfScope ps(pl, st, VOLKS_K_SCATTER, -1);
    k_scatter<<<(unsigned)pl->nfin_blocks, FIN_THREADS, 0, st>>>(pl->d_sched, keys, E, cnt, (CandOut *)d_cands, cand_capacity, nullptr, 0.f, noise, d_ncand);
  }
  return cuda_ok(cudaGetLastError()) ? VOLKS_OK : VOLKS_ECUDA;
}

int volks_zscore_select(const volks_plan *pl, void *d_workspace, float z_thresh, volks_peak *d_peaks,
                        volks_cand *d_cands, uint32_t cand_capacity, uint32_t *d_ncand, void *cuda_stream) {
  if (!pl || !d_workspace || !d_ncand || (!d_cands && cand_capacity > 0) || !(z_thresh == z_thresh)) return VOLKS_EINVAL;
  if (!pl->last_full_index) return VOLKS_EINVAL;   // the last search kept exact indices for its candidates only
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const Sched &s = pl->sched;
  if (s.nwin_total == 0) return cuda_ok(cudaMemsetAsync(d_ncand, 0, sizeof(uint32_t), st)) ? VOLKS_OK : VOLKS_ECUDA;
  char *ws = (char *)d_workspace;
  const u64 *keys = (const u64 *)(ws + pl->off_keys);
  const float *E = (const float *)(ws + pl->off_E);
  uint32_t *cnt = (uint32_t *)(ws + pl->off_cnt);
  double2 *zst = (double2 *)(ws + pl->off_zst);
  const float *noise = pl->ai_nif ? (const float *)(ws + pl->off_noise) : nullptr;
  k_zstat<<<(unsigned)(pl->npair * s.nwidths), 256, 0, st>>>(pl->d_sched, keys, E, zst, noise);
  k_finalize<<<(unsigned)pl->nfin_blocks, FIN_THREADS, 0, st>>>(pl->d_sched, keys, E, (float4 *)d_peaks, cnt, zst, z_thresh, noise);
  k_scan<<<1, 1024, 0, st>>>(cnt, pl->nfin_blocks, d_ncand);
  k_scatter<<<(unsigned)pl->nfin_blocks, FIN_THREADS, 0, st>>>(pl->d_sched, keys, E, cnt, (CandOut *)d_cands, cand_capacity, zst, z_thresh, noise, d_ncand);
  return cuda_ok(cudaGetLastError()) ? VOLKS_OK : VOLKS_ECUDA;
}

int volks_plan_profile(volks_plan *pl, int enable) {
  if (!pl) return VOLKS_EINVAL;
  pl->prof_on = enable != 0;
  pl->prof_kind.clear(); pl->prof_wid.clear();
  return VOLKS_OK;
}

int volks_plan_profile_read(const volks_plan *pl, int32_t capacity, int32_t *kind, int32_t *wid, float *ms,
                            int32_t *n) {
  if (!pl || !n || capacity < 0 || (capacity > 0 && (!kind || !wid || !ms))) return VOLKS_EINVAL;
  *n = (int32_t)pl->prof_kind.size();
  for (int32_t i = 0; i < *n && i < capacity; ++i) {
    if (!cuda_ok(cudaEventSynchronize(pl->prof_ev[2 * i + 1]))) return VOLKS_ECUDA;
    if (!cuda_ok(cudaEventElapsedTime(&ms[i], pl->prof_ev[2 * i], pl->prof_ev[2 * i + 1]))) return VOLKS_ECUDA;
    kind[i] = pl->prof_kind[i]; wid[i] = pl->prof_wid[i];
  }
  return VOLKS_OK;
}

// Host: sweep over candidates sorted by start AP inside each (bl, ifq) group.  Interval-overlap
// connected components are exactly the maximal runs whose start lies before the running end.
int volks_window_match(const volks_cand *cands, uint32_t ncand, const int32_t *width, int32_t nwidths,
                       int32_t min_widths, volks_pulse *out, uint32_t capacity, uint32_t *nout) {
  if (!width || nwidths < 1 || nwidths > VOLKS_MAX_WIDTHS || !nout || (!cands && ncand) || (!out && capacity))
    return VOLKS_EINVAL;
  struct { const int32_t *width; int nwidths; } s = {width, nwidths};
  std::vector<uint32_t> ord(ncand);
  for (uint32_t i = 0; i < ncand; ++i) {
    if (cands[i].wid < 0 || cands[i].wid >= s.nwidths) return VOLKS_EINVAL;
    ord[i] = i;
  }
  std::stable_sort(ord.begin(), ord.end(), [&](uint32_t a, uint32_t b) {
    const volks_cand &x = cands[a], &y = cands[b];
    if (x.bl != y.bl) return x.bl < y.bl;
    if (x.ifq != y.ifq) return x.ifq < y.ifq;
    return x.t0 < y.t0;
  });
  struct Rec { uint32_t best; int nhit, tb, te; };
  std::vector<Rec> found;
  uint32_t i = 0;
  while (i < ncand) {
    const volks_cand &f = cands[ord[i]];
    int end = f.t0 + s.width[f.wid];
    uint32_t best = ord[i];
    uint32_t mask = 1u << f.wid;
    uint32_t k = i + 1;
    while (k < ncand) {
      const volks_cand &c = cands[ord[k]];
      if (c.bl != f.bl || c.ifq != f.ifq || c.t0 >= end) break;
      end = std::max(end, c.t0 + s.width[c.wid]);
      mask |= 1u << c.wid;
      const volks_cand &b = cands[best];
      if (c.snr > b.snr || (c.snr == b.snr && ord[k] < best)) best = ord[k];
      ++k;
    }
    int nhit = 0;
    for (uint32_t m = mask; m; m &= m - 1) ++nhit;
    if (nhit >= min_widths) found.push_back({best, nhit, f.t0, end});
    i = k;
  }
  std::sort(found.begin(), found.end(), [](const Rec &a, const Rec &b) { return a.best < b.best; });
  *nout = (uint32_t)found.size();
  for (uint32_t n = 0; n < found.size() && n < capacity; ++n) {
    out[n].best = cands[found[n].best];
    out[n].nwidths_hit = found[n].nhit; out[n].t_begin = found[n].tb; out[n].t_end = found[n].te;
  }
  return found.size() > capacity ? VOLKS_EOVERFLOW : VOLKS_OK;
}

// Host: interval-overlap components over ALL pulses = maximal runs, in t_begin order, whose start lies
// before the running end.
int volks_baseline_match(const volks_pulse *pulses, uint32_t npulse, int32_t min_baselines, volks_detection *out,
                         uint32_t capacity, uint32_t *nout) {
  if (!nout || (!pulses && npulse) || (!out && capacity)) return VOLKS_EINVAL;
  std::vector<uint32_t> ord(npulse);
  for (uint32_t i = 0; i < npulse; ++i) ord[i] = i;
  std::stable_sort(ord.begin(), ord.end(), [&](uint32_t x, uint32_t y) { return pulses[x].t_begin < pulses[y].t_begin; });
  uint32_t found = 0, i = 0;
  std::vector<int32_t> bls;
  while (i < npulse) {
    const volks_pulse &f = pulses[ord[i]];
    int end = f.t_end;
    uint32_t best = ord[i], k = i + 1;
    bls.assign(1, f.best.bl);
    while (k < npulse && pulses[ord[k]].t_begin < end) {
      const volks_pulse &c = pulses[ord[k]];
      end = std::max(end, c.t_end);
      bls.push_back(c.best.bl);
      const volks_pulse &b = pulses[best];
      if (c.best.snr > b.best.snr || (c.best.snr == b.best.snr && ord[k] < best)) best = ord[k];
      ++k;
    }
    std::sort(bls.begin(), bls.end());
    const int nb = (int)(std::unique(bls.begin(), bls.end()) - bls.begin());
    if (nb >= min_baselines) {
      if (found < capacity) {
        out[found].best = pulses[best]; out[found].nbaselines = nb;
        out[found].t_begin = f.t_begin; out[found].t_end = end;
      }
      ++found;
    }
    i = k;
  }
  *nout = found;
  return found > capacity ? VOLKS_EOVERFLOW : VOLKS_OK;
}

int volks_measure_fp32_peak(int32_t repeats, double *tflops_best, double *tflops_mean, double *ms_per_launch,
                            void *cuda_stream) {
  if (repeats < 1 || repeats > 1000 || !tflops_best) return VOLKS_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0;
  if (!cuda_ok(cudaGetDevice(&dev)) || !cuda_ok(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)))
    return VOLKS_ECUDA;
  const int ctas = sms * 8, thr = 256, iters = 65536;     // ~20 ms per launch on B200
  float *buf = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (!cuda_ok(cudaMalloc(&buf, (size_t)ctas * thr * sizeof(float)))) return VOLKS_ECUDA;
  bool ok = cuda_ok(cudaEventCreate(&e0)) && cuda_ok(cudaEventCreate(&e1));
  const double flops = (double)ctas * thr * iters * 32.0 * 2.0;
  double best = 0.0, sum = 0.0, ms_sum = 0.0;
  if (ok) k_fp32_probe<<<ctas, thr, 0, st>>>(buf, iters / 8, 0.999f, 1e-3f);   // warm-up (clocks, code load)
  for (int r = 0; ok && r < repeats; ++r) {
    ok = cuda_ok(cudaEventRecord(e0, st));
    k_fp32_probe<<<ctas, thr, 0, st>>>(buf, iters, 0.999f, 1e-3f);
    ok = ok && cuda_ok(cudaEventRecord(e1, st)) && cuda_ok(cudaEventSynchronize(e1));
    float ms = 0.f;
    ok = ok && cuda_ok(cudaEventElapsedTime(&ms, e0, e1)) && ms > 0.f;
    if (ok) { const double tf = flops / (ms * 1e-3) / 1e12; best = std::max(best, tf); sum += tf; ms_sum += ms; }
  }
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  cudaFree(buf);
  if (!ok) return VOLKS_ECUDA;
  *tflops_best = best;
  if (tflops_mean) *tflops_mean = sum / repeats;
  if (ms_per_launch) *ms_per_launch = ms_sum / repeats;
  return VOLKS_OK;
}

int volks_dm_shifts(double dm, const double *f_chan_mhz, int32_t n, double f_ref_mhz, double ap_seconds,
                    int32_t *shift) {
  if (!f_chan_mhz || !shift || n < 0 || !(f_ref_mhz > 0) || !(ap_seconds > 0) || !(dm == dm)) return VOLKS_EINVAL;
  const double fr = f_ref_mhz * 1e-3;
  for (int32_t i = 0; i < n; ++i) {
    if (!(f_chan_mhz[i] > 0)) return VOLKS_EINVAL;
    const double f = f_chan_mhz[i] * 1e-3;
    shift[i] = (int32_t)llrint(4.148808e-3 * dm * (1.0 / (f * f) - 1.0 / (fr * fr)) / ap_seconds);
  }
  return VOLKS_OK;
}

int volks_bin_to_physical(int32_t nt, int32_t nf, int32_t rate_idx, int32_t delay_idx, double ap_seconds,
                          double chan_hz, double *rate_hz, double *delay_s) {
  if (nt < 1 || nf < 1) return VOLKS_EINVAL;
  if (rate_idx < 0 || rate_idx >= nt || delay_idx < 0 || delay_idx >= nf) return VOLKS_EINVAL;
  if (!(ap_seconds > 0) || !(chan_hz > 0)) return VOLKS_EINVAL;
  const int rs = rate_idx >= (nt + 1) / 2 && nt > 1 ? rate_idx - nt : rate_idx;
  const int ds = delay_idx >= (nf + 1) / 2 && nf > 1 ? delay_idx - nf : delay_idx;
  if (rate_hz) *rate_hz = rs / (nt * ap_seconds);
  if (delay_s) *delay_s = ds / (nf * chan_hz);
  return VOLKS_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// volks_search_noalloc: the same search for callers that cannot allocate (include/volks.h).
// Every intermediate - the window schedule, the twiddle tables, the per-window keys, the per-AP energies, the
// block counts and the delay spectra - lives in ONE file-scope device array that every GPU loading this library
// holds until exit.  g_noalloc_scratch is a HOST-SIDE STAND-IN in host code, not a device address: the address is
// taken once per device with cudaGetSymbolAddress (that device current) and only that pointer goes to kernels.
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_noalloc_scratch[VOLKS_NOALLOC_SCRATCH_BYTES];

namespace {

constexpr int NOALLOC_MAX_DEVICES = 64;
unsigned char *g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {nullptr};   // per device, filled on first use
std::mutex g_noalloc_mutex;

struct NoAllocTables { int nf, nq; int nt[VOLKS_MAX_WIDTHS]; long long off[VOLKS_MAX_WIDTHS]; };

// writes the schedule and the twiddle tables into the scratch (double-precision sincospi, rounded once to float)
__global__ void __launch_bounds__(256) k_noalloc_setup(Sched s, NoAllocTables t, Sched *d_sched, float2 *tab) {
  const long long gid = (long long)blockIdx.x * 256 + threadIdx.x, nthr = (long long)gridDim.x * 256;
  if (gid == 0) *d_sched = s;
  for (long long k = gid; k < t.nf; k += nthr) {
    double sn, cs;
    sincospi(-2.0 * (double)k / (double)t.nf, &sn, &cs);
    tab[k] = make_float2((float)cs, (float)sn);
  }
  for (int q = 0; q < t.nq; ++q)
    for (long long k = gid; k < t.nt[q]; k += nthr) {
      double sn, cs;
      sincospi(-2.0 * (double)k / (double)t.nt[q], &sn, &cs);
      tab[t.off[q] + k] = make_float2((float)cs, (float)sn);
    }
}

// device address of the scratch on the CURRENT device (nullptr + g_cuda_msg on failure); once per device
unsigned char *noalloc_scratch_ptr() {
  int dev = -1;
  if (!cuda_ok(cudaGetDevice(&dev))) return nullptr;
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) { snprintf(g_cuda_msg, sizeof g_cuda_msg, "device ordinal %d not supported", dev); return nullptr; }
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_ptr[dev]) {
    void *p = nullptr;
    if (!cuda_ok(cudaGetSymbolAddress(&p, g_noalloc_scratch)) || !p) return nullptr;
    // the generic row kernel's dynamic shared memory limit: the same maximum volks_plan_create sets (per device)
    if (!cuda_ok(cudaFuncSetAttribute(k_row_fft, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024))) return nullptr;
    g_noalloc_ptr[dev] = (unsigned char *)p;
  }
  return g_noalloc_ptr[dev];
}

}  // namespace

extern "C" int volks_search_noalloc(const volks_params *p, const void *d_vis, volks_peak *d_peaks, volks_cand *d_cands,
                                    uint32_t cand_capacity, uint32_t *d_ncand, void *cuda_stream) {
  if (!p || !d_vis || !d_ncand || (!d_cands && cand_capacity > 0)) return VOLKS_EINVAL;
  if (p->nbl < 1 || p->nif < 1 || p->nap < 0 || p->nchan < 1) return VOLKS_EINVAL;
  if (p->nwidths < 1 || p->nwidths > VOLKS_MAX_WIDTHS || !p->width || !p->stride || !p->nt) return VOLKS_EINVAL;
  if (!is_pow2(p->nf) || p->nf < p->nchan || p->nf > 8192) return VOLKS_EINVAL;
  if (!(p->snr_thresh == p->snr_thresh)) return VOLKS_EINVAL;
  const long long npair = (long long)p->nbl * p->nif;
  Sched s;
  memset(&s, 0, sizeof s);
  s.nwidths = p->nwidths; s.nbl = p->nbl; s.nif = p->nif; s.nap = p->nap; s.nf = p->nf; s.log2nf = ilog2(p->nf);
  s.allif = 0; s.ngs = 1; s.snr_thresh = p->snr_thresh; s.dlo = -1; s.dhi = -1; s.dfirst = 0;
  NoAllocTables t;
  memset(&t, 0, sizeof t);
  t.nf = p->nf; t.nq = p->nwidths;
  long long per_pair = 0, tab_elems = p->nf;
  for (int q = 0; q < p->nwidths; ++q) {
    if (p->width[q] < 1 || p->stride[q] < 1 || !is_pow2(p->nt[q]) || p->nt[q] < p->width[q]) return VOLKS_EINVAL;
    if ((long long)p->nt[q] * p->nf > (1LL << 31)) return VOLKS_EINVAL;
    s.width[q] = p->width[q]; s.stride[q] = p->stride[q]; s.nt[q] = p->nt[q];
    s.nwin[q] = p->nap < p->width[q] ? 0 : (long long)(p->nap - p->width[q]) / p->stride[q] + 1;
    s.offc[q] = per_pair; s.offd[q] = npair * per_pair;
    per_pair += s.nwin[q];
    t.nt[q] = p->nt[q]; t.off[q] = tab_elems; tab_elems += p->nt[q];
    // k_col's grid (one thread per (window, rate residue, delay column)) must fit gridDim.x: checked before any launch
    const long double col_threads = (long double)npair * s.nwin[q] * (p->nt[q] / std::min(16, p->nt[q])) * p->nf;
    if (col_threads / 256 > 2147483000.0L) return VOLKS_ELIMIT;
  }
  s.per_pair = per_pair; s.nwin_total = per_pair * npair;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (s.nwin_total == 0) return cuda_ok(cudaMemsetAsync(d_ncand, 0, sizeof(uint32_t), st)) ? VOLKS_OK : VOLKS_ECUDA;

  // layout inside the static scratch (256-byte aligned pieces); everything beyond its stated size is refused
  const int pitch = p->nf >= 32 ? p->nf + 16 : p->nf, paired = p->nf >= 2 ? 1 : 0;
  const long long nfin = (s.nwin_total + FIN_THREADS * FIN_TILES - 1) / (FIN_THREADS * FIN_TILES);
  const long double need_ld = 1024.0L + 8.0L * tab_elems + 8.0L * s.nwin_total + 4.0L * npair * p->nap + 4.0L * nfin +
                              8.0L * npair * (long double)p->nap * pitch + 6 * 256.0L;
  if (need_ld > (long double)VOLKS_NOALLOC_SCRATCH_BYTES) return VOLKS_ELIMIT;
  size_t off = 0;
  const size_t off_sched = off; off = align_up(off + sizeof(Sched), 256);
  const size_t off_tab = off;   off = align_up(off + (size_t)tab_elems * sizeof(float2), 256);
  const size_t off_keys = off;  off = align_up(off + (size_t)s.nwin_total * sizeof(u64), 256);
  const size_t off_E = off;     off = align_up(off + (size_t)npair * p->nap * sizeof(float), 256);
  const size_t off_cnt = off;   off = align_up(off + (size_t)nfin * sizeof(uint32_t), 256);
  const size_t off_Y = off;     off = align_up(off + (size_t)npair * p->nap * pitch * sizeof(float2), 256);
  if (off > (size_t)VOLKS_NOALLOC_SCRATCH_BYTES) return VOLKS_ELIMIT;
  const long long GMAX = (1LL << 31) - 1;
  if (npair * p->nap > GMAX || nfin > GMAX) return VOLKS_ELIMIT;

  unsigned char *base = noalloc_scratch_ptr();      // the DEVICE address of g_noalloc_scratch on the current device
  if (!base) return VOLKS_ECUDA;
  Sched *d_sched = (Sched *)(base + off_sched);
  float2 *tab = (float2 *)(base + off_tab);
  u64 *keys = (u64 *)(base + off_keys);
  float *E = (float *)(base + off_E);
  uint32_t *cnt = (uint32_t *)(base + off_cnt);
  float2 *Y = (float2 *)(base + off_Y);

  // the scratch keeps the last call's contents: the keys meet in an atomicMax and must start at zero; the schedule,
  // tables, energies, counts and spectra are written in full before they are read
  if (!cuda_ok(cudaMemsetAsync(keys, 0, (size_t)s.nwin_total * sizeof(u64), st))) return VOLKS_ECUDA;
  k_noalloc_setup<<<(unsigned)std::min<long long>(64, (tab_elems + 255) / 256), 256, 0, st>>>(s, t, d_sched, tab);

  RowArgs ra;
  memset(&ra, 0, sizeof ra);
  ra.vis = (const float2 *)d_vis; ra.Y = Y; ra.E = E; ra.twf = tab; ra.row0 = 0; ra.nrows = npair * p->nap;
  ra.nchan = p->nchan; ra.nf = p->nf;
  ra.tpr = p->nf <= 512 ? std::max(1, std::min(32, p->nf / 4)) : std::min(512, p->nf / 4);
  ra.rows_per_cta = std::max(1, 256 / ra.tpr);
  ra.pitch = pitch; ra.paired = paired; ra.keys1 = nullptr; ra.per_pair = per_pair; ra.nap = p->nap; ra.stride1 = 1; ra.nwin1 = 0;
  ra.shift = nullptr; ra.nif = p->nif; ra.allif_nif = 0; ra.allif_nchan = 0; ra.psub = 1; ra.premod = nullptr; ra.cal = nullptr;
  ra.dlo = -1; ra.dhi = -1;
  const size_t row_smem = (size_t)2 * ra.rows_per_cta * p->nf * sizeof(float2) + (size_t)ra.rows_per_cta * 16 * sizeof(u64);
  const long long rblocks = (ra.nrows + ra.rows_per_cta - 1) / ra.rows_per_cta;
  if (ra.nrows > 0) k_row_fft<<<(unsigned)rblocks, ra.tpr * ra.rows_per_cta, row_smem, st>>>(ra);

  for (int q = 0; q < p->nwidths; ++q) {
    if (s.nwin[q] == 0) continue;
    ColArgs ca;
    const int L = std::min(16, p->nt[q]);
    ca.Y = Y; ca.keys = keys; ca.twt = tab + t.off[q]; ca.per_pair = per_pair; ca.offc = s.offc[q]; ca.pair0 = 0;
    ca.nap = p->nap; ca.nf = p->nf; ca.log2nf = s.log2nf; ca.w = p->width[q]; ca.stride = p->stride[q]; ca.nt = p->nt[q];
    ca.log2m = ilog2(p->nt[q] / L); ca.nwin = (int)s.nwin[q]; ca.pitch = pitch; ca.paired = paired;
    ca.total = ((npair * s.nwin[q]) << ca.log2m) * p->nf;
    switch (L) {
      case 1: launch_col<1>(ca, st); break;
      case 2: launch_col<2>(ca, st); break;
      case 4: launch_col<4>(ca, st); break;
      case 8: launch_col<8>(ca, st); break;
      default: launch_col<16>(ca, st); break;
    }
  }
  k_finalize<<<(unsigned)nfin, FIN_THREADS, 0, st>>>(d_sched, keys, E, (float4 *)d_peaks, cnt, nullptr, 0.f, nullptr);
  k_scan<<<1, 1024, 0, st>>>(cnt, nfin, d_ncand);
  k_scatter<<<(unsigned)nfin, FIN_THREADS, 0, st>>>(d_sched, keys, E, cnt, (CandOut *)d_cands, cand_capacity, nullptr, 0.f, nullptr, d_ncand);
  return cuda_ok(cudaGetLastError()) ? VOLKS_OK : VOLKS_ECUDA;
}
