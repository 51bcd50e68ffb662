/*
 * volks.h - C-ABI of the B200-native cross-spectrum fringe search (libvolks_b200.so).
 *
 * The hot path of the VOLKS2 single-pulse search (arXiv 2108.05602; PAPER.md = the paper text):
 * for every baseline, IF, window width and sliding window position, the window of complex
 * visibilities [w x nchan] is zero-padded to [Nt x Nf] and 2-D DFT'd (frequency -> delay, time ->
 * fringe rate), |.|^2 is taken, the peak and a noise statistic are found, an SNR is formed, and
 * the windows above threshold are compacted into an ordered candidate list.
 *
 *   - transform and its sign:  G = sum S e^{-i Phi}, Phi = 2 pi f dtau        PAPER.md:74-79 (Eq. 1)
 *   - FFT search with zero padding; the 2-D (delay x rate) geodetic scheme
 *   - step 5 "for each AP, FFT along the frequency axis"
 *   - step 6 "combine the FFTed APs along the time axis ... find the maximum" PAPER.md:143
 *   - windows of several sizes per baseline
 *   - "selected if its normalized power exceeds the threshold"; "SNR > 6"
 *   - "a single pulse is selected if it appears in at least 2 windows"
 *
 * Definition (DESIGN.md section "Path"): for window (bl, ifq, q, j), t0 = j*stride[q],
 *   F[r][d] = sum_{t<w_q} sum_{k<nchan} vis[bl][ifq][t0+t][k] exp(-2 pi i (r t/Nt_q + d k/Nf))
 *   P = |F|^2, P1 = max P, (r*, d*) = first argmax in row-major order (r major, d minor),
 *   noise = mean of P over the whole padded plane, snr = sqrt(P1/noise) (0 if noise == 0),
 *   candidate iff snr > snr_thresh (strict).
 *
 * All compute runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.  Plain pointers
 * and sizes only: every pointer below is marked HOST or DEVICE.  The caller owns every buffer;
 * volks_fringe_search never allocates.  The plan owns small device tables (twiddles, the width
 * schedule) allocated in volks_plan_create and freed in volks_plan_destroy.
 *
 * Errors: every int-returning call gives 0 (VOLKS_OK) or a negative code; nothing throws, exits or
 * prints.  Non-finite visibilities are a precondition violation (results unspecified, no crash).
 * Threads: a plan holds per-call state (profiling events, the copy stream of volks_search_host); use a
 * plan from one host thread at a time (several plans may run concurrently on different streams).
 * Determinism: identical inputs give bit-identical outputs run to run (the peak reduction is an
 * order-independent max over a total order; the compaction is an ordered scan).
 */
#ifndef VOLKS_H
#define VOLKS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define VOLKS_OK 0
#define VOLKS_EINVAL (-1)    /* bad dims, non-power-of-two pad, nt<w, nf<nchan, null pointer      */
#define VOLKS_ECUDA (-2)     /* CUDA allocation / launch failure (sticky error text: strerror)   */
#define VOLKS_ENOMEM (-3)    /* host allocation failure                                           */
#define VOLKS_EOVERFLOW (-4) /* returned by volks_window_match when capacity < number of pulses   */
#define VOLKS_ELIMIT (-5)    /* volks_search_noalloc: the problem needs more than its static scratch */

#define VOLKS_MAX_WIDTHS 16

/* Search parameters.  HOST memory, copied by volks_plan_create (arrays need not outlive it). */
typedef struct {
  int32_t nbl, nif, nap, nchan; /* vis is cf32[nbl][nif][nap][nchan], channel fastest, DEVICE      */
  int32_t nwidths;              /* 1..VOLKS_MAX_WIDTHS                                             */
  const int32_t *width;         /* HOST [nwidths] w_q >= 1 APs                  */
  const int32_t *stride;        /* HOST [nwidths] s_q >= 1 APs; partial windows are dropped        */
  const int32_t *nt;            /* HOST [nwidths] padded time size: power of two, >= w_q           */
  int32_t nf;                   /* padded frequency size: power of two, nchan <= nf <= 8192        */
                                /* (PAPER.md:83); larger: VOLKS_EINVAL                             */
  float snr_thresh;             /* candidate iff snr > snr_thresh              */
} volks_params;

/* One candidate = one window above threshold.  36 bytes, no padding. */
typedef struct {
  int32_t bl, ifq, wid, win, t0; /* wid = width index q; win = ordinal j; t0 = j*stride[q]         */
  int32_t rate_idx, delay_idx;   /* raw FFT bins r* in [0,Nt_q), d* in [0,Nf); upper half negative */
  float power, snr;              /* P1 and sqrt(P1/noise)                                          */
} volks_cand;

/* Dense per-window peak (optional output).  16 bytes. */
typedef struct {
  float power, snr;
  int32_t rate_idx, delay_idx;
} volks_peak;

/* One matched pulse of volks_window_match. */
typedef struct {
  volks_cand best;     /* max-snr member of the cluster (ties: first in canonical order)          */
  int32_t nwidths_hit; /* distinct width indices in the cluster                                    */
  int32_t t_begin, t_end; /* union AP extent [t_begin, t_end) of the cluster                       */
} volks_pulse;

/* Tuning and test options of a plan.  HOST memory; volks_options_init fills the defaults, then change what is
 * needed and pass it to volks_plan_create_opt / volks_plan_create_allif_opt (NULL = the defaults).  The library
 * reads no environment variables. */
typedef struct {
  int32_t struct_bytes;  /* sizeof(volks_options), set by volks_options_init; a mismatch is VOLKS_EINVAL            */
  int32_t full_index;    /* 0 (default): a search WITHOUT d_peaks finds the exact (rate, delay) bin only of the      */
                         /* windows that can be candidates (and may skip segments of narrow windows that cannot hold  */
                         /* one, see no_prune); candidates are bit-identical either way.  1: every window's peak in   */
                         /* every search - what volks_zscore_select needs from the search before it                  */
  int32_t force_generic; /* 1: the generic kernels (k_row_fft, k_col) for every width (the parity suite runs both)   */
  int32_t slide_seg;     /* windows per exactly restarted segment of the sliding kernel (default 256, >= 16)         */
  int32_t y_pad;         /* padding elements of a row of delay spectra (default 16; even, 0..1024)                   */
  int32_t chunk_mb;      /* MiB of delay spectra per chunk of (bl, ifq) pairs (default 4096; bounds the workspace)    */
  int32_t cf_wpc;        /* windows per CTA of the column-FFT kernels (default 128)                                  */
  int32_t cf2;           /* Nt = 256 / 512: 2 (default) 16-column strips, 1: 32-column, 4: 8-column, 0: k_colfft    */
  int32_t ai_waves;      /* f2: waves of 296 CTAs the window segments of k_allif are sized for (default 2)           */
  int32_t host_split;    /* volks_search_host copies 1/host_split of a plan chunk at a time (default 4)              */
  int32_t no_prune;      /* 1: switch off the exact pruning of the narrow stride-1 widths (full_index = 0 only): by   */
                         /* default a segment of windows whose amplitude-sum bound stays below the threshold in every */
                         /* delay column is not transformed at all (it cannot hold a candidate)                       */
  int32_t prune_seg;     /* windows per pruned segment (default 64; power of two, 16..4096)                          */
  int32_t delay_lo;      /* restricted delay search range ("the delay search range and the related FFT   */
  int32_t delay_hi;      /* size is configured for projected baselines shorter than 3000 km"): the peak is looked for */
                         /* in the bins delay_lo .. delay_hi of the padded delay axis only, wrapping through nf-1 -> 0 */
                         /* when delay_lo > delay_hi (delays around zero: {nf-m .. nf-1, 0 .. m}); the noise statistic */
                         /* stays the whole plane's.  Default 0, -1: the whole axis.  For an all-IF plan: bins of nfa.  */
} volks_options;
void volks_options_init(volks_options *o);

typedef struct volks_plan volks_plan; /* opaque */

/* Validate `p` (HOST), build the window schedule (per width: window count, kernel variant, grid
 * shape, canonical offsets) and upload the twiddle tables.  Uses the current CUDA device.
 * nap < w_q gives zero windows for that width, not an error.  *out receives the plan. */
int volks_plan_create(const volks_params *p, volks_plan **out);
int volks_plan_create_opt(const volks_params *p, const volks_options *opt, volks_plan **out);
int volks_plan_destroy(volks_plan *plan);

/* Sizes the caller needs.  All outputs HOST, each nullable.  nwin_per_width[q] counts windows of
 * ONE (bl, ifq) pair: floor((nap-w_q)/s_q)+1; nwin_total = nbl*nif*sum_q nwin_per_width[q]. */
int volks_plan_query(const volks_plan *plan, size_t *workspace_bytes, int64_t *nwin_per_width,
                     int64_t *nwin_total);

/* The hot path.  Asynchronous: every kernel is enqueued on `cuda_stream` (a cudaStream_t; NULL =
 * legacy default stream); results are valid after the stream is synchronised.
 *   d_vis        DEVICE cf32[nbl][nif][nap][nchan], read-only, 8-byte aligned
 *   d_workspace  DEVICE scratch of >= workspace_bytes (256-byte aligned); contents undefined after
 *   d_peaks      DEVICE volks_peak[nwin_total] or NULL.  Dense layout:
 *                d_peaks[off_q + (bl*nif + ifq)*nwin_q + j], off_q = nbl*nif*sum_{q'<q} nwin_q'
 *   d_cands      DEVICE volks_cand[cand_capacity]; candidates in canonical order (bl, ifq, q, j)
 *   d_ncand      DEVICE uint32: the TRUE total number of candidates; if it exceeds cand_capacity
 *                only the first cand_capacity candidates (canonical order) were written
 * Returns VOLKS_OK, VOLKS_EINVAL (null plan/vis/workspace/ncand, or null d_cands with capacity>0)
 * or VOLKS_ECUDA (a launch failed). */
int volks_fringe_search(const volks_plan *plan, const void *d_vis, void *d_workspace,
                        volks_peak *d_peaks, volks_cand *d_cands, uint32_t cand_capacity,
                        uint32_t *d_ncand, void *cuda_stream);

/* The same search on DEDISPERSED data (step 4 of the paper: "for each frequency
 * point ... a specific time shift"), fused into the slab load: element (t, k) of pair (bl, ifq) is
 * taken from AP t + d_shift[ifq*nchan + k], and is zero where that falls outside [0, nap).
 *   d_shift  DEVICE int32[nif][nchan] AP offsets for one DM (volks_dm_shifts fills a HOST table to
 *            upload), or NULL = volks_fringe_search.  One call per DM value; d_vis is never modified.
 * Everything else as volks_fringe_search. */
int volks_fringe_search_dd(const volks_plan *plan, const void *d_vis, const int32_t *d_shift,
                           void *d_workspace, volks_peak *d_peaks, volks_cand *d_cands,
                           uint32_t cand_capacity, uint32_t *d_ncand, void *cuda_stream);

/* f2 - VOLKS2's own search: ONE delay across all IFs (Eq. 1), rate 0 only.  For every
 * baseline, width and window the per-AP all-IF delay spectra (one zero-padded FFT over the whole band
 * of nif*nchan frequency points per AP; IFs contiguous in frequency, A21) are summed
 * coherently over the window's APs (step 6) and the maximum along the delay axis is found:
 *   A[d] = sum_{t<w} sum_{m<nif*nchan} band[t0+t][m] exp(-2 pi i m d/nfa),  m = n*nchan + j,
 *   P = |A|^2, (P1, d*) first argmax, noise = mean_d P, snr = sqrt(P1/noise), candidate iff snr > snr_thresh.
 * volks_plan_create_allif reads nbl, nif, nap, nchan, nwidths, width[], stride[], snr_thresh and
 * nf = nfa (power of two, 64 <= nfa <= 32768, nif*nchan <= min(nfa, 8192): beyond 8192 the transform is
 * computed as nfa/8192 interleaved 8192-point transforms of the pre-modulated band, which must fit one of
 * them; VOLKS_EINVAL otherwise); nt[] is ignored (may be NULL).
 * volks_allif_search takes the same buffers as volks_fringe_search_dd (d_shift: dedispersion, or NULL);
 * sizes from volks_plan_query (nwin_total = nbl * sum_q nwin_q).  Records: ifq = -1, rate_idx = 0,
 * delay_idx in [0, nfa); canonical order (bl, q, j); dense peaks d_peaks[off_q + bl*nwin_q + j].
 * volks_zscore_select, volks_window_match (ifq = -1 groups a baseline) and volks_baseline_match apply
 * to its results unchanged. */
int volks_plan_create_allif(const volks_params *p, volks_plan **out);
int volks_plan_create_allif_opt(const volks_params *p, const volks_options *opt, volks_plan **out);
int volks_allif_search(const volks_plan *plan, const void *d_vis, const int32_t *d_shift, void *d_workspace,
                       volks_peak *d_peaks, volks_cand *d_cands, uint32_t cand_capacity,
                       uint32_t *d_ncand, void *cuda_stream);

/* The same searches on a HOST slab (pinned memory recommended), for slabs that are produced on the host
 * or do not fit the device: the slab is copied chunk by chunk (the (bl, ifq) pairs - baselines for an
 * all-IF plan - of a quarter of an internal chunk at a time) into the two halves of `d_stage` on an internal copy
 * stream, each copy overlapped with the kernels of the previous chunk; the result is identical to the
 * device-slab calls.  Works with both plan kinds (volks_plan_create / volks_plan_create_allif).
 *   h_vis    HOST cf32[nbl][nif][nap][nchan]; must stay valid until `cuda_stream` has run the call
 *   d_stage  DEVICE scratch of 2 * stage_bytes (volks_plan_query_host), 256-byte aligned
 * Other arguments as volks_fringe_search_dd. */
int volks_plan_query_host(const volks_plan *plan, size_t *stage_bytes);
int volks_search_host(const volks_plan *plan, const void *h_vis, void *d_stage, const int32_t *d_shift,
                      void *d_workspace, volks_peak *d_peaks, volks_cand *d_cands, uint32_t cand_capacity,
                      uint32_t *d_ncand, void *cuda_stream);

/* Across-window normalised power (SURVEY 8(f) f4 - the other reading of PAPER.md:196 "for the time
 * segments series of given window size, a single pulse is selected if its normalized power exceeds
 * the threshold, which is set to 3").  A second pass over the results the LAST volks_fringe_search[_dd]
 * left in `d_workspace` (same plan, workspace untouched since): per (bl, ifq, width) the window peak
 * powers P1_j are normalised across windows, z_j = (P1_j - mean)/std (population std; z = 0 if
 * std = 0); candidate iff z_j > z_thresh.  Outputs as volks_fringe_search, except that the `snr`
 * field of candidates (and of d_peaks, if given) carries z.  Asynchronous on `cuda_stream`.
 * The search before it must have kept every window's exact index: a plan created with volks_options.full_index
 * = 1, or a search that wrote d_peaks; VOLKS_EINVAL otherwise. */
int volks_zscore_select(const volks_plan *plan, void *d_workspace, float z_thresh, volks_peak *d_peaks,
                        volks_cand *d_cands, uint32_t cand_capacity, uint32_t *d_ncand, void *cuda_stream);

/* Initial calibration (step 3 of the paper; the last two terms of Eq. 1, PAPER.md:74-79:
 * Phi = ... + 2 pi f_j dtau0^n + dphi0^n with f_j the j-th frequency point inside IF n, values per IF
 * and baseline), fused into the slab load: every later search with this plan multiplies
 * vis[bl][ifq][t][k] by d_cal[bl][ifq][k] as it is read.
 *   d_cal  DEVICE cf32[nbl][nif][nchan] (the SOURCE shape, also for an all-IF plan), or NULL to switch
 *          it off.  The plan keeps the pointer, not a copy: the table must outlive the searches.
 * volks_cal_phasors (HOST) fills a table with e^{-i (2 pi j chan_hz delay_s[p] + phase_rad[p])},
 * p = bl*nif + ifq, j < nchan: cal is HOST float[2*npair*nchan] (re, im). */
int volks_plan_set_cal(volks_plan *plan, const void *d_cal);
int volks_cal_phasors(const double *delay_s, const double *phase_rad, int32_t npair, int32_t nchan,
                      double chan_hz, float *cal);

/* HOST helper: integer AP shift of every frequency point for dispersion measure `dm` [pc cm^-3]:
 * shift = round(4.148808e-3 s * dm * (f_GHz^-2 - fref_GHz^-2) / ap_seconds) (the textbook cold-plasma
 * delay; the paper states no formula - DESIGN.md R3).  f_chan_mhz, shift: HOST [n]. */
int volks_dm_shifts(double dm, const double *f_chan_mhz, int32_t n, double f_ref_mhz, double ap_seconds,
                    int32_t *shift);

/* Per-baseline multi-window match (reading A13).  HOST call on HOST
 * arrays (integer work on a list of at most a few thousand records).  Within one (bl, ifq),
 * candidates whose AP intervals [t0, t0+width[wid]) overlap are linked; connected components are
 * clusters; a cluster with >= min_widths distinct width indices gives one volks_pulse.  Output is
 * ordered by the canonical position of `best`.  `cands` must be in canonical order; `width` is
 * the HOST [nwidths] width table the candidates' `wid` fields index (needs no plan and no GPU).
 * *nout receives the number of pulses found; returns VOLKS_EOVERFLOW if it exceeds `capacity`
 * (the first `capacity` are written). */
int volks_window_match(const volks_cand *cands, uint32_t ncand, const int32_t *width, int32_t nwidths,
                       int32_t min_widths, volks_pulse *out, uint32_t capacity, uint32_t *nout);

/* One cross-baseline detection of volks_baseline_match. */
typedef struct {
  volks_pulse best;       /* max-snr pulse of the cluster (ties: first in input order)             */
  int32_t nbaselines;     /* distinct `bl` values in the cluster                                     */
  int32_t t_begin, t_end; /* union AP extent [t_begin, t_end) of the cluster                         */
} volks_detection;

/* Multi-baseline cross-match ("A single pulse is identified if it is
 * detected with at least 5 baselines"; reading A19).  HOST call on HOST arrays: the pulses
 * of volks_window_match for ALL (bl, ifq) are clustered by overlap of their AP extents
 * [t_begin, t_end) (connected components); a cluster seen on >= min_baselines distinct baselines
 * gives one volks_detection.  Output ordered by t_begin (ties: position of `best` in the input).
 * *nout = number found; VOLKS_EOVERFLOW if it exceeds `capacity` (the first `capacity` are written). */
int volks_baseline_match(const volks_pulse *pulses, uint32_t npulse, int32_t min_baselines,
                         volks_detection *out, uint32_t capacity, uint32_t *nout);

/* HOST helper: signed physical units from raw bins (upper half of each axis is negative):
 * rate_hz = r_signed/(nt*ap_seconds), delay_s = d_signed/(nf*chan_hz); nt = Nt_q of the width. */
int volks_bin_to_physical(int32_t nt, int32_t nf, int32_t rate_idx, int32_t delay_idx,
                          double ap_seconds, double chan_hz, double *rate_hz, double *delay_s);

/* Number of kernels one volks_fringe_search (without d_peaks) enqueues (for launch accounting). */
int volks_plan_launch_count(const volks_plan *plan);

/* Optional per-launch timing for measurement (bench.py's roofline leg).  When enabled, every kernel
 * volks_fringe_search enqueues is bracketed by CUDA events recorded on the launching stream.
 * volks_plan_profile_read waits for the most recent call's events and returns, per launch in
 * launch order, its kind (VOLKS_K_*), its width index (or -1) and its duration in milliseconds.
 * HOST outputs; *n receives the number of launches (only min(n, capacity) entries are written). */
#define VOLKS_K_ROW 1      /* slab load + zero-pad + delay FFT (+ per-AP energy)                    */
#define VOLKS_K_COL 2      /* rate transform + power + argmax of one width                         */
#define VOLKS_K_FINALIZE 3 /* SNR, dense peaks, threshold count                                    */
#define VOLKS_K_SCAN 4     /* scan of block counts                                                 */
#define VOLKS_K_SCATTER 5  /* ordered candidate scatter                                            */
#define VOLKS_K_SLIDE 6    /* stride-1 widths: sliding-sum rate transform + power + argmax          */
#define VOLKS_K_COLFFT 7   /* any stride, Nt 32..512: two-pass shared-memory column FFT + argmax    */
#define VOLKS_K_ALLIF 8    /* f2: all-IF rate-0 window sums + argmax + noise                          */
#define VOLKS_K_FIXUP 9    /* exact re-evaluation of the sliding widths' outlier windows               */
#define VOLKS_K_WINTHR 10  /* per-window pre-thresholds of the candidates-only index mode              */
#define VOLKS_K_BOUND 11   /* amplitude-sum bound: which segments of the narrow widths can hold candidates */
#define VOLKS_K_SFOLD 14   /* candidates-only mode, wide stride-1 widths: folded sliding sum -> hit masks            */
#define VOLKS_K_SFOLD_EVAL 15 /* ... exact transform of the flagged (window, rate residue, 64-column tile)s        */
#define VOLKS_K_COLEVAL 13 /* one width by the definition in the (window, column) pairs the bound leaves          */
#define VOLKS_K_RECOVER 12 /* peak bin of the stride-1 windows (w >= 16) by exact re-evaluation of one tile */
int volks_plan_profile(volks_plan *plan, int enable);
int volks_plan_profile_read(const volks_plan *plan, int32_t capacity, int32_t *kind, int32_t *wid,
                            float *ms, int32_t *n);

/* Measurement helper (not on the search path): the FP32 FMA issue peak of the current device at the clocks it
 * runs at - the denominator of bench.py's "alu" roofline (SURVEY 8(d) "the builder must
 * measure it").  Launches `repeats` (1..1000) kernels of dependent-free FFMA chains (64 resident warps per SM,
 * about 20 ms each on B200) on `cuda_stream`, times each with CUDA events and SYNCHRONISES; allocates and frees a
 * small device buffer.  HOST outputs: *tflops_best = fastest launch, *tflops_mean, *ms_per_launch (the last two
 * nullable).  Counts 2 flop per FMA per thread. */
int volks_measure_fp32_peak(int32_t repeats, double *tflops_best, double *tflops_mean, double *ms_per_launch,
                            void *cuda_stream);

/* The search for callers that CANNOT ALLOCATE (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): one call, no plan, no workspace.  It computes what volks_fringe_search computes (the
 * definition at the top of this file: every window's peak, snr, the ordered candidate list) with the general
 * kernels (k_row_fft, k_col, finalize / scan / scatter), and keeps EVERY intermediate - window schedule, twiddle
 * tables, per-window keys, per-AP energies, block counts, the delay spectra - in one file-scope device array of
 * VOLKS_NOALLOC_SCRATCH_BYTES (32 MiB) that every GPU loading the library holds until exit.  The call makes no
 * cudaMalloc / cudaFree and no allocating library call; it only enqueues a memset and kernels on `cuda_stream`
 * (asynchronous: results are valid after the stream is synchronised) - the first call on a device also looks up the
 * array's device address (cudaGetSymbolAddress) and raises one kernel's shared-memory limit.
 *   p            HOST search parameters, as for volks_plan_create (nf <= 8192; read during the call only)
 *   d_vis        DEVICE cf32[nbl][nif][nap][nchan], read-only
 *   d_peaks      DEVICE volks_peak[nwin_total] in the dense layout of volks_fringe_search, or NULL
 *   d_cands      DEVICE volks_cand[cand_capacity], canonical order; d_ncand DEVICE uint32, the TRUE total
 * Size limit: 1 KiB + 8 (nf + sum_q nt_q) + 8 nwin_total + 4 nbl nif nap + 8 nbl nif nap pitch (pitch = nf + 16 for
 * nf >= 32, else nf) + small change must fit the 32 MiB; larger problems return VOLKS_ELIMIT before anything is
 * enqueued (BASELINE.json configs 0 and 1 fit; use a plan for the large ones).  It always searches the whole delay
 * axis and every window's exact peak (no options).
 * SHARED STATE: every call on a device uses the same array, which keeps the last call's contents (the call clears
 * what must start at zero).  Two calls that overlap on the GPU - different streams, or different host threads
 * without a common stream order - RACE on it; calls on one stream are ordered and safe.
 * Returns VOLKS_OK, VOLKS_EINVAL (bad parameters / null pointers), VOLKS_ELIMIT, or VOLKS_ECUDA. */
#define VOLKS_NOALLOC_SCRATCH_BYTES (32u << 20)
int volks_search_noalloc(const volks_params *p, const void *d_vis, volks_peak *d_peaks, volks_cand *d_cands,
                         uint32_t cand_capacity, uint32_t *d_ncand, void *cuda_stream);

const char *volks_strerror(int code);
int volks_version(void);

#ifdef __cplusplus
}
#endif
#endif /* VOLKS_H */
