/*
 * volks_oracle.c — float64 CPU oracle for the VOLKS2 2-D fringe search hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing on the product path (paper_2108_05602_b200/) may
 * include, link, import or execute this file; only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs do.  It shares no code, table or
 * constant with the CUDA path.
 *
 * What it computes (PAPER.md = /root/reference/PAPER.md, arXiv 2108.05602):
 *   - the search function is a sum of visibilities times e^{-i Phi}, Phi = 2 pi f dtau
 *     (Eq. 1)  => forward transform with NEGATIVE exponent;
 *   - "delay search is carried out with FFT ... padding is required"; the "standard geodetic
 *     fitting scheme conducts 2-D FFT" => zero-padded 2-D DFT, delay x rate;
 *   - step 5 "For each AP, carry out FFT along the frequency axis" and step 6
 *     "combining the FFTed APs along the time axis ... find out the maximum amplitude"
 *      => rows (per AP) first, then the time axis, then the maximum;
 *   - "normalized power exceeds the threshold" / "SNR > 6":
 *     DESIGN.md reading A3: snr = sqrt(P1 / mean(P)) over the whole padded plane.
 *
 * For window (bl, ifq, q, j), t0 = j*stride_q, W = vis[bl][ifq][t0:t0+w_q][0:nchan]:
 *   F[r][d] = sum_{t<w} sum_{k<nchan} W[t][k] exp(-2 pi i (r t/Nt + d k/Nf)),  r<Nt, d<Nf
 *   P = |F|^2 ; (P1, idx1) = max and FIRST argmax in row-major order (r major, d minor);
 *   (P2, idx2) = second largest value and its first index; S1 = sum P;
 *   noise = S1/(Nt Nf); snr = sqrt(P1/noise) (0 if noise == 0).
 *
 * Three forms of the same sum (all float64, no FFT library):
 *   mode 0  direct   : the double sum written out, O(Nt Nf w nchan)   (tiny planes)
 *   mode 1  fft      : textbook recursive radix-2 FFT on the explicitly zero-padded plane,
 *                      rows then columns, per window independently
 *   mode 2  cached   : each AP's padded row FFT computed once per (bl, ifq) and reused by
 *                      every window/width (the separable sum in another order, PAPER.md:133
 *                      vs 143); used for full sweeps and for timing.
 * Parity pins live in tests/test_oracle_pins.py (closed forms P1-P14 of DESIGN.md).
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o libvolks_oracle.so volks_oracle.c -lm
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

typedef struct {
  double p1;    /* largest power                         */
  double p2;    /* second largest power                  */
  double s1;    /* sum of power over the padded plane    */
  double snr;   /* sqrt(p1 / (s1/(Nt*Nf))), 0 if s1 == 0 */
  int64_t idx1; /* first row-major index of p1 (r*Nf+d)  */
  int64_t idx2; /* first row-major index of p2           */
} vo_peak;

static const double VO_PI = 3.14159265358979323846264338327950288;

static int is_pow2(int n) { return n >= 1 && (n & (n - 1)) == 0; }

/* Textbook recursive radix-2 decimation-in-time FFT, forward (negative exponent).
 * x is read with the given stride; out receives n contiguous values.  tw[k] =
 * exp(-2 pi i k / ntw) for k < ntw/2 is a table for the LARGEST size in use; a size-n
 * transform uses every (ntw/n)-th entry. */
static void fft_rec(const cplx *x, int n, int stride, cplx *out, const cplx *tw, int ntw) {
  if (n == 1) { out[0] = x[0]; return; }
  int h = n / 2;
  fft_rec(x, h, 2 * stride, out, tw, ntw);               /* even samples */
  fft_rec(x + stride, h, 2 * stride, out + h, tw, ntw);  /* odd samples  */
  int step = ntw / n;
  for (int k = 0; k < h; ++k) {
    cplx e = out[k], o = tw[k * step] * out[k + h];
    out[k] = e + o;
    out[k + h] = e - o;
  }
}

static cplx *make_twiddles(int n) {
  int h = n / 2 > 0 ? n / 2 : 1;
  cplx *tw = (cplx *)malloc(sizeof(cplx) * (size_t)h);
  if (!tw) return NULL;
  for (int k = 0; k < h; ++k) {
    double a = -2.0 * VO_PI * (double)k / (double)n;
    tw[k] = cos(a) + I * sin(a);
  }
  return tw;
}

/* Scan a plane of powers in row-major order: max / first argmax, runner-up, sum. */
static void scan_begin(vo_peak *pk) {
  pk->p1 = -1.0; pk->p2 = -1.0; pk->idx1 = -1; pk->idx2 = -1; pk->s1 = 0.0; pk->snr = 0.0;
}
static inline void scan_bin(vo_peak *pk, double p, int64_t i) {
  pk->s1 += p;
  if (p > pk->p1) { pk->p2 = pk->p1; pk->idx2 = pk->idx1; pk->p1 = p; pk->idx1 = i; }
  else if (p > pk->p2) { pk->p2 = p; pk->idx2 = i; }
}
/* Restricted delay search range ("the delay search range and the related FFT size is configured for
 * projected baselines shorter than 3000 km"; reading A14): the maximum is looked for only in the delay
 * bins dlo, dlo+1, ..., dhi of the padded axis, wrapping through nf-1 -> 0 when dlo > dhi (delays around zero are
 * {nf-m .. nf-1, 0 .. m}); the noise statistic S1 stays the sum over the WHOLE plane.  dlo < 0: whole axis. */
static inline int delay_in_range(int d, int dlo, int dhi) {
  if (dlo < 0) return 1;
  return dlo <= dhi ? (d >= dlo && d <= dhi) : (d >= dlo || d <= dhi);
}
/* a bin outside the range still counts for S1 */
static inline void scan_bin_out(vo_peak *pk, double p) { pk->s1 += p; }
static void scan_end(vo_peak *pk, int nt, int nf) {
  double noise = pk->s1 / ((double)nt * (double)nf);
  pk->snr = noise > 0.0 ? sqrt(pk->p1 / noise) : 0.0;
}

/* mode 0: the definition.  win = float32 [w][nchan][2] with row stride `ld` complex samples.
 * If plane != NULL it receives F as [nt][nf] complex128. */
static void window_direct(const float *win, int64_t ld, int w, int nchan, int nt, int nf,
                          cplx *plane, vo_peak *pk, int dlo, int dhi) {
  scan_begin(pk);
  for (int r = 0; r < nt; ++r)
    for (int d = 0; d < nf; ++d) {
      cplx acc = 0.0;
      for (int t = 0; t < w; ++t)
        for (int k = 0; k < nchan; ++k) {
          const float *s = win + 2 * ((int64_t)t * ld + k);
          cplx v = (double)s[0] + I * (double)s[1];
          double ph = -2.0 * VO_PI * ((double)r * (double)t / (double)nt +
                                      (double)d * (double)k / (double)nf);
          acc += v * (cos(ph) + I * sin(ph));
        }
      if (plane) plane[(int64_t)r * nf + d] = acc;
      if (delay_in_range(d, dlo, dhi)) scan_bin(pk, creal(acc) * creal(acc) + cimag(acc) * cimag(acc), (int64_t)r * nf + d);
      else scan_bin_out(pk, creal(acc) * creal(acc) + cimag(acc) * cimag(acc));
    }
  scan_end(pk, nt, nf);
}

/* Zero-padded plane by FFT: rows (frequency -> delay) then columns
 * (time -> fringe rate).  plane is [nt][nf] complex128 scratch/output. */
static void plane_fft(const float *win, int64_t ld, int w, int nchan, int nt, int nf,
                      cplx *plane, const cplx *twf, const cplx *twt) {
  cplx *rowin = (cplx *)calloc((size_t)(nf > nt ? nf : nt), sizeof(cplx));
  cplx *rowout = (cplx *)malloc(sizeof(cplx) * (size_t)(nf > nt ? nf : nt));
  for (int t = 0; t < nt; ++t) {
    if (t < w) {
      for (int k = 0; k < nf; ++k) {
        if (k < nchan) {
          const float *s = win + 2 * ((int64_t)t * ld + k);
          rowin[k] = (double)s[0] + I * (double)s[1];
        } else rowin[k] = 0.0;
      }
      fft_rec(rowin, nf, 1, plane + (int64_t)t * nf, twf, nf);
    } else {
      for (int d = 0; d < nf; ++d) plane[(int64_t)t * nf + d] = 0.0;
    }
  }
  for (int d = 0; d < nf; ++d) {
    for (int t = 0; t < nt; ++t) rowin[t] = plane[(int64_t)t * nf + d];
    fft_rec(rowin, nt, 1, rowout, twt, nt);
    for (int r = 0; r < nt; ++r) plane[(int64_t)r * nf + d] = rowout[r];
  }
  free(rowin); free(rowout);
}

static void scan_plane(const cplx *plane, int nt, int nf, vo_peak *pk, int dlo, int dhi) {
  scan_begin(pk);
  for (int64_t i = 0; i < (int64_t)nt * nf; ++i) {
    double re = creal(plane[i]), im = cimag(plane[i]);
    if (delay_in_range((int)(i % nf), dlo, dhi)) scan_bin(pk, re * re + im * im, i);
    else scan_bin_out(pk, re * re + im * im);
  }
  scan_end(pk, nt, nf);
}

/* ---- exported: one window ------------------------------------------------------------ */

/* vo_window: fringe-search ONE window.  win = float32 interleaved (re,im), [w][ld] complex
 * samples of which the first nchan per row are used.  mode 0 = direct sum, 1 = FFT.
 * plane (nullable) receives F as [nt][nf] complex128.  Returns 0, or -1 on bad arguments. */
int vo_window(int mode, const float *win, int64_t ld, int w, int nchan, int nt, int nf,
              double *plane_out, vo_peak *pk, int dlo, int dhi) {
  if (!win || !pk || w < 1 || nchan < 1 || nt < w || nf < nchan) return -1;
  if (dlo >= nf || dhi >= nf || (dlo >= 0 && dhi < 0)) return -1;
  if (mode == 0) {
    window_direct(win, ld, w, nchan, nt, nf, (cplx *)plane_out, pk, dlo, dhi);
    return 0;
  }
  if (!is_pow2(nt) || !is_pow2(nf)) return -1;
  cplx *twf = make_twiddles(nf), *twt = make_twiddles(nt);
  cplx *plane = plane_out ? (cplx *)plane_out : (cplx *)malloc(sizeof(cplx) * (size_t)nt * nf);
  plane_fft(win, ld, w, nchan, nt, nf, plane, twf, twt);
  scan_plane(plane, nt, nf, pk, dlo, dhi);
  if (!plane_out) free(plane);
  free(twf); free(twt);
  return 0;
}

/* ---- exported: a whole search ----------------------------------------------------------
 * vis = float32 interleaved cf32 [nbl][nif][nap][nchan], channel fastest.
 * Window (bl, ifq, q, j): t0 = j*stride[q]; nwin_q = floor((nap - w_q)/s_q) + 1 (0 if nap<w_q)
 * (A5: partial windows dropped).
 * Output order is CANONICAL: (bl, ifq, q, j), i.e. index
 *     c = (bl*nif + ifq) * sum_q nwin_q + sum_{q'<q} nwin_q' + j.
 * If nsel >= 0, only the canonical indices sel[0..nsel) are computed and out[i] corresponds to
 * sel[i]; if nsel < 0 all windows are computed and out has sum-over-everything entries.
 * mode 0 direct, 1 fft (per window independently), 2 cached rows.
 * nthreads <= 0: OpenMP default.  Returns threads used (>=1) or -1 on bad arguments. */
static int64_t nwin_of(int nap, int w, int s) { return nap < w ? 0 : (int64_t)(nap - w) / s + 1; }

int vo_search(const float *vis, int nbl, int nif, int nap, int nchan, int nwidths,
              const int32_t *width, const int32_t *stride, const int32_t *nt, int nf, int mode,
              const int64_t *sel, int64_t nsel, vo_peak *out, int nthreads, int dlo, int dhi) {
  if (!vis || !out || nbl < 1 || nif < 1 || nap < 0 || nchan < 1 || nwidths < 1) return -1;
  if (dlo >= nf || dhi >= nf || (dlo >= 0 && dhi < 0)) return -1;
  if (nf < nchan || (mode != 0 && !is_pow2(nf))) return -1;
  int ntmax = 1;
  int64_t per_pair = 0;
  for (int q = 0; q < nwidths; ++q) {
    if (width[q] < 1 || stride[q] < 1 || nt[q] < width[q]) return -1;
    if (mode != 0 && !is_pow2(nt[q])) return -1;
    if (nt[q] > ntmax) ntmax = nt[q];
    per_pair += nwin_of(nap, width[q], stride[q]);
  }
  int64_t npair = (int64_t)nbl * nif;
  int64_t total = nsel >= 0 ? nsel : npair * per_pair;
  int used = 1;
#ifdef _OPENMP
  if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
  cplx *twf = mode != 0 ? make_twiddles(nf) : NULL;

  if (mode == 2 && nsel < 0) {
    /* cached rows: per (bl, ifq) compute each AP's padded row FFT once, then
     * for every width and window the rate FFT of each delay column. */
    for (int64_t pair = 0; pair < npair; ++pair) {
      const float *pv = vis + 2 * pair * (int64_t)nap * nchan;
      cplx *Y = (cplx *)malloc(sizeof(cplx) * (size_t)(nap > 0 ? nap : 1) * nf);
#pragma omp parallel
      {
#ifdef _OPENMP
#pragma omp single
        used = omp_get_num_threads();
#endif
        cplx *rowin = (cplx *)malloc(sizeof(cplx) * (size_t)nf);
#pragma omp for schedule(static)
        for (int t = 0; t < nap; ++t) {
          for (int k = 0; k < nf; ++k) {
            if (k < nchan) {
              const float *s = pv + 2 * ((int64_t)t * nchan + k);
              rowin[k] = (double)s[0] + I * (double)s[1];
            } else rowin[k] = 0.0;
          }
          fft_rec(rowin, nf, 1, Y + (int64_t)t * nf, twf, nf);
        }
        free(rowin);
      }
      int64_t off = 0;
      for (int q = 0; q < nwidths; ++q) {
        int w = width[q], s = stride[q], ntq = nt[q];
        int64_t nw = nwin_of(nap, w, s);
        cplx *twt = make_twiddles(ntq);
#pragma omp parallel
        {
          cplx *col = (cplx *)malloc(sizeof(cplx) * (size_t)ntq);
          cplx *fc = (cplx *)malloc(sizeof(cplx) * (size_t)ntq);
          double *P = (double *)malloc(sizeof(double) * (size_t)ntq * nf);
#pragma omp for schedule(dynamic, 16)
          for (int64_t j = 0; j < nw; ++j) {
            int64_t t0 = j * s;
            for (int d = 0; d < nf; ++d) {
              for (int t = 0; t < ntq; ++t) col[t] = t < w ? Y[(t0 + t) * nf + d] : 0.0;
              fft_rec(col, ntq, 1, fc, twt, ntq);
              for (int r = 0; r < ntq; ++r) {
                double re = creal(fc[r]), im = cimag(fc[r]);
                P[(int64_t)r * nf + d] = re * re + im * im;
              }
            }
            vo_peak pk;
            scan_begin(&pk);
            for (int64_t i = 0; i < (int64_t)ntq * nf; ++i) {
              if (delay_in_range((int)(i % nf), dlo, dhi)) scan_bin(&pk, P[i], i);
              else scan_bin_out(&pk, P[i]);
            }
            scan_end(&pk, ntq, nf);
            out[pair * per_pair + off + j] = pk;
          }
          free(col); free(fc); free(P);
        }
        free(twt);
        off += nw;
      }
      free(Y);
    }
    free(twf);
    return used;
  }

  /* per-window independent evaluation (modes 0, 1; mode 2 with a selection falls back to 1:
   * the same separable sum, DESIGN.md oracle forms) */
  int wmode = mode == 0 ? 0 : 1;
#pragma omp parallel
  {
#ifdef _OPENMP
#pragma omp single
    used = omp_get_num_threads();
#endif
    cplx *plane = wmode ? (cplx *)malloc(sizeof(cplx) * (size_t)ntmax * nf) : NULL;
#pragma omp for schedule(dynamic, 4)
    for (int64_t i = 0; i < total; ++i) {
      int64_t c = nsel >= 0 ? sel[i] : i;
      int64_t pair = c / per_pair, rem = c % per_pair;
      int q = 0;
      for (; q < nwidths; ++q) {
        int64_t nw = nwin_of(nap, width[q], stride[q]);
        if (rem < nw) break;
        rem -= nw;
      }
      int64_t t0 = rem * stride[q];
      const float *win = vis + 2 * ((pair * nap + t0) * (int64_t)nchan);
      if (wmode == 0) {
        window_direct(win, nchan, width[q], nchan, nt[q], nf, NULL, &out[i], dlo, dhi);
      } else {
        cplx *twt = make_twiddles(nt[q]);
        plane_fft(win, nchan, width[q], nchan, nt[q], nf, plane, twf, twt);
        scan_plane(plane, nt[q], nf, &out[i], dlo, dhi);
        free(twt);
      }
    }
    free(plane);
  }
  free(twf);
  return used;
}

/* ---- exported: per-baseline multi-window match (A13) ----------
 * cands: n records (bl, ifq, wid, win, t0, w) in canonical order with snr[].  Within one
 * (bl, ifq), two candidates are linked when their AP intervals [t0, t0+w) overlap; clusters
 * are the connected components (O(n^2) pair test + union-find).  A cluster is kept when it
 * contains >= min_widths DISTINCT width indices ("appears in at least 2 windows").
 * Output per kept cluster, ordered by the canonical index of its representative:
 *   rep[i] = index of the max-snr member (ties -> lowest canonical position),
 *   nhit[i] = distinct widths, tb[i], te[i] = union extent [tb, te).
 * Returns number of clusters kept (<= n). */
static int64_t uf_find(int64_t *p, int64_t x) { while (p[x] != x) { p[x] = p[p[x]]; x = p[x]; } return x; }

int64_t vo_window_match(int64_t n, const int32_t *bl, const int32_t *ifq, const int32_t *wid,
                        const int32_t *t0, const int32_t *w, const double *snr, int min_widths,
                        int64_t *rep, int32_t *nhit, int32_t *tb, int32_t *te) {
  if (n <= 0) return 0;
  int64_t *par = (int64_t *)malloc(sizeof(int64_t) * (size_t)n);
  for (int64_t i = 0; i < n; ++i) par[i] = i;
  for (int64_t i = 0; i < n; ++i)
    for (int64_t k = i + 1; k < n; ++k) {
      if (bl[i] != bl[k] || ifq[i] != ifq[k]) continue;
      if (t0[i] < t0[k] + w[k] && t0[k] < t0[i] + w[i]) {
        int64_t a = uf_find(par, i), b = uf_find(par, k);
        if (a != b) par[a > b ? a : b] = a > b ? b : a;
      }
    }
  int64_t nout = 0;
  char *done = (char *)calloc((size_t)n, 1);
  for (int64_t i = 0; i < n; ++i) {
    int64_t root = uf_find(par, i);
    if (done[root]) continue;
    done[root] = 1;
    /* gather the cluster of this root */
    int64_t best = -1; int nd = 0; int32_t lo = 0, hi = 0; uint64_t seen[4] = {0, 0, 0, 0};
    for (int64_t k = 0; k < n; ++k) {
      if (uf_find(par, k) != root) continue;
      if (best < 0) { best = k; lo = t0[k]; hi = t0[k] + w[k]; }
      else {
        if (snr[k] > snr[best]) best = k;
        if (t0[k] < lo) lo = t0[k];
        if (t0[k] + w[k] > hi) hi = t0[k] + w[k];
      }
      int b = wid[k] & 255;
      if (!(seen[b >> 6] >> (b & 63) & 1)) { seen[b >> 6] |= (uint64_t)1 << (b & 63); ++nd; }
    }
    if (nd >= min_widths) { rep[nout] = best; nhit[nout] = nd; tb[nout] = lo; te[nout] = hi; ++nout; }
  }
  /* order by representative's canonical position */
  for (int64_t i = 1; i < nout; ++i) {
    int64_t r = rep[i]; int32_t h = nhit[i], a = tb[i], b = te[i]; int64_t k = i - 1;
    while (k >= 0 && rep[k] > r) { rep[k+1] = rep[k]; nhit[k+1] = nhit[k]; tb[k+1] = tb[k]; te[k+1] = te[k]; --k; }
    rep[k+1] = r; nhit[k+1] = h; tb[k+1] = a; te[k+1] = b;
  }
  free(par); free(done);
  return nout;
}

int vo_sizeof_peak(void) { return (int)sizeof(vo_peak); }
