"""ctypes front end of the float64 CPU oracle (oracle/volks_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  It never imports the CUDA package and shares no code,
table or constant with it.  The arithmetic lives in volks_oracle.c (each function cites the
PAPER.md passage it follows); this file only marshals numpy arrays and applies the threshold /
canonical ordering that DESIGN.md readings A3, A4, A9 fix:

  candidate iff snr > snr_thresh (strict; PAPER.md:196 "exceeds the threshold", :208 "SNR > 6"),
  candidates listed in canonical order (bl, ifq, q, j).

Parity status: every function here is pinned by tests/test_oracle_pins.py (closed forms P1-P14 of
DESIGN.md) except `window_match`, which is pinned only by hand-built constructions and a second
brute-force statement of the same rule (the paper gives no worked example) - see DESIGN.md.
`dedisperse` / `dm_shifts` (step 4) are pinned by test_dedispersion_pins and
test_dedispersed_pulse_closed_form; `allif_search` (Eq. 1) by test_allif_search_pins; `zscore_candidates`
by test_zscore_selection_pins; `baseline_match` by direct constructions and an independent sweep statement
(test_baseline_match_constructions, test_baseline_match_vs_sweep); the restricted delay range (`delay_range`,
PAPER.md:208) by test_delay_range_pins (closed form off the allowed columns, numpy.fft2 masked, Parseval unchanged).
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "volks_oracle.c")
_LIB = os.path.join(_HERE, "libvolks_oracle.so")

PEAK_DTYPE = np.dtype(
    [("p1", "<f8"), ("p2", "<f8"), ("s1", "<f8"), ("snr", "<f8"), ("idx1", "<i8"), ("idx2", "<i8")]
)
CAND_DTYPE = np.dtype(
    [("bl", "<i4"), ("ifq", "<i4"), ("wid", "<i4"), ("win", "<i4"), ("t0", "<i4"),
     ("rate_idx", "<i4"), ("delay_idx", "<i4"), ("power", "<f8"), ("snr", "<f8")]
)
PULSE_DTYPE = np.dtype(
    [("rep", "<i8"), ("nwidths_hit", "<i4"), ("t_begin", "<i4"), ("t_end", "<i4")]
)

MODES = {"direct": 0, "fft": 1, "cached": 2}


def build(force=False):
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        )
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        assert lib.vo_sizeof_peak() == PEAK_DTYPE.itemsize
        lib.vo_window.restype = ctypes.c_int
        lib.vo_search.restype = ctypes.c_int
        lib.vo_window_match.restype = ctypes.c_int64
        _lib = lib
    return _lib


def _as_f32_pairs(a):
    a = np.ascontiguousarray(a, dtype=np.complex64)
    return a, a.view(np.float32)


def _i32(x):
    return np.ascontiguousarray(np.asarray(x, dtype=np.int32))


def nwin(nap, w, s):
    return 0 if nap < w else (nap - w) // s + 1


def _range(delay_range):
    """(dlo, dhi) of a restricted delay search range, or (-1, -1) for the whole axis (A14):
    the maximum is looked for in the padded delay bins dlo..dhi, wrapping through nf-1 -> 0 when dlo > dhi; the noise
    statistic stays the whole plane's."""
    if delay_range is None:
        return -1, -1
    lo, hi = int(delay_range[0]), int(delay_range[1])
    assert lo >= 0 and hi >= 0
    return lo, hi


def window(win, nt, nf, mode="fft", want_plane=False, delay_range=None):
    """Fringe-search one window.  win: complex [w][nchan].  Returns (peak record, plane|None)."""
    lib = _load()
    win, wf = _as_f32_pairs(win)
    w, nchan = win.shape
    pk = np.zeros(1, dtype=PEAK_DTYPE)
    plane = np.zeros((nt, nf), dtype=np.complex128) if want_plane else None
    rc = lib.vo_window(
        ctypes.c_int(MODES[mode]), wf.ctypes.data_as(ctypes.c_void_p), ctypes.c_int64(nchan),
        ctypes.c_int(w), ctypes.c_int(nchan), ctypes.c_int(nt), ctypes.c_int(nf),
        plane.ctypes.data_as(ctypes.c_void_p) if want_plane else None,
        pk.ctypes.data_as(ctypes.c_void_p), ctypes.c_int(_range(delay_range)[0]), ctypes.c_int(_range(delay_range)[1]))
    if rc != 0:
        raise ValueError("vo_window: bad arguments")
    return pk[0], plane


def search(vis, widths, strides, nts, nf, mode="cached", select=None, nthreads=0, delay_range=None):
    """Peak record of every window (or of the canonical indices in `select`).

    vis: complex64 [nbl][nif][nap][nchan].  Output order: canonical (bl, ifq, q, j).
    Returns (peaks PEAK_DTYPE[n], threads_used)."""
    lib = _load()
    vis, vf = _as_f32_pairs(vis)
    nbl, nif, nap, nchan = vis.shape
    widths, strides, nts = _i32(widths), _i32(strides), _i32(nts)
    per_pair = sum(nwin(nap, int(w), int(s)) for w, s in zip(widths, strides))
    if select is None:
        n, sel, selp = nbl * nif * per_pair, None, None
        nsel = -1
    else:
        sel = np.ascontiguousarray(np.asarray(select, dtype=np.int64))
        n, nsel, selp = sel.size, sel.size, sel.ctypes.data_as(ctypes.c_void_p)
    out = np.zeros(n, dtype=PEAK_DTYPE)
    used = lib.vo_search(
        vf.ctypes.data_as(ctypes.c_void_p), ctypes.c_int(nbl), ctypes.c_int(nif),
        ctypes.c_int(nap), ctypes.c_int(nchan), ctypes.c_int(len(widths)),
        widths.ctypes.data_as(ctypes.c_void_p), strides.ctypes.data_as(ctypes.c_void_p),
        nts.ctypes.data_as(ctypes.c_void_p), ctypes.c_int(nf), ctypes.c_int(MODES[mode]),
        selp, ctypes.c_int64(nsel), out.ctypes.data_as(ctypes.c_void_p), ctypes.c_int(nthreads),
        ctypes.c_int(_range(delay_range)[0]), ctypes.c_int(_range(delay_range)[1]))
    if used < 0:
        raise ValueError("vo_search: bad arguments")
    return out, used


K_DM_MS = 4.148808  # cold-plasma dispersion constant [ms GHz^2 cm^3 / pc] (textbook; the paper gives none)


def dm_shifts(dm, f_chan_mhz, f_ref_mhz, t_ap_s):
    """Integer AP shift of every frequency point for a dispersion measure `dm` [pc cm^-3]:
    round(delay / T_ap), delay = 4.148808 ms * DM * (f^-2 - f_ref^-2) with f in GHz.  Step 4 of the
    paper applies "a specific time shift" per frequency point without stating
    the formula; this is the textbook one (reading R3).  f_chan_mhz: array [nif][nchan]."""
    f = np.asarray(f_chan_mhz, dtype=np.float64) * 1e-3
    delay_s = K_DM_MS * 1e-3 * float(dm) * (f ** -2 - (float(f_ref_mhz) * 1e-3) ** -2)
    return np.rint(delay_s / float(t_ap_s)).astype(np.int32)


def dedisperse(vis, shifts):
    """Step 4: for each frequency point a time shift.  out[bl][ifq][t][k] =
    vis[bl][ifq][t + shifts[ifq][k]][k], zero where t + shift falls outside [0, nap).  Written as the
    plain loop over (ifq, k) it is in the paper."""
    vis = np.asarray(vis)
    nbl, nif, nap, nchan = vis.shape
    sh = np.asarray(shifts, dtype=np.int64).reshape(nif, nchan)
    out = np.zeros_like(vis)
    for n in range(nif):
        for k in range(nchan):
            d = int(sh[n, k])
            if d >= nap or d <= -nap:
                continue
            if d >= 0:
                out[:, n, :nap - d, k] = vis[:, n, d:, k]
            else:
                out[:, n, -d:, k] = vis[:, n, :nap + d, k]
    return out


def canonical_table(nbl, nif, nap, widths, strides):
    """(bl, ifq, wid, win, t0) int32 arrays for every window in canonical order."""
    nws = [nwin(nap, int(w), int(s)) for w, s in zip(widths, strides)]
    wid = np.concatenate([np.full(n, q, np.int32) for q, n in enumerate(nws)]) if nws else np.zeros(0, np.int32)
    win = np.concatenate([np.arange(n, dtype=np.int32) for n in nws]) if nws else np.zeros(0, np.int32)
    t0 = win * np.asarray(strides, np.int32)[wid] if wid.size else win
    per = wid.size
    pair = np.repeat(np.arange(nbl * nif, dtype=np.int32), per)
    return (pair // nif, pair % nif, np.tile(wid, nbl * nif), np.tile(win, nbl * nif),
            np.tile(t0, nbl * nif))


def candidates(peaks, nbl, nif, nap, widths, strides, nf, snr_thresh):
    """Threshold (strict >) the full canonical peak array into the canonical candidate list."""
    bl, ifq, wid, win, t0 = canonical_table(nbl, nif, nap, widths, strides)
    keep = np.nonzero(peaks["snr"] > snr_thresh)[0]
    c = np.zeros(keep.size, dtype=CAND_DTYPE)
    c["bl"], c["ifq"], c["wid"], c["win"], c["t0"] = bl[keep], ifq[keep], wid[keep], win[keep], t0[keep]
    c["rate_idx"] = peaks["idx1"][keep] // nf
    c["delay_idx"] = peaks["idx1"][keep] % nf
    c["power"] = peaks["p1"][keep]
    c["snr"] = peaks["snr"][keep]
    return c, keep


def window_match(cands, widths, min_widths=2):
    """Per-(bl, ifq) multi-window match (A13)."""
    lib = _load()
    n = len(cands)
    out = np.zeros(n, dtype=PULSE_DTYPE)
    if n == 0:
        return out
    bl, ifq, wid, t0 = (_i32(cands[k]) for k in ("bl", "ifq", "wid", "t0"))
    w = _i32(np.asarray(widths, np.int32)[wid])
    snr = np.ascontiguousarray(cands["snr"], dtype=np.float64)
    rep = np.zeros(n, np.int64)
    nhit, tb, te = np.zeros(n, np.int32), np.zeros(n, np.int32), np.zeros(n, np.int32)
    p = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    k = lib.vo_window_match(ctypes.c_int64(n), p(bl), p(ifq), p(wid), p(t0), p(w), p(snr),
                            ctypes.c_int(min_widths), p(rep), p(nhit), p(tb), p(te))
    out = out[:k]
    out["rep"], out["nwidths_hit"], out["t_begin"], out["t_end"] = rep[:k], nhit[:k], tb[:k], te[:k]
    return out


def baseline_match(bl, snr, t_begin, t_end, min_baselines=5):
    """Multi-baseline cross-match ("identified if it is detected with at least 5
    baselines"; A19), written as the definition: pulses i, j are linked when their AP
    extents [t_begin, t_end) overlap; connected components (union-find over all O(n^2) pairs) are
    clusters; a cluster with >= min_baselines distinct baselines is a detection.  Returns a list of
    dicts {rep, nbaselines, t_begin, t_end} ordered by (t_begin, rep); rep = max-snr member (ties:
    lowest index).  Pinned by hand constructions only (the paper prints no example)."""
    n = len(bl)
    parent = list(range(n))

    def find(x):
        while parent[x] != x:
            parent[x] = parent[parent[x]]
            x = parent[x]
        return x
    for i in range(n):
        for j in range(i + 1, n):
            if t_begin[i] < t_end[j] and t_begin[j] < t_end[i]:
                parent[find(i)] = find(j)
    groups = {}
    for i in range(n):
        groups.setdefault(find(i), []).append(i)
    out = []
    for members in groups.values():
        nb = len({int(bl[i]) for i in members})
        if nb < min_baselines:
            continue
        rep = max(members, key=lambda i: (float(snr[i]), -i))
        out.append(dict(rep=rep, nbaselines=nb, t_begin=int(min(t_begin[i] for i in members)),
                        t_end=int(max(t_end[i] for i in members))))
    out.sort(key=lambda d: (d["t_begin"], d["rep"]))
    return out


def zscore_candidates(peaks, nbl, nif, nap, widths, strides, nf, z_thresh):
    """f4 - the other reading of PAPER.md:196 ("for the time segments series of given window size, a
    single pulse is selected if its normalized power exceeds the threshold, which is set to 3"):
    per (bl, ifq, width) the series of window peak powers P1_j is normalised across windows,
    z_j = (P1_j - mean_j P1) / std_j P1 (population std; z = 0 when std = 0), candidate iff z > z_thresh.
    Returns (candidates in canonical order with `snr` = z, z of every window in canonical order)."""
    bl, ifq, wid, win, t0 = canonical_table(nbl, nif, nap, widths, strides)
    p1 = np.asarray(peaks["p1"], dtype=np.float64)
    z = np.zeros(len(p1))
    per = len(p1) // max(nbl * nif, 1)
    nws = [nwin(nap, int(w), int(s)) for w, s in zip(widths, strides)]
    for pair in range(nbl * nif):
        off = pair * per
        for n in nws:
            x = p1[off: off + n]
            if n:
                sd = x.std()
                z[off: off + n] = (x - x.mean()) / sd if sd > 0 else 0.0
            off += n
    keep = np.nonzero(z > z_thresh)[0]
    out = np.zeros(len(keep), dtype=CAND_DTYPE)
    out["bl"], out["ifq"], out["wid"], out["win"], out["t0"] = bl[keep], ifq[keep], wid[keep], win[keep], t0[keep]
    out["rate_idx"], out["delay_idx"] = peaks["idx1"][keep] // nf, peaks["idx1"][keep] % nf
    out["power"], out["snr"] = p1[keep], z[keep]
    return out, z


def allif_band(vis):
    """[nbl][nif][nap][nchan] -> [nbl][nap][nif*nchan]: the frequency points of all IFs of one AP in
    sky-frequency order, IFs contiguous (f = f0 + (n*nchan + j)*df; reading A21)."""
    vis = np.asarray(vis)
    nbl, nif, nap, nchan = vis.shape
    return np.ascontiguousarray(vis.transpose(0, 2, 1, 3)).reshape(nbl, nap, nif * nchan)


def allif_search(vis, widths, strides, nfa, delay_range=None):
    """f2 - VOLKS2's own fringe search, Eq. 1: ONE delay across all IFs,
        G(dtau) = sum_n sum_j S(n, j) e^{-i Phi},  Phi = 2 pi f_j^n dtau,
    evaluated with one zero-padded FFT over the whole band per AP ("32768 sized FFT"),
    the APs of a window summed coherently (step 6), then the maximum along the delay axis.
    Per (bl, width, window): A[d] = sum_{t<w} sum_m band[t0+t][m] e^{-2 pi i m d/nfa}; P = |A|^2;
    (P1, idx1) first argmax, (P2, idx2) runner-up, S1 = sum_d P, snr = sqrt(P1/(S1/nfa)) (A3's statistic
    on the delay axis).  Evaluated as the rate-0 row of this oracle's own 2-D plane of the band window
    (pin P4 / PAPER.md:133, 143: summing per-AP spectra == spectrum of the sum).
    delay_range = (lo, hi): the maximum is looked for in the delay bins lo..hi of the nfa axis only (wrapping when
    lo > hi), the noise S1 stays the sum over the whole axis.
    Output order: canonical (bl, q, j); PEAK_DTYPE records."""
    lo, hi = _range(delay_range)
    dd = np.arange(nfa)
    allowed = np.ones(nfa, bool) if lo < 0 else ((dd >= lo) & (dd <= hi) if lo <= hi else (dd >= lo) | (dd <= hi))
    band = allif_band(vis)
    nbl, nap, nm = band.shape
    out = []
    for b in range(nbl):
        for w, s in zip(widths, strides):
            nt = 1
            while nt < w:
                nt *= 2
            for j in range(nwin(nap, int(w), int(s))):
                _, plane = window(band[b, j * s: j * s + w], nt, nfa, mode="fft", want_plane=True)
                a = plane[0]
                pall = a.real * a.real + a.imag * a.imag
                p = np.where(allowed, pall, -1.0)        # bins outside the searched range cannot be the peak
                i1 = int(np.argmax(p))
                q = p.copy()
                q[i1] = -1.0
                i2 = int(np.argmax(q)) if nfa > 1 else i1
                s1 = float(pall.sum())
                noise = s1 / nfa
                out.append((p[i1], max(q[i2], 0.0) if nfa > 1 else 0.0, s1, np.sqrt(p[i1] / noise) if noise > 0 else 0.0, i1, i2))
    return np.array(out, dtype=PEAK_DTYPE) if out else np.zeros(0, dtype=PEAK_DTYPE)


def cal_phasors(delay_s, phase_rad, nchan, chan_hz):
    """Initial-calibration phasors of Eq. 1: the last two terms of
    Phi(n, j) = ... + 2 pi f_j dtau0^n + dphi0^n, with f_j = j * chan_hz the j-th frequency point inside
    the IF, enter G as S(n, j) e^{-i(2 pi f_j dtau0^n + dphi0^n)}.  delay_s, phase_rad: [nbl][nif]
    (per baseline and IF).  Returns complex64 [nbl][nif][nchan]."""
    d = np.asarray(delay_s, dtype=np.float64)[..., None]
    p = np.asarray(phase_rad, dtype=np.float64)[..., None]
    f = np.arange(nchan, dtype=np.float64) * float(chan_hz)
    return np.exp(-1j * (2.0 * np.pi * f * d + p)).astype(np.complex64)


def calibrate(vis, cal):
    """Step 3: vis[bl][ifq][t][k] * cal[bl][ifq][k], formed in double, stored as complex64."""
    v = np.asarray(vis).astype(np.complex128) * np.asarray(cal).astype(np.complex128)[:, :, None, :]
    return v.astype(np.complex64)
