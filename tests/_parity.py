"""Comparison rules CUDA path vs oracle (north_star).

 * per window: (r*, d*) must equal the oracle's first argmax idx1, except where the oracle's top two
   powers differ by < 1e-5 relative: there idx2 is accepted too, and - for planes with MORE than two
   bins inside that margin (e.g. a window with one non-zero AP: every rate row carries the same
   powers) - any bin whose ORACLE power lies within 1e-5 relative of P1 (`plane_power` callback);
 * |P1_gpu - P1| <= 1e-4 P1 and |snr_gpu - snr| <= 1e-4 snr;
 * candidate lists identical and in canonical order, except that a window whose oracle snr lies
   within 1e-4 relative of the threshold may be present or absent.
"""
import numpy as np

RTOL = 1e-4
TIE = 1e-5


def dense_index(nbl, nif, nwin_per_width):
    """dense-layout index (include/volks.h) of every window in canonical order."""
    npair = nbl * nif
    per = int(sum(nwin_per_width))
    out = np.empty(npair * per, dtype=np.int64)
    offd, offc = 0, 0
    for n in nwin_per_width:
        j = np.arange(n, dtype=np.int64)
        for pair in range(npair):
            out[pair * per + offc: pair * per + offc + n] = offd + pair * n + j
        offd += npair * n
        offc += n
    return out


def check_peaks(gpu_peaks, ora, nf, plane_power=None):
    """gpu_peaks: PEAK records aligned with `ora` (oracle PEAK records).  Returns #ties used.
    plane_power(i, idx) -> the oracle's power of bin `idx` of window `i` (for many-way near-ties)."""
    gidx = gpu_peaks["rate_idx"].astype(np.int64) * nf + gpu_peaks["delay_idx"].astype(np.int64)
    p1 = ora["p1"]
    safe = np.where(p1 > 0, p1, 1.0)
    near_tie = (p1 - ora["p2"]) / safe < TIE
    ok_idx = (gidx == ora["idx1"]) | (near_tie & (gidx == ora["idx2"]))
    bad = np.nonzero(~ok_idx)[0]
    if plane_power is not None and bad.size and bad.size <= 200 and np.all(near_tie[bad]):
        still = [i for i in bad if not plane_power(int(i), int(gidx[i])) >= p1[i] * (1.0 - TIE)]
        bad = np.asarray(still, dtype=np.int64)
    assert bad.size == 0, "argmax mismatch at %s: gpu %s oracle %s/%s gap %s" % (
        bad[:5], gidx[bad[:5]], ora["idx1"][bad[:5]], ora["idx2"][bad[:5]], ((p1 - ora["p2"]) / safe)[bad[:5]])
    perr = np.abs(gpu_peaks["power"].astype(np.float64) - p1) / safe
    assert perr.max(initial=0.0) <= RTOL, "power error %g" % perr.max()
    ssafe = np.where(ora["snr"] > 0, ora["snr"], 1.0)
    serr = np.abs(gpu_peaks["snr"].astype(np.float64) - ora["snr"]) / ssafe
    assert serr.max(initial=0.0) <= RTOL, "snr error %g" % serr.max()
    return int(np.count_nonzero(gidx != ora["idx1"])), float(perr.max(initial=0.0)), float(serr.max(initial=0.0))


def check_candidates(gpu_cands, ora_cands, ora_peaks, keep, thresh, nf):
    """Ordered candidate list equality, with the near-threshold exemption: a window whose oracle
    snr lies within RTOL of the threshold may be present or absent.  `keep` = canonical window index
    of every oracle candidate.  Returns (#candidates compared, #marginal windows)."""
    key = lambda c: (int(c["bl"]), int(c["ifq"]), int(c["wid"]), int(c["win"]))
    gk = [key(c) for c in gpu_cands]
    assert gk == sorted(gk), "GPU candidates not in canonical order"
    assert len(set(gk)) == len(gk), "duplicate GPU candidates"
    marg = np.abs(ora_peaks["snr"][keep] - thresh) <= RTOL * thresh        # marginal oracle candidates
    nmarg_all = int(np.count_nonzero(np.abs(ora_peaks["snr"] - thresh) <= RTOL * thresh))
    omap = {key(c): i for i, c in enumerate(ora_cands)}
    gset = set(gk)
    for k_, i in omap.items():                      # every firm oracle candidate must be present
        assert k_ in gset or marg[i], "missing candidate %s (oracle snr %r)" % (k_, ora_cands[i]["snr"])
    extra = [k_ for k_ in gk if k_ not in omap]     # extras are allowed only if marginal
    assert len(extra) <= nmarg_all - int(marg.sum()), "unexpected candidates %s" % extra[:5]
    n = 0
    for g in gpu_cands:
        i = omap.get(key(g))
        if i is None:
            assert abs(float(g["snr"]) - thresh) <= 2 * RTOL * thresh
            continue
        o = ora_cands[i]
        assert g["t0"] == o["t0"]
        assert abs(float(g["power"]) - o["power"]) <= RTOL * o["power"]
        assert abs(float(g["snr"]) - o["snr"]) <= RTOL * o["snr"]
        n += 1
    return n, nmarg_all


def allif_plane_power(oracle, band, nw, widths, strides, nfa):
    """Tie callback for the all-IF search: the ORACLE's power of delay bin `idx` of canonical window i,
    from the rate-0 row of the oracle's own plane of that band window (oracle.allif_search's definition)."""
    per = sum(nw)

    def plane_power(i, idx):
        b, r = divmod(i, per)
        q = 0
        while r >= nw[q]:
            r -= nw[q]
            q += 1
        w, s = widths[q], strides[q]
        nt = 1
        while nt < w:
            nt *= 2
        _, plane = oracle.window(band[b, r * s: r * s + w], nt, nfa, mode="fft", want_plane=True)
        z = plane[0, idx]
        return float(z.real * z.real + z.imag * z.imag)
    return plane_power


def canonical_index(cands, nif, nw, bl0=0):
    """Canonical window index c = (pair * per_pair + offc[q] + j) of candidate records, with pairs counted
    from baseline `bl0` (a search over a slice of baselines)."""
    nw = np.asarray(nw, dtype=np.int64)
    offc = np.concatenate([[0], np.cumsum(nw)[:-1]])
    pair = (cands["bl"].astype(np.int64) - bl0) * nif + cands["ifq"].astype(np.int64)
    return pair * int(nw.sum()) + offc[cands["wid"]] + cands["win"].astype(np.int64)


def check_candidates_whole(gpu_cands, gidx, ora_cands, ora_peaks, keep, thresh):
    """check_candidates for lists of millions of records (vectorised; the same rule): `gidx` / `keep` are
    the canonical window indices of the GPU / oracle candidates.  Ordered, duplicate-free; every firm oracle
    candidate present; every extra marginal BY THE ORACLE'S snr; matched records agree in t0, power, snr.
    Returns (#matched, #missing marginal, #extra marginal, #marginal windows in the slice)."""
    assert np.all(np.diff(gidx) > 0), "GPU candidates not in canonical order / duplicated"
    osnr = ora_peaks["snr"]
    marginal = np.abs(osnr - thresh) <= RTOL * thresh
    in_o = np.isin(gidx, keep, assume_unique=True)
    missing = keep[~np.isin(keep, gidx, assume_unique=True)]
    assert np.all(marginal[missing]), "missing candidates at windows %s (oracle snr %s)" % (missing[:5], osnr[missing[:5]])
    extra = gidx[~in_o]
    assert np.all(marginal[extra]), "unexpected candidates at windows %s (oracle snr %s)" % (extra[:5], osnr[extra[:5]])
    pos = np.searchsorted(keep, gidx[in_o])
    g, o = gpu_cands[in_o], ora_cands[pos]
    assert np.array_equal(g["t0"], o["t0"]) and np.array_equal(g["wid"], o["wid"]) and np.array_equal(g["win"], o["win"])
    assert np.all(np.abs(g["power"].astype(np.float64) - o["power"]) <= RTOL * o["power"])
    assert np.all(np.abs(g["snr"].astype(np.float64) - o["snr"]) <= RTOL * o["snr"])
    return int(in_o.sum()), int(missing.size), int(extra.size), int(marginal.sum())


def check_candidate_bins(gpu_cands, cidx, ora_peaks, nf, plane_power=None):
    """The (rate, delay) bin, power and snr of candidate records against the oracle's peaks of the same windows
    (`cidx` = canonical window index of every record), by the rules of check_peaks."""
    gp = np.zeros(len(gpu_cands), dtype=[("power", "<f4"), ("snr", "<f4"), ("rate_idx", "<i4"), ("delay_idx", "<i4")])
    for f in ("power", "snr", "rate_idx", "delay_idx"):
        gp[f] = gpu_cands[f]
    pp = None if plane_power is None else (lambda i, idx: plane_power(int(cidx[i]), idx))
    return check_peaks(gp, ora_peaks[cidx], nf, pp)
