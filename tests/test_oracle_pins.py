"""Pins of the float64 oracle against what the paper and the mathematics fix (P1-P14).

None of these retype the oracle's formula: they are closed forms (Dirichlet kernel, Parseval),
invariances, brute force in a second language (numpy einsum), a library special case
(numpy.fft) and the statistics of the noise.  CPU only."""
import math
import os

import numpy as np
import pytest

import workloads

TWO_PI = 2 * math.pi


def fringe(w, nchan, tau_c, rho_c, a=1.0, phi0=0.3):
    t = np.arange(w)[:, None]
    k = np.arange(nchan)[None, :]
    return (a * np.exp(1j * (TWO_PI * (tau_c * k + rho_c * t) + phi0))).astype(np.complex64)


def dirichlet(M, x):
    x = np.asarray(x, dtype=np.float64)
    num, den = np.sin(np.pi * M * x), np.sin(np.pi * x)
    out = np.full(x.shape, float(M))
    ok = np.abs(den) > 1e-12
    out[ok] = num[ok] / den[ok]
    return np.abs(out)


@pytest.mark.parametrize("mode", ["direct", "fft"])
@pytest.mark.parametrize("w,nchan,nt,nf,tau,rho", [(8, 32, 16, 64, 5, 2), (4, 16, 8, 64, 15, 3), (16, 8, 16, 8, 7, 15)])
def test_p1_on_bin_fringe_closed_form(oracle, mode, w, nchan, nt, nf, tau, rho):
    """P1: V = a e^{+i(2pi(tau k/nchan + rho t/w)+phi0)} peaks exactly at (rho Nt/w, tau Nf/nchan),
    P1 = (a w nchan)^2, S1 = Nt Nf a^2 w nchan, snr = sqrt(w nchan).  Pins the e^{-i Phi} sign of
    PAPER.md:74-79, the index mapping, the scaling and the SNR reading A3."""
    a = 0.7
    win = fringe(w, nchan, tau / nchan, rho / w, a=a)
    pk, _ = oracle.window(win, nt, nf, mode=mode)
    assert pk["idx1"] == (rho * nt // w) * nf + tau * nf // nchan
    assert pk["p1"] == pytest.approx((a * w * nchan) ** 2, rel=1e-6)   # inputs are float32
    assert pk["s1"] == pytest.approx(nt * nf * a * a * w * nchan, rel=1e-6)
    assert pk["snr"] == pytest.approx(math.sqrt(w * nchan), rel=1e-6)


def test_p1_negative_sign_would_fail(oracle):
    """A conjugated kernel (wrong sign) would put the peak at the mirrored bin."""
    win = fringe(8, 32, 5 / 32, 2 / 8)
    pk, _ = oracle.window(win, 16, 64)
    assert pk["idx1"] == 4 * 64 + 10 and pk["idx1"] != (16 - 4) * 64 + (64 - 10)


@pytest.mark.parametrize("mode", ["direct", "fft"])
def test_p2_parseval(oracle, mode):
    rng = np.random.default_rng(5)
    for (w, nchan, nt, nf) in [(3, 5, 8, 8), (8, 32, 16, 64), (7, 20, 32, 32)]:
        win = (rng.normal(size=(w, nchan)) + 1j * rng.normal(size=(w, nchan))).astype(np.complex64)
        pk, _ = oracle.window(win, nt, nf, mode=mode)
        e = float(np.sum(np.abs(win.astype(np.complex128)) ** 2))
        assert pk["s1"] == pytest.approx(nt * nf * e, rel=1e-9)


def brute_plane(win, nt, nf):
    """Second statement of the definition (numpy einsum over explicit DFT matrices)."""
    w, nchan = win.shape
    Et = np.exp(-1j * TWO_PI * np.outer(np.arange(nt), np.arange(w)) / nt)
    Ef = np.exp(-1j * TWO_PI * np.outer(np.arange(nchan), np.arange(nf)) / nf)
    return Et @ win.astype(np.complex128) @ Ef


def test_p3_brute_force_random_planes(oracle):
    rng = np.random.default_rng(11)
    for (w, nchan, nt, nf) in [(2, 3, 4, 4), (4, 4, 4, 4), (5, 9, 8, 16), (8, 32, 16, 64), (16, 33, 16, 64)]:
        win = (rng.normal(size=(w, nchan)) + 1j * rng.normal(size=(w, nchan))).astype(np.complex64)
        ref = brute_plane(win, nt, nf)
        for mode in ("direct", "fft"):
            pk, plane = oracle.window(win, nt, nf, mode=mode, want_plane=True)
            assert np.max(np.abs(plane - ref)) <= 1e-12 * np.max(np.abs(ref)) * nt * nf
            P = np.abs(ref) ** 2
            assert pk["idx1"] == int(np.argmax(P))
            assert pk["p1"] == pytest.approx(P.max(), rel=1e-12)


def test_p3_config0_all_windows_three_modes(oracle):
    vis, c, _ = workloads.generate(0)
    v = vis.numpy()
    args = (v, c["widths"], c["strides"], c["nts"], c["nf"])
    d, _ = oracle.search(*args, mode="direct")
    f, _ = oracle.search(*args, mode="fft")
    k, _ = oracle.search(*args, mode="cached")
    assert len(d) == 505
    for other in (f, k):
        assert np.array_equal(d["idx1"], other["idx1"])
        assert np.allclose(d["p1"], other["p1"], rtol=1e-12)
        assert np.allclose(d["s1"], other["s1"], rtol=1e-12)
        assert np.allclose(d["p2"], other["p2"], rtol=1e-12)


def test_cached_equals_fft_config1_and_selection(oracle):
    vis, c, _ = workloads.generate(1, nap=300)
    v = vis.numpy()
    args = (v, c["widths"], c["strides"], c["nts"], c["nf"])
    f, _ = oracle.search(*args, mode="fft")
    k, _ = oracle.search(*args, mode="cached")
    assert np.array_equal(f["idx1"], k["idx1"]) and np.array_equal(f["idx2"], k["idx2"])
    assert np.allclose(f["p1"], k["p1"], rtol=1e-12) and np.allclose(f["snr"], k["snr"], rtol=1e-12)
    sel = np.array([0, 5, len(f) - 1, len(f) // 2, 17])
    s, _ = oracle.search(*args, mode="fft", select=sel)
    assert np.array_equal(s["idx1"], f["idx1"][sel]) and np.allclose(s["p1"], f["p1"][sel], rtol=1e-13)


def test_p4_paper_1d_scheme_is_rate_zero_row(oracle):
    """PAPER.md:133 + 143: FFT each AP along frequency, then sum the window's APs == row r=0."""
    rng = np.random.default_rng(3)
    w, nchan, nt, nf = 8, 32, 16, 128
    win = (rng.normal(size=(w, nchan)) + 1j * rng.normal(size=(w, nchan))).astype(np.complex64)
    _, plane = oracle.window(win, nt, nf, want_plane=True)
    per_ap = np.fft.fft(win.astype(np.complex128), n=nf, axis=1)
    assert np.allclose(plane[0], per_ap.sum(axis=0), rtol=0, atol=1e-10)
    assert np.allclose(plane[0], np.fft.fft(win.astype(np.complex128).sum(axis=0), n=nf), atol=1e-10)


def test_p5_off_bin_fringe_dirichlet(oracle):
    w, nchan, nt, nf, a = 8, 32, 16, 64, 0.9
    tau_c, rho_c = 0.1234, -0.3171
    win64 = a * np.exp(1j * (TWO_PI * (tau_c * np.arange(nchan)[None, :] + rho_c * np.arange(w)[:, None]) + 0.4))
    win = win64.astype(np.complex64)
    _, plane = oracle.window(win, nt, nf, want_plane=True)
    r = np.arange(nt)[:, None] / nt
    d = np.arange(nf)[None, :] / nf
    expect = a * dirichlet(w, r - rho_c) * dirichlet(nchan, d - tau_c)
    assert np.max(np.abs(np.abs(plane) - expect)) < 2e-5 * a * w * nchan   # float32 input rounding


def test_p6_delta_input(oracle):
    win = np.zeros((8, 32), np.complex64)
    win[3, 7] = 2 - 1j
    for mode in ("direct", "fft"):
        pk, _ = oracle.window(win, 16, 64, mode=mode)
        assert pk["p1"] == pytest.approx(5.0, rel=1e-12) and pk["snr"] == pytest.approx(1.0, rel=1e-12)
    pk, _ = oracle.window(np.array([[1 + 0j]], np.complex64), 4, 8)
    assert pk["idx1"] == 0 and pk["idx2"] == 1 and pk["p1"] == pk["p2"] == 1.0


def test_p6_all_zero_window(oracle):
    pk, _ = oracle.window(np.zeros((4, 8), np.complex64), 8, 16)
    assert pk["p1"] == 0.0 and pk["snr"] == 0.0 and pk["idx1"] == 0


def test_p7_width_one(oracle):
    rng = np.random.default_rng(9)
    row = (rng.normal(size=(1, 32)) + 1j * rng.normal(size=(1, 32))).astype(np.complex64)
    pk, plane = oracle.window(row, 2, 128, want_plane=True)
    spec = np.abs(np.fft.fft(row[0].astype(np.complex128), n=128)) ** 2
    assert np.allclose(np.abs(plane[0]) ** 2, spec) and np.allclose(np.abs(plane[1]) ** 2, spec)
    assert pk["idx1"] == int(np.argmax(spec))          # r* = 0 (first of the tied rows)
    assert pk["idx1"] < 128 and pk["idx2"] == pk["idx1"] + 128


def test_p8_scaling_and_phase_invariance(oracle):
    vis, c, _ = workloads.generate(0)
    v = vis.numpy()[:, :, :64]
    args = (c["widths"], c["strides"], c["nts"], c["nf"])
    a, _ = oracle.search(v, *args, mode="fft")
    b, _ = oracle.search((v * np.complex64(2j)).astype(np.complex64), *args, mode="fft")
    assert np.array_equal(a["idx1"], b["idx1"])
    assert np.allclose(b["p1"], 4 * a["p1"], rtol=1e-12) and np.allclose(a["snr"], b["snr"], rtol=1e-12)


def test_p9_shift_invariance(oracle):
    vis, c, _ = workloads.generate(1, nap=200)
    v = vis.numpy()
    q = 2
    w, s, nt = c["widths"][q], c["strides"][q], c["nts"][q]
    m = 3
    a, _ = oracle.search(v, [w], [s], [nt], c["nf"], mode="fft")
    b, _ = oracle.search(np.ascontiguousarray(v[:, :, m * s:]), [w], [s], [nt], c["nf"], mode="fft")
    na, nb = workloads.gen.nwin(200, w, s), workloads.gen.nwin(200 - m * s, w, s)
    A, Bv = a.reshape(8, na), b.reshape(8, nb)
    assert np.array_equal(A["idx1"][:, m:], Bv["idx1"]) and np.array_equal(A["p1"][:, m:], Bv["p1"])


def test_p10_padding_consistency(oracle):
    rng = np.random.default_rng(21)
    w, nchan = 8, 16
    win = (rng.normal(size=(w, nchan)) + 1j * rng.normal(size=(w, nchan))).astype(np.complex64)
    _, small = oracle.window(win, 8, 16, want_plane=True)
    _, big = oracle.window(win, 32, 64, want_plane=True)
    assert np.allclose(big[::4, ::4], small, atol=1e-11)


def test_p11_width_doubling_identity(oracle):
    rng = np.random.default_rng(22)
    w, nchan, nf = 4, 16, 32
    x = (rng.normal(size=(2 * w, nchan)) + 1j * rng.normal(size=(2 * w, nchan))).astype(np.complex64)
    _, f1 = oracle.window(x[:w], 2 * w, nf, want_plane=True)
    _, f2 = oracle.window(x[w:], 2 * w, nf, want_plane=True)
    _, fb = oracle.window(x, 4 * w, nf, want_plane=True)
    sign = ((-1.0) ** np.arange(2 * w))[:, None]
    assert np.allclose(fb[::2], f1 + sign * f2, atol=1e-11)


def test_p12_numpy_fft2_special_case(oracle):
    rng = np.random.default_rng(23)
    for (w, nchan, nt, nf) in [(8, 32, 16, 64), (32, 64, 64, 128), (64, 128, 128, 256)]:
        win = (rng.normal(size=(w, nchan)) + 1j * rng.normal(size=(w, nchan))).astype(np.complex64)
        pk, plane = oracle.window(win, nt, nf, want_plane=True)
        ref = np.fft.fft2(win.astype(np.complex128), s=(nt, nf))
        assert np.max(np.abs(plane - ref)) < 1e-10 * np.max(np.abs(ref))
        assert pk["idx1"] == int(np.argmax(np.abs(ref) ** 2))


def test_p13_noise_statistics(oracle):
    vis, c, _ = workloads.generate(0, npulses=0)
    pk, _ = oracle.search(vis.numpy(), [8], [8], [8], 32, mode="fft")     # unpadded, disjoint
    noise = pk["s1"] / (8 * 32)
    assert np.mean(noise) == pytest.approx(8 * 32, rel=0.05)
    emax = np.mean(pk["p1"] / noise)
    assert emax == pytest.approx(math.log(8 * 32) + 0.5772, rel=0.2)


def test_p14_config0_expectation(oracle):
    exp = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "config0_expectation.txt")) as f:
        for line in f:
            if not line.startswith("#"):
                k, v = line.split()
                exp[k] = float(v)
    vis, c, _ = workloads.generate(0)
    pk, _ = oracle.search(vis.numpy(), c["widths"], c["strides"], c["nts"], c["nf"], mode="cached")
    j = int(exp["t0"])
    assert pk["idx1"][j] == int(exp["rate_idx"]) * c["nf"] + int(exp["delay_idx"])
    assert pk["p1"][j] == pytest.approx(exp["signal_power"] + exp["noise_mean"], rel=0.35)
    assert pk["snr"][j] > exp["snr_thresh"]
    cands, keep = oracle.candidates(pk, 1, 1, c["nap"], c["widths"], c["strides"], c["nf"], exp["snr_thresh"])
    assert len(cands) >= 1 and np.all(np.abs(cands["t0"] - 200) <= 3)     # no noise-only candidate
    assert np.all(cands["rate_idx"] == 4) and np.all(cands["delay_idx"] == 10)
    assert list(cands["win"]) == sorted(cands["win"])


def test_candidates_canonical_order_and_strict_threshold(oracle):
    vis, c, _ = workloads.generate(1, nap=400)
    pk, _ = oracle.search(vis.numpy(), c["widths"], c["strides"], c["nts"], c["nf"], mode="cached")
    thr = float(np.sort(pk["snr"])[-20])
    cands, keep = oracle.candidates(pk, 1, 8, 400, c["widths"], c["strides"], c["nf"], thr)
    assert len(cands) == 19                                   # strict >: the 20th is excluded
    key = list(zip(cands["bl"], cands["ifq"], cands["wid"], cands["win"]))
    assert key == sorted(key)
    assert np.all(cands["t0"] == cands["win"] * np.asarray(c["strides"])[cands["wid"]])


# ---- a8 window match: constructions + a second brute-force statement of the rule ----

def _cands(oracle, rows):
    c = np.zeros(len(rows), dtype=oracle.CAND_DTYPE)
    for i, (bl, ifq, wid, win, t0, snr) in enumerate(rows):
        c[i]["bl"], c[i]["ifq"], c[i]["wid"], c[i]["win"], c[i]["t0"], c[i]["snr"] = bl, ifq, wid, win, t0, snr
    return c


def test_window_match_constructions(oracle):
    widths = [4, 8, 16]
    # two widths overlapping -> kept, representative = max snr
    p = oracle.window_match(_cands(oracle, [(0, 0, 0, 10, 10, 7.0), (0, 0, 1, 1, 8, 9.0)]), widths)
    assert len(p) == 1 and p[0]["rep"] == 1 and p[0]["nwidths_hit"] == 2 and (p[0]["t_begin"], p[0]["t_end"]) == (8, 16)
    # one width twice -> dropped
    assert len(oracle.window_match(_cands(oracle, [(0, 0, 0, 10, 10, 7.0), (0, 0, 0, 11, 11, 9.0)]), widths)) == 0
    # chain A-B-C: A and C do not overlap but both overlap B -> one cluster
    p = oracle.window_match(_cands(oracle, [(0, 0, 0, 0, 0, 7.0), (0, 0, 1, 0, 3, 6.5), (0, 0, 0, 2, 10, 8.0)]), widths)
    assert len(p) == 1 and p[0]["rep"] == 2 and (p[0]["t_begin"], p[0]["t_end"]) == (0, 14)
    # touching intervals [0,4) and [4,12) do not overlap
    assert len(oracle.window_match(_cands(oracle, [(0, 0, 0, 0, 0, 7.0), (0, 0, 1, 0, 4, 7.0)]), widths)) == 0
    # different IF or baseline never match
    assert len(oracle.window_match(_cands(oracle, [(0, 0, 0, 0, 0, 7.0), (0, 1, 1, 0, 0, 7.0)]), widths)) == 0
    assert len(oracle.window_match(_cands(oracle, [(0, 0, 0, 0, 0, 7.0), (1, 0, 1, 0, 0, 7.0)]), widths)) == 0
    # snr tie -> lowest canonical position
    p = oracle.window_match(_cands(oracle, [(0, 0, 0, 0, 0, 7.0), (0, 0, 1, 0, 0, 7.0)]), widths)
    assert p[0]["rep"] == 0


def test_window_match_vs_python_graph_search(oracle):
    rng = np.random.default_rng(4)
    widths = [2, 4, 8, 16]
    rows = []
    for _ in range(120):
        wid = int(rng.integers(0, 4))
        rows.append((int(rng.integers(0, 2)), int(rng.integers(0, 2)), wid, 0, int(rng.integers(0, 300)), float(rng.uniform(6, 20))))
    rows.sort(key=lambda r: (r[0], r[1], r[2], r[4]))
    c = _cands(oracle, rows)
    got = oracle.window_match(c, widths, 2)
    # flood fill on the explicit overlap graph
    n = len(rows)
    iv = [(r[4], r[4] + widths[r[2]]) for r in rows]
    adj = [[k for k in range(n) if k != i and rows[i][:2] == rows[k][:2] and iv[i][0] < iv[k][1] and iv[k][0] < iv[i][1]] for i in range(n)]
    seen, expect = set(), []
    for i in range(n):
        if i in seen:
            continue
        comp, stack = [], [i]
        seen.add(i)
        while stack:
            x = stack.pop()
            comp.append(x)
            for y in adj[x]:
                if y not in seen:
                    seen.add(y)
                    stack.append(y)
        if len({rows[x][2] for x in comp}) >= 2:
            best = max(sorted(comp), key=lambda x: (rows[x][5], -x))
            expect.append((best, len({rows[x][2] for x in comp}), min(iv[x][0] for x in comp), max(iv[x][1] for x in comp)))
    expect.sort()
    assert [(int(p["rep"]), int(p["nwidths_hit"]), int(p["t_begin"]), int(p["t_end"])) for p in got] == expect


def test_delay_range_pins(oracle):
    """Restricted delay search range ("the delay search range and the related FFT size is configured for
    projected baselines shorter than 3000 km"; A14): the argmax runs over the allowed delay bins only (a range
    that wraps through zero when lo > hi), the noise statistic stays the whole plane's."""
    w, nchan, nt, nf, a = 8, 32, 16, 64, 0.7
    tau, rho = 5.0, 2.0                              # on-bin fringe: peak at padded (r*, d*) = (4, 10)
    t, k = np.arange(w)[:, None], np.arange(nchan)[None, :]
    win = (a * np.exp(2j * np.pi * (tau * k / nchan + rho * t / w))).astype(np.complex64)
    full, _ = oracle.window(win, nt, nf)
    assert full["idx1"] == 4 * nf + 10
    for rg in [(0, nf - 1), (10, 10), (3, 20), (60, 12)]:         # ranges that contain d* = 10: nothing changes
        r, _ = oracle.window(win, nt, nf, delay_range=rg)
        assert (r["idx1"], r["p1"], r["s1"], r["snr"]) == (full["idx1"], full["p1"], full["s1"], full["snr"])
    # ranges that exclude d*: closed form |F[r][d]| = a |D_w(r/Nt - rho/w)| |D_nchan(d/Nf - tau/nchan)|, D_M(x) =
    # sin(pi M x)/sin(pi x); the rate factor peaks at r = 4 (value w), the delay factor decides among the allowed d
    def dirichlet(m, x):
        x = np.asarray(x, dtype=np.float64)
        den = np.sin(np.pi * x)
        return np.where(np.abs(den) < 1e-12, float(m), np.sin(np.pi * m * x) / np.where(np.abs(den) < 1e-12, 1.0, den))
    for rg in [(12, 30), (40, 8), (11, 11), (0, 9)]:
        lo, hi = rg
        cols = [d for d in range(nf) if (lo <= d <= hi if lo <= hi else (d >= lo or d <= hi))]
        amp = a * w * np.abs(dirichlet(nchan, np.array(cols) / nf - tau / nchan))
        best = int(np.argmax(amp))                   # first maximum = lowest d (cols ascend)
        r, _ = oracle.window(win, nt, nf, delay_range=rg)
        assert r["idx1"] == 4 * nf + cols[best], (rg, r["idx1"], cols[best])
        assert abs(r["p1"] - amp[best] ** 2) <= 1e-6 * max(amp[best] ** 2, 1.0)     # inputs are float32
        assert abs(r["s1"] - full["s1"]) <= 1e-9 * full["s1"]                       # Parseval: the noise is unchanged
        assert abs(r["snr"] - np.sqrt(r["p1"] / (full["s1"] / (nt * nf)))) <= 1e-12 * max(r["snr"], 1.0)
    # library special case on noise: numpy.fft2's plane, masked, in all three modes of a search
    rng = np.random.default_rng(21)
    vis = (rng.normal(size=(1, 2, 40, 12)) + 1j * rng.normal(size=(1, 2, 40, 12))).astype(np.complex64)
    widths, strides, nts, nf2 = [3, 8], [2, 5], [4, 16], 16
    for rg in [(2, 6), (13, 1), (7, 7)]:
        lo, hi = rg
        allowed = np.array([(lo <= d <= hi if lo <= hi else (d >= lo or d <= hi)) for d in range(nf2)])
        res = {m: oracle.search(vis, widths, strides, nts, nf2, mode=m, delay_range=rg)[0] for m in ("direct", "fft", "cached")}
        i = 0
        for pair in range(2):
            for wq, sq, ntq in zip(widths, strides, nts):
                for j in range(oracle.nwin(40, wq, sq)):
                    P = np.abs(np.fft.fft2(vis[0, pair, j * sq: j * sq + wq].astype(np.complex128), s=(ntq, nf2))) ** 2
                    Pm = np.where(allowed[None, :], P, -1.0)
                    for m in res:
                        r = res[m][i]
                        assert r["idx1"] == int(np.argmax(Pm)) and abs(r["p1"] - Pm.max()) <= 1e-9 * Pm.max()
                        assert abs(r["s1"] - P.sum()) <= 1e-9 * P.sum()
                    i += 1
    with pytest.raises(ValueError):
        oracle.window(win, nt, nf, delay_range=(0, nf))
    # f2 (all-IF): the same masked argmax on the nfa axis against numpy.fft of the summed band, noise unchanged
    v2 = (rng.normal(size=(1, 3, 20, 8)) + 1j * rng.normal(size=(1, 3, 20, 8))).astype(np.complex64)
    band = v2.transpose(0, 2, 1, 3).reshape(1, 20, 24)
    for rg in [(60, 3), (5, 30)]:
        res = oracle.allif_search(v2, [1, 4], [1, 2], 64, delay_range=rg)
        allowed = np.array([(d >= rg[0] or d <= rg[1]) if rg[0] > rg[1] else rg[0] <= d <= rg[1] for d in range(64)])
        i = 0
        for wq, sq in zip([1, 4], [1, 2]):
            for j in range(oracle.nwin(20, wq, sq)):
                P = np.abs(np.fft.fft(band[0, j * sq: j * sq + wq].astype(np.complex128).sum(axis=0), 64)) ** 2
                Pm = np.where(allowed, P, -1.0)
                assert res[i]["idx1"] == int(np.argmax(Pm)) and abs(res[i]["p1"] - Pm.max()) <= 1e-9 * Pm.max()
                assert abs(res[i]["s1"] - P.sum()) <= 1e-9 * P.sum()
                i += 1
    assert np.array_equal(oracle.allif_search(v2, [4], [2], 64, delay_range=(0, 63)), oracle.allif_search(v2, [4], [2], 64))


def test_baseline_match_constructions(oracle):
    """f3 pins ON THE ORACLE ("identified if it is detected with at least 5 baselines";
    DESIGN.md A19): hand-built pulse lists whose answer is fixed by the rule itself."""
    def run(rows, m):
        bl, tb, te, snr = (np.array(x) for x in zip(*rows))
        return oracle.baseline_match(bl, snr, tb, te, m)
    # five baselines, pairwise overlapping extents -> one detection; extent = union; rep = max snr
    five = [(b, 100 + b, 110 + b, 7.0 + b) for b in range(5)]
    d = run(five, 5)
    assert d == [dict(rep=4, nbaselines=5, t_begin=100, t_end=114)]
    # four of them -> dropped at min_baselines 5, kept at 4
    assert run(five[:4], 5) == []
    assert run(five[:4], 4) == [dict(rep=3, nbaselines=4, t_begin=100, t_end=113)]
    # the same baseline twice counts once
    rep = [(0, 10, 20, 8.0), (0, 12, 22, 9.0), (1, 15, 25, 7.0)]
    assert run(rep, 3) == []
    assert run(rep, 2) == [dict(rep=1, nbaselines=2, t_begin=10, t_end=25)]
    # chain: A and C do not overlap but both overlap B -> one cluster of 3 baselines; D is apart
    chain = [(0, 0, 10, 6.5), (1, 9, 20, 6.6), (2, 19, 30, 6.4), (3, 40, 50, 9.0)]
    assert run(chain, 3) == [dict(rep=1, nbaselines=3, t_begin=0, t_end=30)]
    assert [x["rep"] for x in run(chain, 1)] == [1, 3]
    # touching extents [0, 10) and [10, 20) do NOT link (half-open AP intervals)
    touch = [(0, 0, 10, 7.0), (1, 10, 20, 7.0)]
    assert run(touch, 2) == []
    assert [x["nbaselines"] for x in run(touch, 1)] == [1, 1]
    # ... one AP of overlap does
    assert run([(0, 0, 11, 7.0), (1, 10, 20, 7.0)], 2) == [dict(rep=0, nbaselines=2, t_begin=0, t_end=20)]
    # containment links; snr tie -> lowest index; output ordered by t_begin
    two = [(0, 300, 400, 7.0), (1, 350, 360, 7.0), (2, 100, 120, 9.0), (3, 110, 130, 8.0)]
    assert run(two, 2) == [dict(rep=2, nbaselines=2, t_begin=100, t_end=130), dict(rep=0, nbaselines=2, t_begin=300, t_end=400)]
    # input order must not matter (components of a graph): permute the chain
    perm = [chain[i] for i in (3, 2, 0, 1)]
    d = run(perm, 3)
    assert len(d) == 1 and (d[0]["nbaselines"], d[0]["t_begin"], d[0]["t_end"]) == (3, 0, 30) and perm[d[0]["rep"]][3] == 6.6
    assert oracle.baseline_match(np.zeros(0, int), np.zeros(0), np.zeros(0, int), np.zeros(0, int), 1) == []


def test_baseline_match_vs_sweep(oracle):
    """Independent statement of the same rule: interval-overlap components on a line are the maximal
    runs, in t_begin order, whose start lies before the running end (a sweep, no graph)."""
    rng = np.random.default_rng(12)
    for trial in range(30):
        n = int(rng.integers(1, 70))
        bl = rng.integers(0, 8, n)
        tb = rng.integers(0, 500, n)
        te = tb + rng.integers(1, 25, n)
        snr = rng.integers(60, 90, n) / 10.0
        got = oracle.baseline_match(bl, snr, tb, te, 3)
        order = sorted(range(n), key=lambda i: (tb[i], i))
        exp, i = [], 0
        while i < n:
            end, k, members = te[order[i]], i + 1, [order[i]]
            while k < n and tb[order[k]] < end:
                end = max(end, te[order[k]])
                members.append(order[k])
                k += 1
            if len({int(bl[m]) for m in members}) >= 3:
                best = max(sorted(members), key=lambda m: (snr[m], -m))
                exp.append(dict(rep=best, nbaselines=len({int(bl[m]) for m in members}), t_begin=int(tb[order[i]]), t_end=int(end)))
            i = k
        exp.sort(key=lambda d: (d["t_begin"], d["rep"]))
        assert got == exp


def test_dedispersion_pins(oracle):
    """f1: per frequency point a time shift.  Pins: zero shift is the identity; a
    pulse dispersed by known shifts is restored sample for sample; samples shifted in from beyond the
    end are zero; the textbook delay 4.148808 ms DM (f^-2 - f_ref^-2) at a hand-computed point."""
    rng = np.random.default_rng(5)
    nbl, nif, nap, nchan = 2, 3, 40, 8
    clean = (rng.normal(size=(nbl, nif, nap, nchan)) + 1j * rng.normal(size=(nbl, nif, nap, nchan))).astype(np.complex64)
    assert np.array_equal(oracle.dedisperse(clean, np.zeros((nif, nchan), np.int32)), clean)
    sh = rng.integers(0, 7, size=(nif, nchan)).astype(np.int32)
    disp = np.zeros_like(clean)                      # channel k arrives sh[k] APs late
    for n in range(nif):
        for k in range(nchan):
            d = int(sh[n, k])
            disp[:, n, d:, k] = clean[:, n, :nap - d, k]
    back = oracle.dedisperse(disp, sh)
    for n in range(nif):
        for k in range(nchan):
            d = int(sh[n, k])
            assert np.array_equal(back[:, n, :nap - d, k], clean[:, n, :nap - d, k])
            assert np.all(back[:, n, nap - d:, k] == 0)
    # DM 100 pc cm^-3, 1400 MHz against 1500 MHz: 4.148808e-3 s * 100 * (1/1.4^2 - 1/1.5^2) = 27.2821 ms
    d = oracle.dm_shifts(100.0, np.array([[1400.0, 1500.0]]), 1500.0, 1e-3)
    assert d.tolist() == [[27, 0]]
    assert abs(4.148808e-3 * 100 * (1 / 1.4 ** 2 - 1 / 1.5 ** 2) - 0.0272821) < 1e-6


def test_dedispersed_pulse_closed_form(oracle):
    """A noiseless on-bin fringe, dispersed channel by channel, then dedispersed with the matching
    shifts, peaks where the undispersed one does with P1 = (a w nchan)^2 (pin P1 through step 4)."""
    w, nchan, nt, nf, a, tau, rho = 8, 16, 16, 32, 0.7, 3, 2
    nap, tp = 64, 20
    t = np.arange(w)[:, None]
    k = np.arange(nchan)[None, :]
    pulse = (a * np.exp(2j * np.pi * (tau * k / nchan + rho * t / w))).astype(np.complex64)
    sh = (np.arange(nchan)[::-1] // 2).astype(np.int32).reshape(1, nchan)     # low channels later
    vis = np.zeros((1, 1, nap, nchan), np.complex64)
    for kk in range(nchan):
        d = int(sh[0, kk])
        vis[0, 0, tp + d: tp + d + w, kk] = pulse[:, kk]
    ded = oracle.dedisperse(vis, sh)
    pk, _ = oracle.search(ded, [w], [1], [nt], nf, mode="fft")
    o = pk[tp]
    assert o["idx1"] == (rho * nt // w) * nf + tau * nf // nchan
    assert abs(o["p1"] - (a * w * nchan) ** 2) < 1e-6 * o["p1"]
    raw, _ = oracle.search(vis, [w], [1], [nt], nf, mode="fft")
    assert raw["p1"].max() < 0.5 * o["p1"]            # without step 4 the pulse is smeared


def test_zscore_selection_pins(oracle):
    """f4: hand-computed series.  P1 = [1, 1, 1, 1, 9]: mean 2.6, population std 3.2 -> z = [-0.5]*4 + [2.0];
    strict threshold; a constant series (std 0) selects nothing; series of different (pair, width) are
    normalised separately."""
    def peaks_of(p):
        pk = np.zeros(len(p), dtype=oracle.PEAK_DTYPE)
        pk["p1"] = p
        pk["idx1"] = 7
        return pk
    c, z = oracle.zscore_candidates(peaks_of([1, 1, 1, 1, 9]), 1, 1, 5, [1], [1], 4, 1.9)
    assert np.allclose(z, [-0.5, -0.5, -0.5, -0.5, 2.0]) and len(c) == 1 and c[0]["win"] == 4 and c[0]["snr"] == 2.0
    assert (c[0]["rate_idx"], c[0]["delay_idx"]) == (1, 3)
    assert len(oracle.zscore_candidates(peaks_of([1, 1, 1, 1, 9]), 1, 1, 5, [1], [1], 4, 2.0)[0]) == 0   # strict >
    assert len(oracle.zscore_candidates(peaks_of([3, 3, 3, 3, 3]), 1, 1, 5, [1], [1], 4, 0.0)[0]) == 0
    # two pairs x two widths (nap = 4: widths 1 and 2 -> 4 + 3 windows per pair)
    p = [1, 1, 1, 9,   2, 2, 8,    5, 5, 5, 5,   0, 10, 0]
    c, z = oracle.zscore_candidates(peaks_of(p), 2, 1, 4, [1, 2], [1, 1], 4, 1.0)
    assert np.allclose(z[:4], (np.array([1, 1, 1, 9]) - 3) / np.std([1, 1, 1, 9]))
    assert np.allclose(z[7:11], 0) and np.allclose(z[11:], (np.array([0, 10, 0]) - 10 / 3) / np.std([0, 10, 0]))
    assert [(int(r["bl"]), int(r["wid"]), int(r["win"])) for r in c] == [(0, 0, 3), (0, 1, 2), (1, 1, 1)]


def test_allif_search_pins(oracle):
    """f2 (Eq. 1).  Closed form: a noiseless fringe with one delay across all IFs,
    S = a e^{+2 pi i tau m / (nif nchan)} on every AP of the window, peaks at d = tau nfa/(nif nchan) with
    P1 = (a w nif nchan)^2 and snr = sqrt(nif nchan); the sign-flipped fringe must land at -tau.  Library
    special case: numpy.fft.fft of the time-summed band.  Parseval: S1 = nfa sum_m |sum_t S|^2.  A delay
    that is NOT common to the IFs (a per-IF fringe restarting its phase in every IF) must not reach that peak."""
    nbl, nif, nap, nchan, w, nfa, a, tau = 2, 4, 12, 8, 4, 128, 0.5, 5
    m = np.arange(nif * nchan)
    fr = (a * np.exp(2j * np.pi * tau * m / (nif * nchan))).astype(np.complex64).reshape(nif, 1, nchan)
    vis = np.zeros((nbl, nif, nap, nchan), np.complex64)
    vis[0, :, 3:3 + w, :] = fr
    vis[1, :, 3:3 + w, :] = np.conj(fr)
    pk = oracle.allif_search(vis, [w], [1], nfa)
    nwin = nap - w + 1
    o = pk[3]
    assert o["idx1"] == tau * nfa // (nif * nchan) and abs(o["p1"] - (a * w * nif * nchan) ** 2) < 1e-6 * o["p1"]   # complex64 inputs
    assert abs(o["snr"] - np.sqrt(nif * nchan)) < 1e-6
    assert pk[nwin + 3]["idx1"] == nfa - tau * nfa // (nif * nchan)
    rng = np.random.default_rng(11)
    noise = (rng.normal(size=vis.shape) + 1j * rng.normal(size=vis.shape)).astype(np.complex64)
    pk = oracle.allif_search(noise, [w, 2], [3, 1], nfa)
    band = oracle.allif_band(noise).astype(np.complex128)
    k = 0
    for b in range(nbl):
        for ww, s in ((w, 3), (2, 1)):
            for j in range((nap - ww) // s + 1):
                ref = np.abs(np.fft.fft(band[b, j * s: j * s + ww].sum(axis=0), nfa)) ** 2
                assert pk[k]["idx1"] == int(np.argmax(ref)) and abs(pk[k]["p1"] - ref.max()) < 1e-9 * ref.max()
                assert abs(pk[k]["s1"] - nfa * (np.abs(band[b, j * s: j * s + ww].sum(axis=0)) ** 2).sum()) < 1e-9 * pk[k]["s1"]
                k += 1
    assert k == len(pk)
    per_if = np.zeros((1, nif, nap, nchan), np.complex64)
    # phase restarting in every IF with a half-integer per-IF delay: adjacent IFs are pi apart
    per_if[0, :, 3:3 + w, :] = (a * np.exp(2j * np.pi * 2.5 * np.arange(nchan) / nchan)).astype(np.complex64)
    assert oracle.allif_search(per_if, [w], [1], nfa)[3]["p1"] < 0.9 * (a * w * nif * nchan) ** 2


def test_initial_calibration_pins(oracle):
    """Eq. 1's calibration terms.  A band-coherent fringe corrupted by per-IF
    delays and phases ("the large IF delay ... discrepancies of initial delay and phase between IFs")
    loses coherence across IFs; multiplying by cal_phasors of the same values restores the closed-form
    all-IF peak P1 = (a w nif nchan)^2 at the injected delay ("after calibration, fringe phase become
    flat and aligned across IFs").  Zero delay and phase give unit phasors; a pure phase is a constant."""
    nbl, nif, nap, nchan, w, nfa, a, tau = 1, 4, 10, 16, 4, 256, 0.8, 3
    chan_hz = 16e6 / nchan
    rng = np.random.default_rng(3)
    d0 = rng.uniform(-40e-9, 40e-9, (nbl, nif))
    p0 = rng.uniform(-np.pi, np.pi, (nbl, nif))
    assert np.allclose(oracle.cal_phasors(np.zeros((1, 2)), np.zeros((1, 2)), 8, 1e6), 1.0)
    c = oracle.cal_phasors(np.zeros((1, 1)), np.full((1, 1), 0.5), 8, 1e6)
    assert np.allclose(c, np.exp(-0.5j), atol=1e-7)
    m = np.arange(nif * nchan).reshape(nif, 1, nchan)
    clean = a * np.exp(2j * np.pi * tau * m / (nif * nchan))
    j = np.arange(nchan)[None, None, :]
    corrupt = clean * np.exp(1j * (2 * np.pi * (j * chan_hz) * d0[0][:, None, None] + p0[0][:, None, None]))
    vis = np.zeros((nbl, nif, nap, nchan), np.complex64)
    vis[0, :, 2:2 + w, :] = corrupt.astype(np.complex64)
    before = oracle.allif_search(vis, [w], [1], nfa)[2]
    cal = oracle.cal_phasors(d0, p0, nchan, chan_hz)
    after = oracle.allif_search(oracle.calibrate(vis, cal), [w], [1], nfa)[2]
    full = (a * w * nif * nchan) ** 2
    assert abs(after["p1"] - full) < 1e-5 * full and after["idx1"] == tau * nfa // (nif * nchan)
    assert before["p1"] < 0.8 * full
