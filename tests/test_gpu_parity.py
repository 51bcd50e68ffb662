"""Parity of the CUDA path (through the C-ABI binding) against the float64 oracle on the same
seeded inputs.  Needs a GPU (B200)."""
import numpy as np
import pytest
import torch

import workloads
from _parity import (allif_plane_power, canonical_index, check_candidate_bins, check_candidates, check_peaks,
                     dense_index)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def vb():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2108_05602_b200 as v
    v.lib()          # must load: no fallback
    return v


def make_plane_power(oracle, vis_np, c):
    """Oracle power of one bin of one canonical window (recomputes that window's plane)."""
    nbl, nif, nap, nchan = vis_np.shape
    bl, ifq, wid, win, t0 = oracle.canonical_table(nbl, nif, nap, c["widths"], c["strides"])

    def plane_power(i, idx):
        q = int(wid[i])
        slab = vis_np[bl[i], ifq[i], t0[i]: t0[i] + c["widths"][q]]
        _, plane = oracle.window(slab, c["nts"][q], c["nf"], mode="fft", want_plane=True)
        z = plane.reshape(-1)[idx]
        return float(z.real * z.real + z.imag * z.imag)
    return plane_power


def run_both(vb, oracle, vis, c, thresh=None, mode="cached", options=None, delay_range=None):
    thresh = c["snr_thresh"] if thresh is None else thresh
    nbl, nif, nap, nchan = vis.shape
    if delay_range is not None:
        options = dict(options or {}, delay_lo=delay_range[0], delay_hi=delay_range[1])
    cands, n, peaks = vb.fringe_search(vis.cuda(), c["widths"], c["strides"], c["nts"], c["nf"], thresh,
                                       want_peaks=True, options=options)
    # the same search without the dense peak array: the candidates-only index mode (volks_options.full_index = 0:
    # untagged / pruned / folded-sum kernels); its list is pinned to the ORACLE below by the same rules
    cands2, n2, _ = vb.fringe_search(vis.cuda(), c["widths"], c["strides"], c["nts"], c["nf"], thresh, options=options)
    assert n2 == len(cands2)
    ora, _ = oracle.search(vis.cpu().numpy(), c["widths"], c["strides"], c["nts"], c["nf"], mode=mode, delay_range=delay_range)
    nw = [workloads.gen.nwin(nap, w, s) for w, s in zip(c["widths"], c["strides"])]
    di = dense_index(nbl, nif, nw)
    assert len(ora) == len(peaks) == len(di)
    stats = check_peaks(peaks[di], ora, c["nf"], make_plane_power(oracle, vis.cpu().numpy(), c))
    oc, keep = oracle.candidates(ora, nbl, nif, nap, c["widths"], c["strides"], c["nf"], thresh)
    assert n == len(cands)
    ncand, nmarg = check_candidates(cands, oc, ora, keep, thresh, c["nf"])
    # candidates-only mode: the same windows (marginal ones aside), each record's bin / power / snr against the oracle
    check_candidates(cands2, oc, ora, keep, thresh, c["nf"])
    cidx2 = canonical_index(cands2, nif, nw)
    check_candidate_bins(cands2, cidx2, ora, c["nf"], make_plane_power(oracle, vis.cpu().numpy(), c))
    assert abs(n2 - n) <= nmarg
    if n2 == n and np.array_equal(cidx2, canonical_index(cands, nif, nw)):
        # between the modes: identical windows; bins equal unless the oracle calls it a near-tie; powers to 2e-4 (each
        # mode is held to 1e-4 of the oracle above)
        safe = np.where(ora["p1"][cidx2] > 0, ora["p1"][cidx2], 1.0)
        tie = (ora["p1"][cidx2] - ora["p2"][cidx2]) / safe < 1e-5
        same = (cands2["rate_idx"] == cands["rate_idx"]) & (cands2["delay_idx"] == cands["delay_idx"])
        assert np.all(same | tie)
        assert np.all(np.abs(cands2["power"].astype(np.float64) - cands["power"]) <= 2e-4 * np.maximum(cands["power"], 1e-30))
    return stats, ncand, cands, ora


def test_config0_full(vb, oracle):
    vis, c, _ = workloads.generate(0)
    stats, ncand, cands, ora = run_both(vb, oracle, vis, c)
    assert ncand >= 1 and all(cands["rate_idx"] == 4) and all(cands["delay_idx"] == 10)


def test_config1_full(vb, oracle):
    vis, c, _ = workloads.generate(1)
    stats, ncand, cands, ora = run_both(vb, oracle, vis, c)
    assert ncand >= 1


@pytest.mark.parametrize("cfg,over", [
    (2, dict(nbl=2, nif=1, nap=400, npulses=3)),
    (3, dict(nbl=3, nif=2, nap=1000, npulses=4)),
    (4, dict(nbl=1, nif=1, nap=600, npulses=1)),
])
def test_reduced_configs(vb, oracle, cfg, over):
    """configs 2-4 at reduced extent (same nchan / widths / strides / padding): several tiles and a
    ragged tail, every window compared."""
    vis, c, _ = workloads.generate(cfg, **over)
    run_both(vb, oracle, vis, c)
    run_both(vb, oracle, vis, c, thresh=3.0)      # PAPER.md:196 stress threshold


@pytest.mark.parametrize("cfg,over", [
    (2, dict(nbl=1, nif=2, nap=700, npulses=3)),
    (3, dict(nbl=2, nif=2, nap=900, npulses=4)),
])
def test_generic_and_sliding_paths_agree_with_oracle(vb, oracle, cfg, over):
    """The same stride-1 inputs through the generic kernels (volks_options.force_generic) and through the
    sliding-sum kernels with a short restart interval (several segments + a ragged tail)."""
    vis, c, _ = workloads.generate(cfg, **over)
    run_both(vb, oracle, vis, c, options=dict(force_generic=1))
    run_both(vb, oracle, vis, c, thresh=3.0, options=dict(slide_seg=128))
    run_both(vb, oracle, vis, c, options=dict(slide_seg=1024))
    run_both(vb, oracle, vis, c, options=dict(full_index=1))


@pytest.mark.parametrize("shape", [
    # nbl nif nap nchan widths strides nts nf
    (1, 1, 40, 20, [1, 3, 5], [1, 2, 7], [2, 4, 8], 32),       # ragged: non-pow2 nchan / widths, stride > w
    (2, 1, 33, 5, [2, 4], [1, 3], [2, 4], 8),                  # tiny planes (M*nf < 32 path), nt == w
    (1, 2, 10, 8, [4, 16], [1, 1], [8, 16], 8),                # nap < w for one width -> zero windows
    (1, 1, 70, 64, [8], [4], [64], 64),                        # pad x8 in time
    (1, 1, 50, 3, [2], [1], [4], 4),                           # nf = 4
    (1, 1, 17, 1, [4], [1], [8], 1),                           # single channel, nf = 1
    (1, 1, 300, 100, [32, 64], [5, 9], [64, 128], 512),        # big nf, odd strides
    (1, 1, 90, 300, [16, 40], [8, 10], [32, 64], 1024),        # nf = 1024 row kernel, pruned inputs
    (1, 1, 70, 2048, [8], [1], [16], 2048),                    # nf = 2048, nchan = nf (no pruning)
])
def test_edge_shapes(vb, oracle, shape):
    nbl, nif, nap, nchan, widths, strides, nts, nf = shape
    g = torch.Generator().manual_seed(nap * 7 + nchan)
    vis = torch.view_as_complex(torch.randn((nbl, nif, nap, nchan, 2), generator=g) * 0.7071)
    c = dict(widths=widths, strides=strides, nts=nts, nf=nf, snr_thresh=2.5)
    run_both(vb, oracle, vis, c, mode="fft")


@pytest.mark.parametrize("shape", [
    # stride-1, pad x2 widths on nf >= 64: the sliding-sum kernels (every L / M variant), ragged tails
    (1, 1, 20, 33, [2, 4, 8], [1, 1, 1], [4, 8, 16], 64),        # fewer windows than one unrolled block
    (2, 1, 47, 64, [16, 32], [1, 1], [32, 64], 64),              # M = 2, 4; nwin = 32, 16
    (1, 2, 300, 40, [2, 64, 128], [1, 1, 1], [4, 128, 256], 128),  # M = 8, 16; segment seam at 256
    (1, 1, 530, 17, [8, 16], [1, 1], [16, 32], 256),             # several column groups per CTA
])
def test_sliding_kernel_shapes(vb, oracle, shape):
    nbl, nif, nap, nchan, widths, strides, nts, nf = shape
    g = torch.Generator().manual_seed(nap * 11 + nchan)
    vis = torch.view_as_complex(torch.randn((nbl, nif, nap, nchan, 2), generator=g) * 0.7071)
    vis[0, 0, nap // 2: nap // 2 + 5] += 1.5 + 0.5j              # a coherent burst (a clear peak)
    c = dict(widths=widths, strides=strides, nts=nts, nf=nf, snr_thresh=2.5)
    run_both(vb, oracle, vis, c, mode="fft")


@pytest.mark.parametrize("cf2", ["4", "2", "1", "0"])
@pytest.mark.parametrize("shape", [
    # Nt = 256 / 512 with stride != 1 or pad != 2: k_colfft2 (16- and 32-column strips) and k_colfft, every NZ
    (1, 2, 300, 20, [1, 20, 40], [3, 7, 16], [256, 256, 512], 32),        # NZ = 1, 2, 4; one 32-column tile
    (1, 1, 700, 50, [100, 200, 256], [25, 64, 100], [512, 256, 256], 64), # NZ = 8, 16, 16 (nt == w: no padding)
    (2, 1, 600, 33, [300, 512], [50, 30], [512, 512], 128),               # NZ = 32 (nt == w), several strips
])
def test_colfft2_variants(vb, oracle, shape, cf2):
    """The two-columns-per-thread rate kernel (kernels_colfft2.cuh) in both strip widths, and the kernel it
    replaced, against the oracle on the same inputs: every pruning depth NZ, windows of one CTA range,
    a burst that gives a clear peak, and an all-zero span (tie-break -> index 0)."""
    opts = dict(cf2=int(cf2), cf_wpc=8)                                   # several window ranges per strip
    nbl, nif, nap, nchan, widths, strides, nts, nf = shape
    g = torch.Generator().manual_seed(nap * 13 + nchan)
    vis = torch.view_as_complex(torch.randn((nbl, nif, nap, nchan, 2), generator=g) * 0.7071)
    k = torch.arange(nchan)
    vis[0, 0, nap // 3: nap // 3 + 30] += 0.8 * torch.exp(2j * np.pi * 3.0 * k / nf)   # delay bin 3
    vis[0, 0, : 40] = 0                                                   # flagged span at the start
    c = dict(widths=widths, strides=strides, nts=nts, nf=nf, snr_thresh=2.5)
    run_both(vb, oracle, vis, c, mode="fft", options=opts)
    # run to run bit-identical (the two parity pipelines of a CTA meet only in the ordered key maximum)
    ref = None
    for _ in range(3):
        cands, n, peaks = vb.fringe_search(vis.cuda(), widths, strides, nts, nf, 2.5, want_peaks=True, options=opts)
        blob = (peaks.tobytes(), cands.tobytes())
        assert ref is None or blob == ref
        ref = blob


def test_zero_windows_and_empty(vb):
    vis = torch.zeros((1, 1, 3, 8), dtype=torch.complex64)
    cands, n, peaks = vb.fringe_search(vis.cuda(), [4], [1], [8], 8, 6.0, want_peaks=True)
    assert n == 0 and len(cands) == 0 and len(peaks) == 0


def test_degenerate_inputs_tie_break(vb, oracle):
    """A8: all-zero windows (snr 0, argmax (0,0)); a delta input (constant plane -> (0,0), snr 1);
    w = 1 (identical rate rows -> r* = 0)."""
    vis = torch.zeros((1, 1, 64, 32), dtype=torch.complex64)
    vis[0, 0, 20, 0] = 2 - 1j      # channel 0: every delay twiddle is exactly 1
    c = dict(widths=[1, 8], strides=[1, 1], nts=[2, 16], nf=64, snr_thresh=0.5)
    cands, n, peaks = vb.fringe_search(vis.cuda(), c["widths"], c["strides"], c["nts"], c["nf"], 0.5, want_peaks=True)
    hit = peaks["power"] > 0
    assert np.allclose(peaks["power"][hit], 5.0, rtol=1e-6) and np.allclose(peaks["snr"][hit], 1.0, rtol=1e-6)
    assert np.all(peaks["snr"][~hit] == 0) and hit.sum() == 1 + 8 and n == 9
    # all-zero windows: constant plane, first index wins
    assert np.all(peaks["rate_idx"][~hit] == 0) and np.all(peaks["delay_idx"][~hit] == 0)
    # exactly constant planes (all twiddles exactly 1): w = 1 at AP 20, and w = 8 starting at AP 20
    assert tuple(peaks[20][["rate_idx", "delay_idx"]]) == (0, 0)
    assert tuple(peaks[64 + 20][["rate_idx", "delay_idx"]]) == (0, 0)
    g = torch.Generator().manual_seed(3)
    v1 = torch.view_as_complex(torch.randn((1, 1, 50, 32, 2), generator=g))
    cands, n, peaks = vb.fringe_search(v1.cuda(), [1], [1], [2], 128, 6.0, want_peaks=True)
    assert np.all(peaks["rate_idx"] == 0)
    ora, _ = oracle.search(v1.numpy(), [1], [1], [2], 128, mode="fft")
    assert np.array_equal(peaks["delay_idx"], ora["idx1"] % 128)


def test_capacity_overflow_and_determinism(vb):
    vis, c, _ = workloads.generate(1, nap=500)
    v = vis.cuda()
    a, na, pa = vb.fringe_search(v, c["widths"], c["strides"], c["nts"], c["nf"], 3.0, want_peaks=True)
    b, nb, pb = vb.fringe_search(v, c["widths"], c["strides"], c["nts"], c["nf"], 3.0, want_peaks=True)
    assert na == nb and a.tobytes() == b.tobytes() and pa.tobytes() == pb.tobytes()   # bit-identical
    assert na > 10
    s, ns, _ = vb.fringe_search(v, c["widths"], c["strides"], c["nts"], c["nf"], 3.0, cand_capacity=7)
    assert ns == na and len(s) == 7 and s.tobytes() == a[:7].tobytes()                # true count, first 7
    z, nz, _ = vb.fringe_search(v, c["widths"], c["strides"], c["nts"], c["nf"], 3.0, cand_capacity=0)
    assert nz == na and len(z) == 0


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,over", [
    (2, dict(nbl=2, nif=2, nap=3000, npulses=6)),    # pruned widths, k_pairfold + k_coleval, the folded sliding sum + its list
    (3, dict(nbl=2, nif=2, nap=4000, npulses=6)),    # k_row128, all widths pruned
    (4, dict(nbl=1, nif=2, nap=2500, npulses=3)),    # k_colfft2e (flags between the parity halves), k_colfft2<SKIP>
])
def test_candidates_only_mode_is_deterministic(vb, cfg, over):
    """The candidates-only search (atomics into lists and flags, independently running CTA halves) must give the same
    bytes run after run: five searches of one plan and a fresh plan, threshold 6 (every bound active)."""
    vis, c, _ = workloads.generate(cfg, **over)
    v = vis.cuda()
    ref = None
    for _ in range(6):
        a, na, _ = vb.fringe_search(v, c["widths"], c["strides"], c["nts"], c["nf"], c["snr_thresh"])
        assert na == len(a) and na > 0
        if ref is None:
            ref = a.tobytes()
        assert a.tobytes() == ref


def test_peaks_optional_same_candidates(vb):
    vis, c, _ = workloads.generate(0)
    a, na, _ = vb.fringe_search(vis.cuda(), c["widths"], c["strides"], c["nts"], c["nf"], 6.0, want_peaks=False)
    b, nb, _ = vb.fringe_search(vis.cuda(), c["widths"], c["strides"], c["nts"], c["nf"], 6.0, want_peaks=True)
    assert na == nb and a.tobytes() == b.tobytes()


def test_non_default_stream(vb):
    vis, c, _ = workloads.generate(0)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        a, na, _ = vb.fringe_search(vis.cuda(), c["widths"], c["strides"], c["nts"], c["nf"], 6.0)
    b, nb, _ = vb.fringe_search(vis.cuda(), c["widths"], c["strides"], c["nts"], c["nf"], 6.0)
    assert na == nb and a.tobytes() == b.tobytes()


def test_cpu_tensor_is_rejected_loudly(vb):
    vis, c, _ = workloads.generate(0)
    with pytest.raises(RuntimeError):
        vb.fringe_search(vis, c["widths"], c["strides"], c["nts"], c["nf"], 6.0)


def test_window_match_on_gpu_candidates(vb, oracle):
    vis, c, _ = workloads.generate(1)
    cands, n, _ = vb.fringe_search(vis.cuda(), c["widths"], c["strides"], c["nts"], c["nf"], 4.0)
    got = vb.window_match(cands, c["widths"], 2)
    oc = np.zeros(len(cands), dtype=oracle.CAND_DTYPE)
    for k in ("bl", "ifq", "wid", "win", "t0", "snr"):
        oc[k] = cands[k]
    exp = oracle.window_match(oc, c["widths"], 2)
    assert len(got) == len(exp) and len(got) >= 1
    for g, e in zip(got, exp):
        assert g["best"].tobytes() == cands[int(e["rep"])].tobytes()
        assert (g["nwidths_hit"], g["t_begin"], g["t_end"]) == (e["nwidths_hit"], e["t_begin"], e["t_end"])


@pytest.mark.parametrize("cfg,over", [
    (2, dict(nbl=1, nif=2, nap=500, npulses=2)),      # k_row2 + sliding kernels
    (4, dict(nbl=1, nif=1, nap=700, npulses=1)),      # k_row3 + column FFT
    (1, dict(nap=600)),                               # k_row2 (nf = 128) + generic / column FFT
])
def test_dedispersed_search_matches_oracle(vb, oracle, cfg, over):
    """f1: dedispersion fused into the slab load == oracle.dedisperse followed by the plain search."""
    vis, c, _ = workloads.generate(cfg, **over)
    nbl, nif, nap, nchan = vis.shape
    f = 1400.0 + 16.0 * np.arange(nif)[:, None] + (16.0 / nchan) * np.arange(nchan)[None, :]
    sh = vb.dm_shifts(300.0, f, f.max(), c["t_ap"])
    assert sh.max() > 3 and sh.min() == 0
    cands, n, peaks = vb.fringe_search(vis.cuda(), c["widths"], c["strides"], c["nts"], c["nf"], c["snr_thresh"],
                                       want_peaks=True, shifts=sh)
    ded = oracle.dedisperse(vis.numpy(), sh)
    ora, _ = oracle.search(ded, c["widths"], c["strides"], c["nts"], c["nf"], mode="cached")
    nw = [workloads.gen.nwin(nap, w, s) for w, s in zip(c["widths"], c["strides"])]
    check_peaks(peaks[dense_index(nbl, nif, nw)], ora, c["nf"], make_plane_power(oracle, ded, c))
    oc, keep = oracle.candidates(ora, nbl, nif, nap, c["widths"], c["strides"], c["nf"], c["snr_thresh"])
    check_candidates(cands, oc, ora, keep, c["snr_thresh"], c["nf"])
    # negative shifts and shifts past the end are legal: zero fill
    sh2 = sh.copy(); sh2[0, 0] = -5; sh2[-1, -1] = nap + 3
    _, _, p2 = vb.fringe_search(vis.cuda(), c["widths"], c["strides"], c["nts"], c["nf"], c["snr_thresh"], want_peaks=True, shifts=sh2)
    ora2, _ = oracle.search(oracle.dedisperse(vis.numpy(), sh2), c["widths"], c["strides"], c["nts"], c["nf"], mode="cached")
    check_peaks(p2[dense_index(nbl, nif, nw)], ora2, c["nf"], make_plane_power(oracle, oracle.dedisperse(vis.numpy(), sh2), c))


def test_flagged_zero_span_inside_data(vb, oracle):
    """Exact zeros (flagged APs) after ordinary data: windows inside the span have an identically
    zero plane (P1 = 0 at (0,0), snr 0) - the sliding sum must not leak rounding residue there."""
    vis, c, _ = workloads.generate(2, nbl=1, nif=1, nap=700, npulses=2)
    vis[0, 0, 300:420] = 0
    stats, ncand, cands, ora = run_both(vb, oracle, vis, c)
    assert np.count_nonzero(ora["p1"] == 0) > 100


def test_detection_chain_on_gpu_candidates(vb, oracle):
    """a7 -> a8 -> f3 on config 2 at reduced extent (10 baselines): candidates -> per-baseline
    multi-window match -> multi-baseline cross-match (>= 5 baselines).  The host chain
    must equal the oracle chain on the same candidates, find the station-consistent injected pulses
    and drop the single-baseline RFI."""
    vis, c, truth = workloads.generate(2, nbl=10, nif=1, nap=3000, npulses=4)
    cands, n, _ = vb.fringe_search(vis.cuda(), c["widths"], c["strides"], c["nts"], c["nf"], c["snr_thresh"])
    pulses = vb.window_match(cands, c["widths"], 2)
    dets = vb.baseline_match(pulses, 5)
    exp = oracle.baseline_match(pulses["best"]["bl"], pulses["best"]["snr"], pulses["t_begin"], pulses["t_end"], 5)
    assert len(dets) == len(exp)
    for d, e in zip(dets, exp):
        assert d["best"].tobytes() == pulses[e["rep"]].tobytes()
        assert (d["nbaselines"], d["t_begin"], d["t_end"]) == (e["nbaselines"], e["t_begin"], e["t_end"])
    strong = [p for p in truth["pulses"] if p["amp"] * np.sqrt(p["width"] * c["nchan"]) >= 1.5 * c["snr_thresh"] and p["width"] >= 4]
    assert strong, "the reduced workload must contain a detectable pulse"
    for p in strong:
        assert any(d["t_begin"] < p["t0"] + p["width"] and p["t0"] < d["t_end"] for d in dets), p
    assert all(d["nbaselines"] >= 5 for d in dets)
    # only the injected pulses are common to >= 5 baselines: every detection must sit on one of them
    for d in dets:
        assert any(d["t_begin"] < p["t0"] + p["width"] + 64 and p["t0"] - 64 < d["t_end"] for p in truth["pulses"]), d


@pytest.mark.parametrize("cfg,over", [(2, dict(nbl=2, nif=1, nap=900, npulses=3)), (1, dict(nap=700))])
def test_zscore_selection_matches_oracle(vb, oracle, cfg, over):
    """f4: across-window normalised power on the workspace of the last search vs the oracle's
    definition applied to the oracle's peaks (z within 1e-4 of the z scale; list identical except
    windows whose oracle z lies within that margin of the threshold)."""
    vis, c, _ = workloads.generate(cfg, **over)
    nbl, nif, nap, nchan = vis.shape
    # the z-score pass needs every window's exact index from the search before it: volks_options.full_index
    plan = vb.Plan(nbl, nif, nap, nchan, c["widths"], c["strides"], c["nts"], c["nf"], c["snr_thresh"],
                   options=dict(full_index=1))
    dev = torch.device("cuda")
    ws = torch.empty(plan.workspace_bytes, dtype=torch.uint8, device=dev)
    cap = 1 << 16
    cands = torch.empty(cap * vb.CAND_DTYPE.itemsize, dtype=torch.uint8, device=dev)
    ncand = torch.zeros(1, dtype=torch.int32, device=dev)
    peaks = torch.empty(plan.nwin_total * vb.PEAK_DTYPE.itemsize, dtype=torch.uint8, device=dev)
    plan.fringe_search(vis.cuda(), ws, cands, ncand)
    zth = 3.0
    plan.zscore_select(ws, zth, cands, ncand, peaks)
    torch.cuda.synchronize()
    n = int(ncand.item())
    got = cands[: n * vb.CAND_DTYPE.itemsize].cpu().numpy().view(vb.CAND_DTYPE)
    pk = peaks.cpu().numpy().view(vb.PEAK_DTYPE)
    ora, _ = oracle.search(vis.numpy(), c["widths"], c["strides"], c["nts"], c["nf"], mode="cached")
    exp, z = oracle.zscore_candidates(ora, nbl, nif, nap, c["widths"], c["strides"], c["nf"], zth)
    nw = [workloads.gen.nwin(nap, w, s) for w, s in zip(c["widths"], c["strides"])]
    gz = pk[dense_index(nbl, nif, nw)]["snr"].astype(np.float64)
    tol = 1e-4 * max(1.0, np.abs(z).max())
    assert np.abs(gz - z).max() <= tol
    key = lambda r: (int(r["bl"]), int(r["ifq"]), int(r["wid"]), int(r["win"]))
    gk, ek = [key(r) for r in got], [key(r) for r in exp]
    assert gk == sorted(gk) and n >= 1
    marginal = {k for k, zz in zip([key(r) for r in exp], exp["snr"]) if abs(zz - zth) <= tol}
    assert set(ek) - set(gk) <= marginal
    for r in got:
        if key(r) not in set(ek):
            assert abs(float(r["snr"]) - zth) <= 2 * tol
    plan.close()


@pytest.mark.parametrize("shape", [
    # nbl nif nap nchan widths strides nfa dm
    (2, 4, 300, 32, [2, 8, 16], [1, 1, 1], 256, 0.0),      # k_row2, sliding windows, several segments? (seg 256)
    (1, 8, 700, 64, [4, 32], [1, 1], 2048, 0.0),           # pad x4 like the paper (8 IF x 64 ch x 4), k_row3
    (2, 2, 200, 100, [3, 10], [2, 5], 512, 0.0),           # ragged band (200 of 512): direct sums (2s > w) and stride-5 sliding
    (1, 2, 900, 32, [64, 16], [16, 4], 128, 0.0),          # config-4-like strides w/4: sliding by blocks over several segments
    (1, 4, 400, 32, [4, 16], [1, 1], 256, 300.0),          # dedispersed all-IF search
    (1, 2, 120, 1024, [8], [1], 4096, 0.0),                # nfa = 4096: generic row kernel, 2 column pairs per thread
    (1, 2, 40, 1024, [4], [1], 16384, 0.0),                # nfa = 16384 = 2 interleaved 8192-point transforms
    (2, 8, 26, 1024, [2, 4], [1, 1], 32768, 0.0),          # the paper's shape: 8 IF x 1024 x pad 4
    (1, 8, 30, 512, [4], [2], 32768, 300.0),               # pad x8, dedispersed, stride 2
    (2, 4, 150, 64, [1, 4], [1, 2], 1024, 0.0),            # w = 1: peaks from the row kernel, noise = the AP's energy
])
def test_allif_search_matches_oracle(vb, oracle, shape):
    """f2: one delay across all IFs (Eq. 1) vs oracle.allif_search on the same inputs."""
    nbl, nif, nap, nchan, widths, strides, nfa, dm = shape
    g = torch.Generator().manual_seed(nap + nchan)
    vis = torch.view_as_complex(torch.randn((nbl, nif, nap, nchan, 2), generator=g) * 0.7071)
    m = torch.arange(nif * nchan, dtype=torch.float64).reshape(nif, 1, nchan)
    vis[0, :, nap // 3: nap // 3 + 12] += torch.polar(torch.full((nif, 1, nchan), 0.4, dtype=torch.float64),
                                                      2 * np.pi * 0.0137 * m).to(torch.complex64)   # one delay, all IFs
    vis[-1, :, nap // 2: nap // 2 + 20] = 0                                                           # flagged span
    sh = None
    src = vis.numpy()
    if dm:
        f = 1400.0 + 16.0 * np.arange(nif)[:, None] + (16.0 / nchan) * np.arange(nchan)[None, :]
        sh = vb.dm_shifts(dm, f, f.max(), 1e-3)
        src = oracle.dedisperse(src, sh)
    thresh = 4.0
    cands, n, peaks = vb.allif_search(vis.cuda(), widths, strides, nfa, thresh, want_peaks=True, shifts=sh)
    ora = oracle.allif_search(src, widths, strides, nfa)
    nw = [workloads.gen.nwin(nap, w, s) for w, s in zip(widths, strides)]
    pk = peaks[dense_index(nbl, 1, nw)]
    assert np.all(pk["rate_idx"] == 0)
    band = oracle.allif_band(src)

    check_peaks(pk, ora, nfa, allif_plane_power(oracle, band, nw, widths, strides, nfa))
    exp = np.nonzero(ora["snr"] > thresh)[0]
    marg = np.abs(ora["snr"] - thresh) <= 1e-4 * thresh
    assert abs(n - len(exp)) <= int(marg.sum()) and n >= 1
    assert np.all(cands["ifq"] == -1) and np.all(cands["rate_idx"] == 0)
    key = [(int(c["bl"]), int(c["wid"]), int(c["win"])) for c in cands]
    assert key == sorted(key)
    hit = [c for c in cands if c["bl"] == 0 and nap // 3 - 16 <= c["t0"] <= nap // 3 + 12]
    res = max(1, nfa // (nif * nchan))            # one unpadded resolution element of the delay axis
    assert hit and all(abs(int(c["delay_idx"]) - round(0.0137 * nfa)) <= res for c in hit if c["snr"] > 8)


@pytest.mark.parametrize("chunk_mb", ["1", "8"])   # 8 MB: several pairs per plan chunk, the host path takes a quarter at a time
@pytest.mark.parametrize("allif", [False, True])
def test_host_slab_search_is_identical(vb, allif, chunk_mb):
    """volks_search_host (slab in pinned host memory, chunked copies overlapped with the kernels) must
    give bit-identical candidates and peaks to the device-slab call; small chunks force several
    copy/compute rounds through both stage halves, twice in a row (stage reuse across calls)."""
    opts = dict(chunk_mb=int(chunk_mb))
    vis, c, _ = workloads.generate(2, nbl=3, nif=3, nap=600, npulses=3)
    nbl, nif, nap, nchan = vis.shape
    if allif:
        plan = vb.Plan(nbl, nif, nap, nchan, c["widths"], c["strides"], None, 1024, 4.0, allif=True, options=opts)
    else:
        plan = vb.Plan(nbl, nif, nap, nchan, c["widths"], c["strides"], c["nts"], c["nf"], 4.0, options=opts)
    dev = torch.device("cuda")
    ws = torch.empty(plan.workspace_bytes, dtype=torch.uint8, device=dev)
    cap = 1 << 16
    mk = lambda: (torch.empty(cap * vb.CAND_DTYPE.itemsize, dtype=torch.uint8, device=dev),
                  torch.zeros(1, dtype=torch.int32, device=dev),
                  torch.empty(plan.nwin_total * vb.PEAK_DTYPE.itemsize, dtype=torch.uint8, device=dev))
    c0, n0, p0 = mk()
    plan.fringe_search(vis.cuda(), ws, c0, n0, p0)
    torch.cuda.synchronize()
    ref = (int(n0.item()), c0.cpu().numpy()[: int(n0.item()) * 36].tobytes(), p0.cpu().numpy().tobytes())
    assert ref[0] >= 1
    h = vis.pin_memory()
    stage = torch.empty(2 * plan.stage_bytes, dtype=torch.uint8, device=dev)
    assert plan.stage_bytes < h.numel() * 8 / 2          # several chunks
    for _ in range(2):
        c1, n1, p1 = mk()
        plan.search_host(h, stage, ws, c1, n1, p1)
        torch.cuda.synchronize()
        assert int(n1.item()) == ref[0]
        assert c1.cpu().numpy()[: ref[0] * 36].tobytes() == ref[1] and p1.cpu().numpy().tobytes() == ref[2]
    plan.close()


def test_search_is_cuda_graph_capturable(vb):
    """The search is stream-asynchronous with no host synchronisation or allocation inside, so a
    launch-bound small search (config 1) can be captured once in a CUDA graph and replayed."""
    vis, c, _ = workloads.generate(1)
    nbl, nif, nap, nchan = vis.shape
    plan = vb.Plan(nbl, nif, nap, nchan, c["widths"], c["strides"], c["nts"], c["nf"], c["snr_thresh"])
    dev = torch.device("cuda")
    d_vis = vis.cuda()
    ws = torch.empty(plan.workspace_bytes, dtype=torch.uint8, device=dev)
    cap = 1 << 14
    cands = torch.zeros(cap * vb.CAND_DTYPE.itemsize, dtype=torch.uint8, device=dev)
    ncand = torch.zeros(1, dtype=torch.int32, device=dev)
    plan.fringe_search(d_vis, ws, cands, ncand)
    torch.cuda.synchronize()
    ref = (int(ncand.item()), cands.cpu().numpy().tobytes())
    graph = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        with torch.cuda.graph(graph, stream=side):
            plan.fringe_search(d_vis, ws, cands, ncand, stream=side)
    for _ in range(3):
        cands.zero_(); ncand.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert (int(ncand.item()), cands.cpu().numpy().tobytes()) == ref
    plan.close()


def test_calibration_fused_into_slab_load(vb, oracle):
    """Eq. 1's calibration terms applied while the slab is read == oracle.calibrate followed by the
    plain search; per-IF 2-D search (with and without dedispersion) and the all-IF search, where the
    calibration is what makes the IFs coherent."""
    vis, c, _ = workloads.generate(2, nbl=2, nif=4, nap=400, npulses=2)
    nbl, nif, nap, nchan = vis.shape
    rng = np.random.default_rng(8)
    d0, p0 = rng.uniform(-40e-9, 40e-9, (nbl, nif)), rng.uniform(-np.pi, np.pi, (nbl, nif))
    chan_hz = 16e6 / nchan
    cal = vb.cal_phasors(d0, p0, nchan, chan_hz)
    # corrupt the data with the inverse phasors, so that calibration restores the injected pulses
    raw = (vis.numpy().astype(np.complex128) * np.conj(cal.astype(np.complex128))[:, :, None, :]).astype(np.complex64)
    d_raw, d_cal = torch.from_numpy(raw).cuda(), torch.from_numpy(cal).cuda()
    nw = [workloads.gen.nwin(nap, w, s) for w, s in zip(c["widths"], c["strides"])]
    f = 1400.0 + 16.0 * np.arange(nif)[:, None] + (16.0 / nchan) * np.arange(nchan)[None, :]
    sh = vb.dm_shifts(200.0, f, f.max(), c["t_ap"])
    for shifts in (None, sh):
        plan = vb.Plan(nbl, nif, nap, nchan, c["widths"], c["strides"], c["nts"], c["nf"], c["snr_thresh"])
        plan.set_cal(d_cal)
        cands, n, peaks = vb.fringe_search(d_raw, want_peaks=True, plan=plan, shifts=shifts)
        src = oracle.calibrate(raw, cal)
        if shifts is not None:
            src = oracle.dedisperse(src, shifts)
        ora, _ = oracle.search(src, c["widths"], c["strides"], c["nts"], c["nf"], mode="cached")
        check_peaks(peaks[dense_index(nbl, nif, nw)], ora, c["nf"], make_plane_power(oracle, src, c))
        plan.set_cal(None)
        _, _, p_off = vb.fringe_search(d_raw, want_peaks=True, plan=plan, shifts=shifts)
        assert not np.array_equal(p_off["delay_idx"], peaks["delay_idx"])      # switching it off changes the result
        plan.close()
    # all-IF: coherent only after calibration
    nfa = 1024
    plan = vb.Plan(nbl, nif, nap, nchan, c["widths"], c["strides"], None, nfa, 5.0, allif=True)
    plan.set_cal(d_cal)
    cands, n, peaks = vb.fringe_search(d_raw, want_peaks=True, plan=plan)
    ora = oracle.allif_search(oracle.calibrate(raw, cal), c["widths"], c["strides"], nfa)
    pk = peaks[dense_index(nbl, 1, nw)]
    perr = np.abs(pk["power"] - ora["p1"]) / ora["p1"]
    gap = (ora["p1"] - ora["p2"]) / ora["p1"]
    ok = (pk["delay_idx"] == ora["idx1"]) | ((gap < 1e-5) & (pk["delay_idx"] == ora["idx2"]))
    assert perr.max() <= 1e-4 and ok.all()
    plan.set_cal(None)
    _, n_off, _ = vb.fringe_search(d_raw, want_peaks=True, plan=plan)
    assert n > n_off                                  # uncalibrated IFs do not add up
    plan.close()


def test_dynamic_range_after_strong_samples(vb, oracle):
    """A 3000x burst followed by ordinary noise, then a nearly empty stretch (one surviving sample per
    window): the running sums would carry the burst's rounding residue; the exact re-evaluation
    (k_fixup / k_allif's direct re-sum) keeps every window within the 1e-4 bound."""
    vis, c, _ = workloads.generate(2, nbl=1, nif=2, nap=700, npulses=2)
    vis[0, :, 100:104] *= 3000.0
    vis[0, 0, 300:500] = 0
    vis[0, 0, 400, 7] = 0.3 + 0.1j
    # a threshold-level 64-AP pulse whose windows start right after the burst has left them (window 104 on): the folded
    # sliding sum (candidates-only mode) must not test them with sums that still carry the burst's rounding residue
    nchan = vis.shape[3]
    k = torch.arange(nchan, dtype=torch.float64)
    ph = torch.polar(torch.full((nchan,), 7.5 / np.sqrt(64 * nchan), dtype=torch.float64), 2 * np.pi * 5.0 * k / nchan)
    vis[0, 1, 106:170] += ph.to(torch.complex64)
    stats, ncand, cands, ora = run_both(vb, oracle, vis, c)
    w64 = cands[(cands["wid"] == len(c["widths"]) - 1) & (cands["ifq"] == 1)]
    assert np.any((w64["t0"] >= 104) & (w64["t0"] <= 112))       # the pulse is found in the windows just behind the burst
    cands, n, peaks = vb.allif_search(vis.cuda(), c["widths"], c["strides"], 512, 4.0, want_peaks=True)
    ora = oracle.allif_search(vis.numpy(), c["widths"], c["strides"], 512)
    nw = [workloads.gen.nwin(vis.shape[2], w, s) for w, s in zip(c["widths"], c["strides"])]
    pk = peaks[dense_index(1, 1, nw)]
    ok = ora["p1"] > 0
    assert (np.abs(pk["power"][ok] - ora["p1"][ok]) / ora["p1"][ok]).max() <= 1e-4
    assert np.all(pk["power"][~ok] == 0)


@pytest.mark.parametrize("seed", list(range(10)))
def test_random_shapes(vb, oracle, seed):
    """Seeded random small problems across every kernel-selection branch (row kernels by nf, sliding /
    column-FFT / generic rate kernels by width, stride and padding), every window compared."""
    rng = np.random.default_rng(1000 + seed)
    nf = int(2 ** rng.integers(3, 10))                      # 8 .. 512
    nchan = int(rng.integers(max(1, nf // 4), nf + 1))
    nbl, nif = int(rng.integers(1, 3)), int(rng.integers(1, 3))
    nwid = int(rng.integers(1, 5))
    widths, strides, nts = [], [], []
    for _ in range(nwid):
        w = int(rng.choice([1, 2, 3, 4, 6, 8, 16, 20, 32]))
        pad = int(rng.choice([1, 2, 2, 2, 4]))
        nt = 1
        while nt < w * pad:
            nt *= 2
        widths.append(w); nts.append(nt)
        strides.append(1 if rng.random() < 0.6 else int(rng.integers(1, w + 3)))
    nap = int(rng.integers(max(widths), max(widths) + 400))
    g = torch.Generator().manual_seed(seed)
    vis = torch.view_as_complex(torch.randn((nbl, nif, nap, nchan, 2), generator=g) * 0.7071)
    t0 = int(rng.integers(0, max(1, nap - 8)))
    vis[0, 0, t0:t0 + 8] += 1.0 + 1.0j
    c = dict(widths=widths, strides=strides, nts=nts, nf=nf, snr_thresh=3.0)
    run_both(vb, oracle, vis, c, mode="fft")


@pytest.mark.parametrize("seed", list(range(8)))
def test_random_gather_shapes(vb, oracle, seed):
    """Seeded random problems through the gather modes of every row kernel (k_row2: nf 64..256, k_row3:
    512..2048, k_rowbig: 4096 / 8192, generic: the rest): random per-channel shifts (negative and past the
    end included), a ragged band (nchan < nf), optional calibration phasors; per-IF search vs
    oracle.calibrate + oracle.dedisperse + oracle.search, every window compared."""
    rng = np.random.default_rng(7000 + seed)
    nf = int([64, 128, 256, 512, 1024, 2048, 4096, 8192][seed])
    nchan = int(rng.integers(nf // 8 + 1, nf + 1))
    nbl, nif = int(rng.integers(1, 3)), int(rng.integers(1, 4))
    widths, strides, nts = [], [], []
    for w in rng.choice([1, 2, 4, 8, 16], size=2, replace=False):
        w = int(w)
        widths.append(w); strides.append(1 if rng.random() < 0.5 else int(rng.integers(1, w + 2)))
        nts.append(int(workloads.gen.next_pow2(w * int(rng.choice([1, 2])))))
    nap = int(rng.integers(40, 90)) if nf >= 1024 else int(rng.integers(60, 300))
    g = torch.Generator().manual_seed(900 + seed)
    vis = torch.view_as_complex(torch.randn((nbl, nif, nap, nchan, 2), generator=g) * 0.7071)
    vis[0, 0, nap // 2: nap // 2 + 6] += 1.0 + 0.5j
    sh = rng.integers(-3, 13, size=(nif, nchan)).astype(np.int32)
    sh[0, 0] = nap + 2
    raw = vis.numpy()
    cal = None
    if seed % 2:
        cal = vb.cal_phasors(rng.uniform(-30e-9, 30e-9, (nbl, nif)), rng.uniform(-np.pi, np.pi, (nbl, nif)), nchan, 16e6 / nchan)
    plan = vb.Plan(nbl, nif, nap, nchan, widths, strides, nts, nf, 3.0)
    if cal is not None:
        plan.set_cal(torch.from_numpy(cal).cuda())
    cands, n, peaks = vb.fringe_search(vis.cuda(), want_peaks=True, plan=plan, shifts=sh)
    plan.close()
    src = oracle.dedisperse(oracle.calibrate(raw, cal) if cal is not None else raw, sh)
    c = dict(widths=widths, strides=strides, nts=nts, nf=nf)
    ora, _ = oracle.search(src, widths, strides, nts, nf, mode="cached")
    nw = [workloads.gen.nwin(nap, w, s) for w, s in zip(widths, strides)]
    check_peaks(peaks[dense_index(nbl, nif, nw)], ora, nf, make_plane_power(oracle, src, c))
    oc, keep = oracle.candidates(ora, nbl, nif, nap, widths, strides, nf, 3.0)
    check_candidates(cands, oc, ora, keep, 3.0, nf)


@pytest.mark.parametrize("seed", list(range(6)))
def test_random_allif_shapes(vb, oracle, seed):
    """Seeded random all-IF searches (f2): nfa 256..16384 (k_row2, k_row3, generic, k_rowbig, interleaved
    sub-rows), random per-channel shifts, a band that does not fill nfa, optional calibration; every window
    against oracle.allif_search."""
    rng = np.random.default_rng(8100 + seed)
    nfa = int([256, 1024, 2048, 4096, 8192, 16384][seed])
    nif = int(rng.integers(1, 5))
    nchan = int(rng.integers(max(1, nfa // (8 * nif)), min(nfa, 8192) // nif + 1))     # the band fits one 8192-point row
    nbl = int(rng.integers(1, 3))
    widths = [int(w) for w in rng.choice([1, 2, 3, 4, 8, 16, 24], size=2, replace=False)]
    strides = [1 if rng.random() < 0.5 else int(rng.integers(1, w + 2)) for w in widths]
    nap = int(rng.integers(40, 80)) if nfa >= 4096 else int(rng.integers(80, 400))
    g = torch.Generator().manual_seed(300 + seed)
    vis = torch.view_as_complex(torch.randn((nbl, nif, nap, nchan, 2), generator=g) * 0.7071)
    sh = rng.integers(-2, 9, size=(nif, nchan)).astype(np.int32)
    raw = vis.numpy()
    cal = None
    if seed % 2 == 0:
        cal = vb.cal_phasors(rng.uniform(-30e-9, 30e-9, (nbl, nif)), rng.uniform(-np.pi, np.pi, (nbl, nif)), nchan, 16e6 / nchan)
    plan = vb.Plan(nbl, nif, nap, nchan, widths, strides, None, nfa, 3.0, allif=True)
    if cal is not None:
        plan.set_cal(torch.from_numpy(cal).cuda())
    cands, n, peaks = vb.fringe_search(vis.cuda(), want_peaks=True, plan=plan, shifts=sh)
    plan.close()
    src = oracle.dedisperse(oracle.calibrate(raw, cal) if cal is not None else raw, sh)
    ora = oracle.allif_search(src, widths, strides, nfa)
    nw = [workloads.gen.nwin(nap, w, s) for w, s in zip(widths, strides)]
    band = oracle.allif_band(src)

    check_peaks(peaks[dense_index(nbl, 1, nw)], ora, nfa, allif_plane_power(oracle, band, nw, widths, strides, nfa))
    marg = np.abs(ora["snr"] - 3.0) <= 1e-4 * 3.0
    assert abs(n - np.count_nonzero(ora["snr"] > 3.0)) <= int(marg.sum())


def test_cufft_cross_check(vb, oracle):
    """Pin P12 on the GPU side (north_star: "cuFFT only as a cross-check"; the transform is PAPER.md:83): a
    handful of zero-padded planes formed by torch.fft.fft2 (cuFFT C2C, complex64) as a third opinion beside
    the library's dense peaks and the oracle.  Test-only: nothing under paper_2108_05602_b200/ touches cuFFT."""
    for cfg, over in [(1, {}), (2, dict(nbl=1, nif=2, nap=300, npulses=2)), (4, dict(nbl=1, nif=1, nap=300, npulses=1))]:
        vis, c, _ = workloads.generate(cfg, **over)
        nbl, nif, nap, nchan = vis.shape
        dv = vis.cuda()
        _, _, peaks = vb.fringe_search(dv, c["widths"], c["strides"], c["nts"], c["nf"], c["snr_thresh"], want_peaks=True)
        nw = [workloads.gen.nwin(nap, w, s) for w, s in zip(c["widths"], c["strides"])]
        rng = np.random.default_rng(40 + cfg)
        for _ in range(6):
            q = int(rng.integers(0, len(nw)))
            pair, j = int(rng.integers(0, nbl * nif)), int(rng.integers(0, nw[q]))
            w, s, nt, nf = c["widths"][q], c["strides"][q], c["nts"][q], c["nf"]
            win = dv[pair // nif, pair % nif, j * s: j * s + w]
            P = torch.fft.fft2(win, s=(nt, nf)).abs().square().double().cpu().numpy().reshape(-1)   # cuFFT
            g = peaks[nbl * nif * sum(nw[:q]) + pair * nw[q] + j]
            o, _ = oracle.window(win.cpu().numpy(), nt, nf, mode="fft")
            gi = int(g["rate_idx"]) * nf + int(g["delay_idx"])
            # cuFFT is itself fp32: the library's bin must carry cuFFT's maximum to within fp32 rounding, and
            # where the oracle's argmax is unambiguous all three name the same bin
            assert P[gi] >= P.max() * (1 - 1e-5)
            assert abs(P.max() - o["p1"]) <= 1e-4 * o["p1"] and abs(float(g["power"]) - P.max()) <= 1e-4 * P.max()
            if (o["p1"] - o["p2"]) / o["p1"] > 1e-4:
                assert int(np.argmax(P)) == o["idx1"] == gi
            assert abs(P.sum() / (nt * nf) - o["s1"] / (nt * nf)) <= 1e-4 * o["s1"] / (nt * nf)
            noise = P.sum() / (nt * nf)
            assert abs(float(g["snr"]) - np.sqrt(P.max() / noise)) <= 1e-4 * o["snr"]


def test_sliding_sum_adversarial(vb, oracle):
    """The worst case the sliding kernels can meet without the fix-up stepping in (the 1e-4 bound of the
    sliding sum is statistical): one delay column driven by a coherent burst whose power stays just UNDER the fix-up
    ratio (1000x) of the windows that follow, and after it the same weak noiseless tone in every AP, so that every
    window of the rest of the segment has the same small peak and any residue of the burst shows directly.  Every
    window of every sliding width must stay within 1e-4 of the oracle, in both index modes."""
    nchan, nap, nf = 64, 900, 128
    widths, strides, nts = [2, 4, 8, 16, 32, 64], [1] * 6, [4, 8, 16, 32, 64, 128]
    k = torch.arange(nchan, dtype=torch.float64)
    tone = torch.polar(torch.full((nchan,), 0.01, dtype=torch.float64), 2 * np.pi * 9.0 * k / nf)   # on delay bin 9
    vis = tone.to(torch.complex64).repeat(nap, 1).reshape(1, 1, nap, nchan).clone()
    # the peak power of a tone window is (a w nchan)^2; with 4 burst APs at 480 a inside, a w = 64 window peaks at
    # ((60 + 4 * 480) a nchan)^2 = 957 x the later windows: just under the fix-up ratio for the width with the longest
    # memory, far above it for the narrow ones (their windows after the burst are re-evaluated, which is tested too)
    vis[0, 0, 130:134] = (tone * 480.0).to(torch.complex64)
    g = torch.Generator().manual_seed(5)
    vis += (torch.view_as_complex(torch.randn((1, 1, nap, nchan, 2), generator=g)) * 1e-6)   # breaks exact ties only
    c = dict(widths=widths, strides=strides, nts=nts, nf=nf, snr_thresh=6.0)
    (nties, perr, serr), ncand, cands, ora = run_both(vb, oracle, vis, c, mode="fft")
    assert perr <= 1e-4 and serr <= 1e-4 and ncand > 1000          # (nearly every window is a candidate: a pure tone)
    run_both(vb, oracle, vis, c, mode="fft", options=dict(slide_seg=1024))   # the longest segment the option allows here


@pytest.mark.parametrize("prune_seg", [16, 64, 256])
def test_pruning_keeps_every_candidate(vb, oracle, prune_seg):
    """Candidates-only mode (volks_options defaults) against the full-index mode and the oracle on data where the
    amplitude-sum bound prunes most segments: weak and strong pulses at segment seams, a pulse in the last windows, an
    RFI burst, a flagged (zero) span.  Within one plan the two index modes must agree bit for bit (run_both asserts it);
    across segment lengths / pruning off / full_index the arithmetic of the sliding sum differs in the last bits, so
    there the lists must hold the same windows and bins with powers equal to 1e-5."""
    vis, c, _ = workloads.generate(3, nbl=2, nif=2, nap=2100, npulses=0)
    nbl, nif, nap, nchan = vis.shape
    k = torch.arange(nchan, dtype=torch.float64)
    def pulse(bl, ifq, t0, w, a, tau):
        ph = torch.polar(torch.full((nchan,), a, dtype=torch.float64), 2 * np.pi * tau * k / nchan)
        vis[bl, ifq, t0:t0 + w] += ph.to(torch.complex64)
    pulse(0, 0, 60, 8, 1.2, 3.0)          # inside one segment of 64
    pulse(0, 1, 63, 2, 2.5, -5.0)         # straddles a seam at 64
    pulse(1, 0, 255, 16, 0.9, 1.0)        # straddles a seam at 256
    pulse(1, 1, nap - 5, 5, 3.0, 7.0)     # the last windows of the slab
    pulse(0, 0, 1000, 1, 6.0, 0.0)        # a single-AP burst
    pulse(1, 0, 1500, 4, 0.45, 2.0)       # weak: near the threshold for some widths
    vis[1, 1, 700:900] = 0                # flagged span
    ref = None
    for opts in (dict(prune_seg=prune_seg), dict(no_prune=1), dict(full_index=1)):
        stats, ncand, cands, ora = run_both(vb, oracle, vis, c, options=opts)
        assert ncand >= 20
        if ref is not None:
            for f in ("bl", "ifq", "wid", "win", "t0", "rate_idx", "delay_idx"):
                assert np.array_equal(cands[f], ref[f]), f
            assert np.all(np.abs(cands["power"] - ref["power"]) <= 1e-5 * ref["power"])
        ref = cands
    plan = vb.Plan(nbl, nif, nap, nchan, c["widths"], c["strides"], c["nts"], c["nf"], c["snr_thresh"])
    ws = torch.empty(plan.workspace_bytes, dtype=torch.uint8, device="cuda")
    cbuf = torch.empty(1 << 16, dtype=torch.uint8, device="cuda")
    nc = torch.zeros(1, dtype=torch.int32, device="cuda")
    plan.fringe_search(vis.cuda(), ws, cbuf, nc)
    with pytest.raises(vb.VolksError):                 # the candidates-only search left no exact index for every window
        plan.zscore_select(ws, 3.0, cbuf, nc)
    plan.close()


@pytest.mark.gpu
def test_folded_column_bound_every_residue(vb, oracle):
    """The column bits of the w = 32 width come from k_pairfold's folded bound, four sliding sums of
    |y[t] + (-i)^rho y[t + 16]| (rho = rate bin mod 4).  Pulses barely above the threshold whose rate falls into each of
    the four residues - a wrong sign in one of the four combinations would lose exactly one of them - placed at the
    kernel's tile seam (window 256), at the first and the last windows, plus two tones (the dense rule) on one pair.  Candidates-only and full-index lists are checked against the oracle by run_both."""
    vis, c, _ = workloads.generate(2, nbl=2, nif=2, nap=900, npulses=0)
    nbl, nif, nap, nchan = vis.shape
    k = torch.arange(nchan, dtype=torch.float64)
    t = torch.arange(nap, dtype=torch.float64)
    def pulse(bl, ifq, t0, w, a, tau, r, nt=64):
        # delay tau (channels -> columns) and rate bin r of an Nt-point transform: + signs (workloads/gen.py)
        ph = 2 * np.pi * tau * k[None, :] / nchan + 2 * np.pi * r * t[t0:t0 + w, None] / nt
        vis[bl, ifq, t0:t0 + w] += torch.polar(torch.full(ph.shape, a, dtype=torch.float64), ph).to(torch.complex64)
    a32 = 7.5 / np.sqrt(32 * nchan)             # amplitude of a 32-AP pulse at S/N 7.5 in the w = 32 plane (noise power 1 per sample)
    # (baseline 0 carries configs[2]'s own interference - a dense pair; the pulses go on baseline 1)
    pulse(1, 0, 100, 32, a32, 3.0, 0)
    pulse(1, 0, 240, 32, a32, -7.0, 1)          # straddles window 256
    pulse(1, 1, 400, 32, a32, 11.0, 2)
    pulse(1, 1, 520, 32, a32, 0.5, 3)
    pulse(1, 0, 0, 32, a32, 20.0, 5)            # the first windows, residue 1
    pulse(1, 0, nap - 32, 32, a32, -15.0, 62)   # the last window, residue 2
    pulse(1, 1, 640, 32, a32, 2.0, 31)          # residue 3
    # two tones (one alone never reaches S/N 6 at w = 32: its own energy raises the noise estimate to S/N -> sqrt(32));
    # where they add coherently - 40 % of the delay columns - every window's bit is set: the dense rule
    for ch in (7, 50):
        vis[0, 1, :, ch] += (30.0 * torch.exp(2j * np.pi * 0.003 * t)).to(torch.complex64)
    cc = dict(c, widths=[32, 64], strides=[1, 1], nts=[64, 128])
    # (prune_seg = 128 switches the column-level rule off: w = 32 then runs on the folded sliding sum with M = 4 residues)
    for opts in (None, dict(full_index=1), dict(prune_seg=128)):
        stats, ncand, cands, ora = run_both(vb, oracle, vis, cc, options=opts)
        got = {(int(x["bl"]), int(x["ifq"]), int(x["wid"])) for x in cands}
        assert {(0, 1, 0), (1, 0, 0), (1, 1, 0)} <= got                 # the tones' pair and both pulse pairs have w = 32 candidates
        w32 = cands[(cands["wid"] == 0) & (cands["bl"] == 1)]
        assert {int(r) % 4 for r in w32["rate_idx"]} == {0, 1, 2, 3}


@pytest.mark.parametrize("cfg,over,ranges", [
    (2, dict(nbl=1, nif=2, nap=500, npulses=3), [(250, 5), (3, 40), (100, 100), (64, 127), (1, 255)]),   # nf 256: sliding kernels, all widths
    (3, dict(nbl=2, nif=1, nap=700, npulses=3), [(120, 7), (0, 63), (9, 9)]),                            # nf 128, incl. w = 1 (row kernel peaks)
    (4, dict(nbl=1, nif=1, nap=400, npulses=1), [(2040, 7), (100, 1500)]),                               # nf 2048: k_row3 + k_colfft2
    (1, dict(nap=500), [(120, 8), (5, 70)]),                                                             # stride > 1: k_colfft / k_col
])
def test_delay_range_restriction(vb, oracle, cfg, over, ranges):
    """volks_options.delay_lo / delay_hi ("the delay search range ... is configured for projected baselines
    shorter than 3000 km"): the peak is searched in the allowed delay bins only (wrapping ranges around zero delay, a
    single bin, whole 64-column groups in and out), the noise statistic is the whole plane's; every window and the
    candidate lists of both index modes against the oracle's restricted scan."""
    vis, c, _ = workloads.generate(cfg, **over)
    full = run_both(vb, oracle, vis, c)
    for rg in ranges:
        stats, ncand, cands, ora = run_both(vb, oracle, vis, c, delay_range=rg)
        lo, hi = rg
        d = cands["delay_idx"]
        assert np.all((d >= lo) & (d <= hi) if lo <= hi else (d >= lo) | (d <= hi))
        run_both(vb, oracle, vis, c, thresh=3.0, delay_range=rg)
    # the whole axis given explicitly is the unrestricted search
    same = run_both(vb, oracle, vis, c, delay_range=(0, c["nf"] - 1))
    assert same[2].tobytes() == full[2].tobytes()


def test_delay_range_allif(vb, oracle):
    """The same restriction on f2 (the paper's own all-IF search): bins of the nfa axis, incl. nfa > 8192 (interleaved
    sub-rows); the noise is still the mean over the whole delay axis."""
    for (nbl, nif, nap, nchan, nfa, rg) in [(2, 4, 120, 64, 512, (500, 11)), (1, 8, 40, 1024, 32768, (32000, 700)), (1, 2, 90, 32, 128, (17, 17))]:
        g = torch.Generator().manual_seed(nfa)
        vis = torch.view_as_complex(torch.randn((nbl, nif, nap, nchan, 2), generator=g) * 0.7071)
        widths, strides = [1, 4, 8], [1, 1, 3]
        cands, n, peaks = vb.allif_search(vis.cuda(), widths, strides, nfa, 2.0, want_peaks=True,
                                          options=dict(delay_lo=rg[0], delay_hi=rg[1]))
        ora = oracle.allif_search(vis.numpy(), widths, strides, nfa, delay_range=rg)
        nw = [workloads.gen.nwin(nap, w, s) for w, s in zip(widths, strides)]
        pk = peaks[dense_index(nbl, 1, nw)]
        lo, hi = rg
        d = pk["delay_idx"]
        assert np.all((d >= lo) | (d <= hi) if lo > hi else (d >= lo) & (d <= hi))
        band = oracle.allif_band(vis.numpy())
        check_peaks(pk, ora, nfa, allif_plane_power(oracle, band, nw, widths, strides, nfa))
        assert n == np.count_nonzero(ora["snr"] > 2.0) or np.any(np.abs(ora["snr"] - 2.0) <= 2e-4)
