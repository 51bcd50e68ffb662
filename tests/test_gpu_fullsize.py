"""Full-size runs of BASELINE.json configs 2-4 in the launch configuration bench.py times, checked
against the oracle on sampled windows (the oracle computes any one window from its [w x nchan]
slab): every window overlapping an injected pulse start, every GPU candidate (capped), and a
seeded random sample; plus properties that hold at any size."""
import numpy as np
import pytest
import torch

import workloads
from _parity import RTOL, TIE

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def vb():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2108_05602_b200 as v
    v.lib()
    return v


@pytest.mark.parametrize("cfg,nrandom", [(2, 300), (3, 400), (4, 24)])
def test_fullsize_sampled(vb, oracle, cfg, nrandom):
    vis, c, truth = workloads.generate(cfg, device="cuda")
    nbl, nif, nap, nchan = vis.shape
    plan = vb.Plan(nbl, nif, nap, nchan, c["widths"], c["strides"], c["nts"], c["nf"], c["snr_thresh"])
    cands, n, peaks = vb.fringe_search(vis, None, None, None, None, None, want_peaks=True, cand_capacity=1 << 22, plan=plan)
    nw = plan.nwin_per_width
    assert plan.nwin_total == workloads.gen.nwin_total(c) == len(peaks)
    # properties at full size
    assert np.all(peaks["power"] >= 0) and np.all(np.isfinite(peaks["snr"]))
    for q, ntq in enumerate(c["nts"]):
        lo = nbl * nif * sum(nw[:q])
        seg = peaks[lo: lo + nbl * nif * nw[q]]
        assert seg["rate_idx"].min() >= 0 and seg["rate_idx"].max() < ntq
        assert seg["delay_idx"].min() >= 0 and seg["delay_idx"].max() < c["nf"]
        assert np.all(seg["snr"] <= np.sqrt(c["widths"][q] * nchan) * (1 + 1e-4))     # Cauchy-Schwarz bound
    assert n == np.count_nonzero(peaks["snr"] > c["snr_thresh"])
    keys = list(zip(cands["bl"], cands["ifq"], cands["wid"], cands["win"]))
    assert keys == sorted(keys)
    # sample: (pair, q, j)
    rng = np.random.default_rng(100 + cfg)
    sample = set()
    for _ in range(nrandom):
        q = int(rng.integers(0, len(nw)))
        sample.add((int(rng.integers(0, nbl * nif)), q, int(rng.integers(0, nw[q]))))
    for p in truth["pulses"][:10]:
        for q, (w, s) in enumerate(zip(c["widths"], c["strides"])):
            j = min(max(p["t0"] // s, 0), nw[q] - 1)
            sample.add((int(rng.integers(0, nbl * nif)), q, int(j)))
    for cd in cands[:: max(1, len(cands) // 60)][:60]:
        sample.add((int(cd["bl"]) * nif + int(cd["ifq"]), int(cd["wid"]), int(cd["win"])))
    nties = 0
    for (pair, q, j) in sorted(sample):
        w, s, ntq = c["widths"][q], c["strides"][q], c["nts"][q]
        t0 = j * s
        slab = vis[pair // nif, pair % nif, t0:t0 + w].cpu().numpy()
        o, _ = oracle.window(slab, ntq, c["nf"], mode="fft")
        g = peaks[nbl * nif * sum(nw[:q]) + pair * nw[q] + j]
        gi = int(g["rate_idx"]) * c["nf"] + int(g["delay_idx"])
        tie = (o["p1"] - o["p2"]) / o["p1"] < TIE
        assert gi == o["idx1"] or (tie and gi == o["idx2"]), (pair, q, j, gi, o)
        nties += gi != o["idx1"]
        assert abs(float(g["power"]) - o["p1"]) <= RTOL * o["p1"]
        assert abs(float(g["snr"]) - o["snr"]) <= RTOL * o["snr"]
        assert (o["snr"] > c["snr_thresh"]) == (float(g["snr"]) > c["snr_thresh"]) or abs(o["snr"] - c["snr_thresh"]) < RTOL * c["snr_thresh"]
    plan.close()


def test_fullsize_allif_sampled(vb, oracle):
    """f2 at the paper's size in the launch configuration `bench.py --config 5 --allif --dm 26.8` times
    (21 baselines x 3906 APs x 8 IF x 1024 points, nfa 32768 = 4 interleaved 8192-point transforms, dedispersed):
    sampled windows against oracle.dedisperse + oracle.allif_search on the window's own APs."""
    cfg = 5
    vis, c, _ = workloads.generate(cfg, device="cuda")
    nbl, nif, nap, nchan = vis.shape
    nfa = workloads.gen.next_pow2(4 * nif * nchan)
    assert nfa == 32768
    f = 1400.0 + 16.0 * np.arange(nif)[:, None] + (16.0 / nchan) * np.arange(nchan)[None, :]
    sh = vb.dm_shifts(26.8, f, f.max(), c["t_ap"])
    plan = vb.Plan(nbl, nif, nap, nchan, c["widths"], c["strides"], None, nfa, c["snr_thresh"], allif=True)
    cands, n, peaks = vb.fringe_search(vis, None, None, None, None, None, want_peaks=True, cand_capacity=1 << 20,
                                       plan=plan, shifts=sh)
    nw = plan.nwin_per_width
    per = sum(nw)
    assert len(peaks) == nbl * per == plan.nwin_total
    assert np.all(peaks["rate_idx"] == 0) and peaks["delay_idx"].min() >= 0 and peaks["delay_idx"].max() < nfa
    assert np.all(np.isfinite(peaks["snr"])) and np.all(peaks["power"] >= 0)
    assert n == np.count_nonzero(peaks["snr"] > c["snr_thresh"])
    keys = list(zip(cands["bl"], cands["wid"], cands["win"]))
    assert keys == sorted(keys) and np.all(cands["ifq"] == -1)
    rng = np.random.default_rng(505)
    for bl in (0, int(rng.integers(1, nbl - 1)), nbl - 1):
        src = oracle.dedisperse(vis[bl:bl + 1].cpu().numpy(), sh)
        sample = {(q, int(rng.integers(0, nw[q]))) for q in range(len(nw)) for _ in range(4)}
        sample |= {(q, 0) for q in range(len(nw))} | {(q, nw[q] - 1) for q in range(len(nw))}   # zero-filled head / tail
        sample |= {(int(cd["wid"]), int(cd["win"])) for cd in cands[cands["bl"] == bl][:6]}
        for (q, j) in sorted(sample):
            w, s = c["widths"][q], c["strides"][q]
            o = oracle.allif_search(src[:, :, j * s: j * s + w], [w], [1], nfa)[0]
            g = peaks[nbl * sum(nw[:q]) + bl * nw[q] + j]      # dense peaks are laid out [width][baseline][window]
            gi = int(g["delay_idx"])
            tie = o["p1"] > 0 and (o["p1"] - o["p2"]) / o["p1"] < TIE
            assert gi == o["idx1"] or (tie and gi == o["idx2"]), (bl, q, j, gi, o)
            assert abs(float(g["power"]) - o["p1"]) <= RTOL * o["p1"]
            assert abs(float(g["snr"]) - o["snr"]) <= RTOL * max(o["snr"], 1e-30)
    plan.close()
