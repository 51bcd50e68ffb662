"""volks_search_noalloc (include/volks.h): the search for callers that cannot allocate - no plan, no workspace, every
intermediate in the library's static 32 MiB device array.  Checked against the existing path (volks_fringe_search
through a plan) on the same inputs, with the comparison rules the parity tests use (tests/_parity.py: power / snr to
1e-4 relative, the peak bin equal unless the top two powers lie within 1e-5), on two calls in a row with DIFFERENT
inputs and shapes, so that anything the scratch keeps from the first call would show in the second.

This file sorts last on purpose (pytest -x: a failure here hides nothing after it).  It passes
alone in a fresh process and after the other tests: it shares nothing with them but the loaded library."""
import numpy as np
import pytest
import torch

import workloads

pytestmark = pytest.mark.gpu

RTOL, TIE = 1e-4, 1e-5


@pytest.fixture(scope="module")
def vb():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2108_05602_b200 as v
    v.lib()
    return v


def _noalloc(vb, dvis, c, thresh, cap=1 << 16):
    nbl, nif, nap, nchan = dvis.shape
    nwin_total = nbl * nif * sum(workloads.gen.nwin(nap, w, s) for w, s in zip(c["widths"], c["strides"]))
    dev = dvis.device
    cands = torch.empty(cap * vb.CAND_DTYPE.itemsize, dtype=torch.uint8, device=dev)
    ncand = torch.full((1,), -7, dtype=torch.int32, device=dev)
    peaks = torch.empty(max(nwin_total, 1) * vb.PEAK_DTYPE.itemsize, dtype=torch.uint8, device=dev)
    rc = vb.search_noalloc(dvis, c["widths"], c["strides"], c["nts"], c["nf"], thresh, cands, ncand, peaks)
    assert rc == 0, vb.lib().volks_strerror(rc)
    torch.cuda.synchronize(dev)
    n = int(ncand.item())
    return (cands[: min(n, cap) * vb.CAND_DTYPE.itemsize].cpu().numpy().view(vb.CAND_DTYPE), n,
            peaks[: nwin_total * vb.PEAK_DTYPE.itemsize].cpu().numpy().view(vb.PEAK_DTYPE))


def _compare(vb, vis, c, thresh):
    dvis = vis.cuda()
    rc_, rn, rp = vb.fringe_search(dvis, c["widths"], c["strides"], c["nts"], c["nf"], thresh, want_peaks=True)   # existing path
    gc, gn, gp = _noalloc(vb, dvis, c, thresh)
    assert len(gp) == len(rp) > 0
    nf = c["nf"]
    ref_p = rp["power"].astype(np.float64)
    safe = np.where(ref_p > 0, ref_p, 1.0)
    assert np.all(np.abs(gp["power"] - ref_p) <= RTOL * safe)
    assert np.all(np.abs(gp["snr"].astype(np.float64) - rp["snr"]) <= RTOL * np.maximum(rp["snr"], 1e-30))
    same = (gp["rate_idx"] == rp["rate_idx"]) & (gp["delay_idx"] == rp["delay_idx"])
    # a differing bin is only allowed where the two paths' powers agree to the near-tie margin (both are maxima of the
    # same plane: the rule of tests/_parity.py with the existing path in the oracle's place)
    diff = np.nonzero(~same)[0]
    assert np.all(np.abs(gp["power"][diff] - ref_p[diff]) <= 2 * TIE * safe[diff]) and diff.size <= max(2, len(gp) // 200), diff[:5]
    # candidate lists: the same windows in canonical order, except windows whose snr sits on the threshold
    key = lambda a: list(zip(a["bl"].tolist(), a["ifq"].tolist(), a["wid"].tolist(), a["win"].tolist()))
    gk, rk = key(gc), key(rc_)
    assert gk == sorted(gk)
    marg = int(np.count_nonzero(np.abs(rp["snr"] - thresh) <= RTOL * thresh))
    assert len(set(gk) ^ set(rk)) <= marg and abs(gn - rn) <= marg
    rmap = {k: i for i, k in enumerate(rk)}
    for k, g in zip(gk, gc):
        if k in rmap:
            r = rc_[rmap[k]]
            assert g["t0"] == r["t0"] and abs(float(g["power"]) - float(r["power"])) <= RTOL * float(r["power"])
            assert abs(float(g["snr"]) - float(r["snr"])) <= RTOL * float(r["snr"])
    return gn


def test_noalloc_matches_existing_path_twice_in_a_row(vb):
    # call 1: BASELINE.json configs[0] (w = 8, plane 16 x 64; the injected pulse gives candidates)
    vis0, c0, _ = workloads.generate(0)
    n0 = _compare(vb, vis0, c0, c0["snr_thresh"])
    assert n0 >= 1
    # call 2, right after, another shape and other data: configs[1] at reduced extent (4 widths, stride w/2, 8 IFs)
    vis1, c1, _ = workloads.generate(1, nap=600)
    n1 = _compare(vb, vis1, c1, 4.0)
    assert n1 >= 1
    # call 3: the first problem again - the scratch now holds call 2's leftovers; the answer must be call 1's
    assert _compare(vb, vis0, c0, c0["snr_thresh"]) == n0


def test_noalloc_rejects_what_does_not_fit(vb):
    """Sizes beyond the static scratch are refused with VOLKS_ELIMIT before anything is enqueued; bad parameters with
    VOLKS_EINVAL; a search with no windows writes a zero count."""
    dev = torch.device("cuda")
    cands = torch.empty(36 * 16, dtype=torch.uint8, device=dev)
    ncand = torch.full((1,), 123, dtype=torch.int32, device=dev)
    big = torch.zeros((1, 1, 40000, 128), dtype=torch.complex64, device=dev)          # Y alone: 40000 x 272 x 8 B = 87 MB
    rc = vb.search_noalloc(big, [8], [1], [16], 256, 6.0, cands, ncand)
    assert rc == vb.binding.VOLKS_ELIMIT and b"static scratch" in vb.lib().volks_strerror(rc)
    torch.cuda.synchronize()
    assert int(ncand.item()) == 123                                                   # nothing ran
    small = torch.zeros((1, 1, 10, 8), dtype=torch.complex64, device=dev)
    assert vb.search_noalloc(small, [4], [1], [6], 8, 6.0, cands, ncand) == vb.binding.VOLKS_EINVAL      # nt not a power of two
    assert vb.search_noalloc(small, [4], [1], [8], 4, 6.0, cands, ncand) == vb.binding.VOLKS_EINVAL      # nf < nchan
    assert vb.search_noalloc(small, [16], [1], [16], 8, 6.0, cands, ncand) == 0                          # nap < w: no windows
    torch.cuda.synchronize()
    assert int(ncand.item()) == 0
