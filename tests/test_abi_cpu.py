"""CPU-side checks of the boundary: the library loads, exports every symbol include/volks.h
declares, validates parameters before touching CUDA, and the host-side calls work without a GPU."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def vb():
    from paper_2108_05602_b200 import build
    build.build()
    import paper_2108_05602_b200 as v
    return v


def test_exports_every_declared_symbol(vb):
    hdr = open(os.path.join(ROOT, "include", "volks.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(volks_[a-z0-9_]+)\s*\(", hdr))
    assert {"volks_plan_create", "volks_fringe_search", "volks_window_match"} <= declared
    L = vb.lib()
    for name in declared:
        assert hasattr(L, name), name
    from paper_2108_05602_b200 import binding
    assert declared == set(binding.EXPORTS)


def test_struct_sizes_match_header(vb):
    assert vb.CAND_DTYPE.itemsize == 36 and vb.PEAK_DTYPE.itemsize == 16 and vb.PULSE_DTYPE.itemsize == 48


@pytest.mark.parametrize("kw", [
    dict(nts=[12]), dict(nts=[4]), dict(nf=48), dict(nf=16), dict(widths=[0]), dict(strides=[0]),
    dict(nbl=0), dict(nchan=0), dict(nap=-1), dict(widths=[], strides=[], nts=[]),
])
def test_plan_create_rejects_bad_params_before_cuda(vb, kw):
    a = dict(nbl=1, nif=1, nap=512, nchan=32, widths=[8], strides=[1], nts=[16], nf=64, snr_thresh=6.0)
    a.update(kw)
    rc, h = vb.plan_create_raw(**a)
    assert rc == -1 and not h


def test_options_defaults_and_validation_before_cuda(vb):
    """volks_options: defaults from volks_options_init; bad values and a mismatched struct size are rejected
    before any CUDA call; nf above the row kernels' 8192 points is an explicit VOLKS_EINVAL."""
    o = vb.make_options()
    assert (o.struct_bytes, o.full_index, o.force_generic, o.slide_seg, o.y_pad, o.chunk_mb, o.cf_wpc, o.cf2, o.ai_waves,
            o.host_split, o.no_prune, o.prune_seg, o.delay_lo, o.delay_hi) == (56, 0, 0, 256, 16, 4096, 128, 2, 2, 4, 0, 64, 0, -1)
    a = dict(nbl=1, nif=1, nap=512, nchan=32, widths=[8], strides=[1], nts=[16], nf=64, snr_thresh=6.0)
    for bad in (dict(slide_seg=8), dict(y_pad=3), dict(y_pad=-2), dict(chunk_mb=0), dict(cf2=3), dict(ai_waves=0),
                dict(host_split=0), dict(cf_wpc=0), dict(prune_seg=48), dict(prune_seg=8),
                dict(delay_lo=0, delay_hi=64), dict(delay_lo=-1, delay_hi=3), dict(delay_lo=64, delay_hi=3), dict(delay_hi=-2)):
        rc, h = vb.plan_create_raw(options=bad, **a)
        assert rc == -1 and not h, bad
    o = vb.make_options()
    o.struct_bytes = 48
    rc, h = vb.plan_create_raw(options=o, **a)
    assert rc == -1 and not h
    with pytest.raises(KeyError):
        vb.make_options(no_such_option=1)
    rc, h = vb.plan_create_raw(**dict(a, nf=16384))
    assert rc == -1 and not h
    src = open(os.path.join(ROOT, "paper_2108_05602_b200", "csrc", "volks_api.cu")).read()
    assert "getenv" not in src          # the library reads no environment variables


def test_strerror_and_version(vb):
    L = vb.lib()
    assert L.volks_version() >= 100
    assert L.volks_strerror(0) == b"ok" and b"invalid" in L.volks_strerror(-1)


def test_null_arguments(vb):
    L = vb.lib()
    assert L.volks_plan_create(None, None) == -1
    assert L.volks_plan_destroy(None) == -1
    assert L.volks_plan_query(None, None, None, None) == -1
    assert L.volks_fringe_search(None, None, None, None, None, 0, None, None) == -1


def test_no_oracle_or_fallback_in_product():
    """The product path must not import or link anything under oracle/ (nor any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2108_05602_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no CPU fallback", ""), f
                assert "cufft" not in src.lower(), f


def _mk(vb, rows):
    c = np.zeros(len(rows), dtype=vb.CAND_DTYPE)
    for i, (bl, ifq, wid, win, t0, snr) in enumerate(rows):
        c[i]["bl"], c[i]["ifq"], c[i]["wid"], c[i]["win"], c[i]["t0"], c[i]["snr"] = bl, ifq, wid, win, t0, snr
    return c


def test_window_match_host_vs_oracle(vb, oracle):
    """a8 runs on the host (integer work): product sweep vs the oracle's O(n^2) union-find."""
    rng = np.random.default_rng(8)
    widths = [2, 4, 8, 16, 32]
    for trial in range(20):
        rows = []
        for _ in range(int(rng.integers(0, 150))):
            rows.append((int(rng.integers(0, 3)), int(rng.integers(0, 2)), int(rng.integers(0, 5)), 0,
                         int(rng.integers(0, 400)), float(rng.integers(60, 90)) / 10))
        rows.sort(key=lambda r: (r[0], r[1], r[2], r[4]))
        got = vb.window_match(_mk(vb, rows), widths, 2)
        oc = np.zeros(len(rows), dtype=oracle.CAND_DTYPE)
        for i, r in enumerate(rows):
            oc[i]["bl"], oc[i]["ifq"], oc[i]["wid"], oc[i]["win"], oc[i]["t0"], oc[i]["snr"] = r
        exp = oracle.window_match(oc, widths, 2)
        assert len(got) == len(exp)
        for g, e in zip(got, exp):
            r = rows[int(e["rep"])]
            assert (g["best"]["bl"], g["best"]["ifq"], g["best"]["wid"], g["best"]["t0"]) == (r[0], r[1], r[2], r[4])
            assert g["best"]["snr"] == np.float32(r[5])
            assert (g["nwidths_hit"], g["t_begin"], g["t_end"]) == (e["nwidths_hit"], e["t_begin"], e["t_end"])


def test_window_match_capacity_and_errors(vb):
    L = vb.lib()
    c = _mk(vb, [(0, 0, 0, 0, 0, 7.0), (0, 0, 1, 0, 1, 8.0), (0, 0, 0, 50, 50, 7.0), (0, 0, 1, 25, 50, 7.5)])
    w = np.array([4, 8], np.int32)
    out = np.zeros(1, dtype=vb.PULSE_DTYPE)
    n = ctypes.c_uint32()
    rc = L.volks_window_match(c.ctypes.data, 4, w.ctypes.data, 2, 2, out.ctypes.data, 1, ctypes.byref(n))
    assert rc == -4 and n.value == 2 and out[0]["best"]["t0"] == 1
    bad = c.copy(); bad[0]["wid"] = 5
    assert L.volks_window_match(bad.ctypes.data, 4, w.ctypes.data, 2, 2, out.ctypes.data, 1, ctypes.byref(n)) == -1


def test_bin_to_physical(vb):
    r, d = vb.bin_to_physical(16, 64, 4, 10, 1e-3, 5e5)
    assert r == pytest.approx(4 / (16 * 1e-3)) and d == pytest.approx(10 / (64 * 5e5))
    r, d = vb.bin_to_physical(16, 64, 12, 54, 1e-3, 5e5)
    assert r == pytest.approx(-4 / (16 * 1e-3)) and d == pytest.approx(-10 / (64 * 5e5))
    r, d = vb.bin_to_physical(16, 64, 8, 32, 1e-3, 5e5)          # Nyquist bins are negative
    assert r < 0 and d < 0
    with pytest.raises(vb.VolksError):
        vb.bin_to_physical(16, 64, 16, 0, 1e-3, 5e5)


def test_dm_shifts_host_vs_oracle(vb, oracle):
    f = 1400.0 + 16.0 * np.arange(8)[:, None] + 0.25 * np.arange(64)[None, :]
    for dm in (0.0, 26.8, 557.0):
        got = vb.dm_shifts(dm, f, f.max(), 1.024e-3)
        assert np.array_equal(got, oracle.dm_shifts(dm, f, f.max(), 1.024e-3))
    assert vb.dm_shifts(100.0, np.array([1400.0, 1500.0]), 1500.0, 1e-3).tolist() == [27, 0]


def test_baseline_match_host_vs_oracle(vb, oracle):
    """f3: constructions (5 baselines overlapping -> kept; 4 -> dropped; same baseline repeated does
    not count twice; chain overlap A-B-C is one cluster) and random lists against the O(n^2) oracle."""
    def mk(rows):
        p = np.zeros(len(rows), dtype=vb.PULSE_DTYPE)
        for i, (bl, tb, te, snr) in enumerate(rows):
            p[i]["best"]["bl"], p[i]["best"]["snr"], p[i]["t_begin"], p[i]["t_end"] = bl, snr, tb, te
        return p
    five = mk([(b, 100 + b, 110 + b, 7.0 + b) for b in range(5)])
    d = vb.baseline_match(five, 5)
    assert len(d) == 1 and d[0]["nbaselines"] == 5 and (d[0]["t_begin"], d[0]["t_end"]) == (100, 114)
    assert d[0]["best"]["best"]["bl"] == 4
    assert len(vb.baseline_match(five[:4], 5)) == 0
    rep = mk([(0, 10, 20, 8.0), (0, 12, 22, 9.0), (1, 15, 25, 7.0)])
    assert len(vb.baseline_match(rep, 3)) == 0 and vb.baseline_match(rep, 2)[0]["nbaselines"] == 2
    chain = mk([(0, 0, 10, 6.5), (1, 9, 20, 6.6), (2, 19, 30, 6.4), (3, 40, 50, 9.0)])
    d = vb.baseline_match(chain, 3)
    assert len(d) == 1 and (d[0]["t_begin"], d[0]["t_end"], d[0]["nbaselines"]) == (0, 30, 3)
    rng = np.random.default_rng(9)
    for trial in range(20):
        n = int(rng.integers(0, 60))
        rows = [(int(rng.integers(0, 10)), int(t), int(t + rng.integers(1, 30)), float(rng.integers(60, 90)) / 10)
                for t in rng.integers(0, 600, n)]
        p = mk(rows)
        got = vb.baseline_match(p, 3)
        exp = oracle.baseline_match(p["best"]["bl"], p["best"]["snr"], p["t_begin"], p["t_end"], 3)
        assert len(got) == len(exp)
        for g, e in zip(got, exp):
            assert g["best"].tobytes() == p[e["rep"]].tobytes()
            assert (g["nbaselines"], g["t_begin"], g["t_end"]) == (e["nbaselines"], e["t_begin"], e["t_end"])
    cap = (ctypes.c_uint32(), np.zeros(1, dtype=vb.DETECTION_DTYPE))
    two = mk([(b, 100, 110, 7.0) for b in range(5)] + [(b, 300, 310, 7.0) for b in range(5)])
    rc = vb.lib().volks_baseline_match(two.ctypes.data, len(two), 5, cap[1].ctypes.data, 1, ctypes.byref(cap[0]))
    assert rc == -4 and cap[0].value == 2


def test_cal_phasors_host_vs_oracle(vb, oracle):
    rng = np.random.default_rng(2)
    d, p = rng.uniform(-50e-9, 50e-9, (3, 4)), rng.uniform(-3, 3, (3, 4))
    got = vb.cal_phasors(d, p, 64, 250e3)
    exp = oracle.cal_phasors(d, p, 64, 250e3)
    assert got.shape == exp.shape == (3, 4, 64) and np.abs(got - exp).max() < 3e-7
    assert np.allclose(np.abs(got), 1.0, atol=1e-6)
