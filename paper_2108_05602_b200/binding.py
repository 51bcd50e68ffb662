"""Thin ctypes binding of libvolks_b200.so (include/volks.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  torch is used for device memory and
streams.  There is no CPU fallback: if the shared library is missing this module raises."""
import ctypes
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libvolks_b200.so")

VOLKS_OK, VOLKS_EINVAL, VOLKS_ECUDA, VOLKS_ENOMEM, VOLKS_EOVERFLOW, VOLKS_ELIMIT = 0, -1, -2, -3, -4, -5
NOALLOC_SCRATCH_BYTES = 32 << 20      # VOLKS_NOALLOC_SCRATCH_BYTES

EXPORTS = (
    "volks_plan_create", "volks_plan_destroy", "volks_plan_query", "volks_fringe_search",
    "volks_window_match", "volks_bin_to_physical", "volks_plan_launch_count", "volks_strerror",
    "volks_version", "volks_plan_profile", "volks_plan_profile_read", "volks_fringe_search_dd", "volks_dm_shifts",
    "volks_baseline_match", "volks_zscore_select", "volks_plan_create_allif", "volks_allif_search",
    "volks_plan_query_host", "volks_search_host", "volks_plan_set_cal", "volks_cal_phasors",
    "volks_measure_fp32_peak", "volks_options_init", "volks_plan_create_opt", "volks_plan_create_allif_opt",
    "volks_search_noalloc",
)


class volks_params(ctypes.Structure):
    _fields_ = [("nbl", ctypes.c_int32), ("nif", ctypes.c_int32), ("nap", ctypes.c_int32),
                ("nchan", ctypes.c_int32), ("nwidths", ctypes.c_int32),
                ("width", ctypes.POINTER(ctypes.c_int32)), ("stride", ctypes.POINTER(ctypes.c_int32)),
                ("nt", ctypes.POINTER(ctypes.c_int32)), ("nf", ctypes.c_int32),
                ("snr_thresh", ctypes.c_float)]


class volks_options(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in ("struct_bytes", "full_index", "force_generic", "slide_seg", "y_pad",
                                              "chunk_mb", "cf_wpc", "cf2", "ai_waves", "host_split", "no_prune", "prune_seg",
                                              "delay_lo", "delay_hi")]


CAND_DTYPE = np.dtype([("bl", "<i4"), ("ifq", "<i4"), ("wid", "<i4"), ("win", "<i4"), ("t0", "<i4"),
                       ("rate_idx", "<i4"), ("delay_idx", "<i4"), ("power", "<f4"), ("snr", "<f4")])
PEAK_DTYPE = np.dtype([("power", "<f4"), ("snr", "<f4"), ("rate_idx", "<i4"), ("delay_idx", "<i4")])
PULSE_DTYPE = np.dtype([("best", CAND_DTYPE), ("nwidths_hit", "<i4"), ("t_begin", "<i4"), ("t_end", "<i4")])
DETECTION_DTYPE = np.dtype([("best", PULSE_DTYPE), ("nbaselines", "<i4"), ("t_begin", "<i4"), ("t_end", "<i4")])
assert CAND_DTYPE.itemsize == 36 and PEAK_DTYPE.itemsize == 16 and PULSE_DTYPE.itemsize == 48
assert DETECTION_DTYPE.itemsize == 60

_lib = None


def lib():
    """Load the C-ABI library; fails loudly if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(
                "libvolks_b200.so is missing: run `python -m paper_2108_05602_b200.build` "
                "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        L.volks_strerror.restype = ctypes.c_char_p
        L.volks_strerror.argtypes = [ctypes.c_int]
        L.volks_plan_create.argtypes = [ctypes.POINTER(volks_params), ctypes.POINTER(ctypes.c_void_p)]
        L.volks_plan_create_allif.argtypes = [ctypes.POINTER(volks_params), ctypes.POINTER(ctypes.c_void_p)]
        L.volks_options_init.argtypes = [ctypes.POINTER(volks_options)]
        L.volks_options_init.restype = None
        L.volks_plan_create_opt.argtypes = [ctypes.POINTER(volks_params), ctypes.POINTER(volks_options), ctypes.POINTER(ctypes.c_void_p)]
        L.volks_plan_create_allif_opt.argtypes = [ctypes.POINTER(volks_params), ctypes.POINTER(volks_options), ctypes.POINTER(ctypes.c_void_p)]
        L.volks_allif_search.argtypes = [ctypes.c_void_p] * 6 + [ctypes.c_uint32, ctypes.c_void_p, ctypes.c_void_p]
        L.volks_plan_query_host.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_size_t)]
        L.volks_search_host.argtypes = [ctypes.c_void_p] * 7 + [ctypes.c_uint32, ctypes.c_void_p, ctypes.c_void_p]
        L.volks_plan_set_cal.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
        L.volks_cal_phasors.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int32, ctypes.c_int32,
                                        ctypes.c_double, ctypes.c_void_p]
        L.volks_measure_fp32_peak.argtypes = [ctypes.c_int32, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double),
                                              ctypes.POINTER(ctypes.c_double), ctypes.c_void_p]
        L.volks_search_noalloc.argtypes = [ctypes.POINTER(volks_params), ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                           ctypes.c_uint32, ctypes.c_void_p, ctypes.c_void_p]
        L.volks_plan_destroy.argtypes = [ctypes.c_void_p]
        L.volks_plan_query.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_size_t),
                                       ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_int64)]
        L.volks_fringe_search.argtypes = [ctypes.c_void_p] * 5 + [ctypes.c_uint32, ctypes.c_void_p, ctypes.c_void_p]
        L.volks_fringe_search_dd.argtypes = [ctypes.c_void_p] * 6 + [ctypes.c_uint32, ctypes.c_void_p, ctypes.c_void_p]
        L.volks_dm_shifts.argtypes = [ctypes.c_double, ctypes.c_void_p, ctypes.c_int32, ctypes.c_double,
                                      ctypes.c_double, ctypes.c_void_p]
        L.volks_zscore_select.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_float, ctypes.c_void_p,
                                          ctypes.c_void_p, ctypes.c_uint32, ctypes.c_void_p, ctypes.c_void_p]
        L.volks_baseline_match.argtypes = [ctypes.c_void_p, ctypes.c_uint32, ctypes.c_int32, ctypes.c_void_p,
                                           ctypes.c_uint32, ctypes.POINTER(ctypes.c_uint32)]
        L.volks_window_match.argtypes = [ctypes.c_void_p, ctypes.c_uint32, ctypes.c_void_p, ctypes.c_int32,
                                         ctypes.c_int32, ctypes.c_void_p, ctypes.c_uint32,
                                         ctypes.POINTER(ctypes.c_uint32)]
        L.volks_bin_to_physical.argtypes = [ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32,
                                            ctypes.c_double, ctypes.c_double,
                                            ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
        L.volks_plan_launch_count.argtypes = [ctypes.c_void_p]
        L.volks_plan_profile.argtypes = [ctypes.c_void_p, ctypes.c_int]
        L.volks_plan_profile_read.argtypes = [ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p, ctypes.c_void_p,
                                              ctypes.c_void_p, ctypes.POINTER(ctypes.c_int32)]
        _lib = L
    return _lib


class VolksError(RuntimeError):
    def __init__(self, code):
        self.code = code
        super().__init__("volks error %d: %s" % (code, lib().volks_strerror(code).decode()))


def _check(rc):
    if rc != VOLKS_OK:
        raise VolksError(rc)


def make_options(**kw):
    """volks_options_init + keyword overrides (full_index, force_generic, slide_seg, y_pad, chunk_mb, cf_wpc, cf2,
    ai_waves, host_split, no_prune, prune_seg, delay_lo, delay_hi)."""
    o = volks_options()
    lib().volks_options_init(ctypes.byref(o))
    for k, v in kw.items():
        if k not in dict(volks_options._fields_) or k == "struct_bytes":
            raise KeyError("unknown volks option %r" % k)
        setattr(o, k, int(v))
    return o


def plan_create_raw(nbl, nif, nap, nchan, widths, strides, nts, nf, snr_thresh, allif=False, options=None):
    """volks_plan_create[_allif][_opt]; returns (rc, handle) without raising (for error-path tests).
    options: None (defaults), a dict of overrides, or a volks_options."""
    n = len(widths)
    arr = lambda v: (ctypes.c_int32 * max(len(v), 1))(*[int(x) for x in v])
    w, s, t = arr(widths), arr(strides), arr(nts)
    p = volks_params(nbl, nif, nap, nchan, n, w, s, t, nf, float(snr_thresh))
    h = ctypes.c_void_p()
    if options is None:
        rc = (lib().volks_plan_create_allif if allif else lib().volks_plan_create)(ctypes.byref(p), ctypes.byref(h))
    else:
        o = make_options(**options) if isinstance(options, dict) else options
        rc = (lib().volks_plan_create_allif_opt if allif else lib().volks_plan_create_opt)(
            ctypes.byref(p), ctypes.byref(o), ctypes.byref(h))
    return rc, h


class Plan:
    """volks_plan_* : validated parameters + window schedule + device tables."""

    def __init__(self, nbl, nif, nap, nchan, widths, strides, nts, nf, snr_thresh, allif=False, options=None):
        """allif=True: the f2 plan (volks_plan_create_allif; `nts` ignored, nf = nfa).
        options: dict of volks_options overrides (e.g. dict(full_index=1)) or None."""
        self.allif = bool(allif)
        nts = [1] * len(widths) if allif else nts
        self.shape = (nbl, nif, nap, nchan)
        self.widths, self.strides, self.nts, self.nf = list(widths), list(strides), list(nts), nf
        self.snr_thresh = float(snr_thresh)
        rc, self._h = plan_create_raw(nbl, nif, nap, nchan, widths, strides, nts, nf, snr_thresh, allif, options)
        _check(rc)
        ws, tot = ctypes.c_size_t(), ctypes.c_int64()
        per = (ctypes.c_int64 * len(widths))()
        _check(lib().volks_plan_query(self._h, ctypes.byref(ws), per, ctypes.byref(tot)))
        self.workspace_bytes, self.nwin_total, self.nwin_per_width = ws.value, tot.value, list(per)
        self.launches = lib().volks_plan_launch_count(self._h)

    def close(self):
        if getattr(self, "_h", None):
            lib().volks_plan_destroy(self._h)
            self._h = None

    __del__ = close

    def fringe_search(self, vis, workspace, cands, ncand, peaks=None, stream=None, shift=None):
        """volks_fringe_search[_dd] on torch CUDA tensors (asynchronous on `stream`).
        vis complex64 [nbl][nif][nap][nchan]; workspace uint8 >= workspace_bytes;
        cands uint8 [capacity*36]; ncand int32/uint32 [1]; peaks uint8 [nwin_total*16] or None;
        shift int32 CUDA [nif][nchan] dedispersion AP offsets or None."""
        assert vis.is_cuda and vis.dtype == torch.complex64 and vis.is_contiguous()
        assert tuple(vis.shape) == self.shape
        assert workspace.is_cuda and workspace.numel() * workspace.element_size() >= self.workspace_bytes
        cap = cands.numel() * cands.element_size() // CAND_DTYPE.itemsize
        if peaks is not None:
            assert peaks.numel() * peaks.element_size() >= self.nwin_total * PEAK_DTYPE.itemsize
        st = (stream or torch.cuda.current_stream(vis.device)).cuda_stream
        if shift is not None:
            assert shift.is_cuda and shift.dtype == torch.int32 and shift.is_contiguous()
            assert tuple(shift.shape) == (self.shape[1], self.shape[3])
        _check((lib().volks_allif_search if self.allif else lib().volks_fringe_search_dd)(
            self._h, vis.data_ptr(), shift.data_ptr() if shift is not None else None, workspace.data_ptr(),
            peaks.data_ptr() if peaks is not None else None, cands.data_ptr() if cap else None, cap,
            ncand.data_ptr(), st))

    def set_cal(self, cal):
        """volks_plan_set_cal: cal = CUDA complex64 [nbl][nif][nchan] (kept alive by this object) or None."""
        if cal is not None:
            assert cal.is_cuda and cal.dtype == torch.complex64 and cal.is_contiguous()
            assert tuple(cal.shape) == (self.shape[0], self.shape[1], self.shape[3])
        self._cal = cal
        _check(lib().volks_plan_set_cal(self._h, cal.data_ptr() if cal is not None else None))

    @property
    def stage_bytes(self):
        """volks_plan_query_host: bytes of ONE half of the staging buffer of search_host."""
        n = ctypes.c_size_t()
        _check(lib().volks_plan_query_host(self._h, ctypes.byref(n)))
        return n.value

    def search_host(self, h_vis, stage, workspace, cands, ncand, peaks=None, stream=None, shift=None):
        """volks_search_host: h_vis is a HOST complex64 tensor (pinned recommended), `stage` a CUDA uint8
        tensor of >= 2 * stage_bytes; copies overlap the kernels chunk by chunk.  Asynchronous."""
        assert (not h_vis.is_cuda) and h_vis.dtype == torch.complex64 and h_vis.is_contiguous()
        assert tuple(h_vis.shape) == self.shape
        assert stage.is_cuda and stage.numel() * stage.element_size() >= 2 * self.stage_bytes
        cap = cands.numel() * cands.element_size() // CAND_DTYPE.itemsize
        st = (stream or torch.cuda.current_stream(stage.device)).cuda_stream
        _check(lib().volks_search_host(
            self._h, h_vis.data_ptr(), stage.data_ptr(), shift.data_ptr() if shift is not None else None,
            workspace.data_ptr(), peaks.data_ptr() if peaks is not None else None,
            cands.data_ptr() if cap else None, cap, ncand.data_ptr(), st))

    def zscore_select(self, workspace, z_thresh, cands, ncand, peaks=None, stream=None):
        """volks_zscore_select: across-window normalised selection on the last search's workspace."""
        cap = cands.numel() * cands.element_size() // CAND_DTYPE.itemsize
        st = (stream or torch.cuda.current_stream(workspace.device)).cuda_stream
        _check(lib().volks_zscore_select(self._h, workspace.data_ptr(), float(z_thresh),
                                         peaks.data_ptr() if peaks is not None else None,
                                         cands.data_ptr() if cap else None, cap, ncand.data_ptr(), st))

    def profile(self, enable=True):
        """volks_plan_profile: bracket every launch of later searches with CUDA events."""
        _check(lib().volks_plan_profile(self._h, 1 if enable else 0))

    def profile_read(self):
        """volks_plan_profile_read -> list of (kind, width index, milliseconds), launch order."""
        n = ctypes.c_int32()
        _check(lib().volks_plan_profile_read(self._h, 0, None, None, None, ctypes.byref(n)))
        kind, wid = np.zeros(n.value, np.int32), np.zeros(n.value, np.int32)
        ms = np.zeros(n.value, np.float32)
        _check(lib().volks_plan_profile_read(self._h, n.value, kind.ctypes.data, wid.ctypes.data,
                                             ms.ctypes.data, ctypes.byref(n)))
        return [(int(k), int(w), float(m)) for k, w, m in zip(kind, wid, ms)]

    def window_match(self, cands, min_widths=2):
        return window_match(cands, self.widths, min_widths)

    def bin_to_physical(self, wid, rate_idx, delay_idx, ap_seconds, chan_hz):
        return bin_to_physical(self.nts[wid], self.nf, rate_idx, delay_idx, ap_seconds, chan_hz)


def window_match(cands, widths, min_widths=2):
    """volks_window_match on a host numpy CAND_DTYPE array (canonical order)."""
    cands = np.ascontiguousarray(cands, dtype=CAND_DTYPE)
    w = np.ascontiguousarray(widths, dtype=np.int32)
    out = np.zeros(max(len(cands), 1), dtype=PULSE_DTYPE)
    n = ctypes.c_uint32()
    _check(lib().volks_window_match(cands.ctypes.data, len(cands), w.ctypes.data, len(w), min_widths,
                                    out.ctypes.data, len(out), ctypes.byref(n)))
    return out[:n.value]


def cal_phasors(delay_s, phase_rad, nchan, chan_hz):
    """volks_cal_phasors: complex64 [..., nchan] calibration phasors for delay_s / phase_rad of shape [...]."""
    d = np.ascontiguousarray(delay_s, dtype=np.float64)
    p = np.ascontiguousarray(phase_rad, dtype=np.float64)
    assert d.shape == p.shape
    out = np.zeros(d.shape + (nchan, 2), dtype=np.float32)
    _check(lib().volks_cal_phasors(d.ctypes.data, p.ctypes.data, d.size, nchan, float(chan_hz), out.ctypes.data))
    return out.view(np.complex64)[..., 0]


def baseline_match(pulses, min_baselines=5):
    """volks_baseline_match on a host numpy PULSE_DTYPE array (the output of window_match)."""
    pulses = np.ascontiguousarray(pulses, dtype=PULSE_DTYPE)
    out = np.zeros(max(len(pulses), 1), dtype=DETECTION_DTYPE)
    n = ctypes.c_uint32()
    _check(lib().volks_baseline_match(pulses.ctypes.data, len(pulses), min_baselines, out.ctypes.data, len(out),
                                      ctypes.byref(n)))
    return out[:n.value]


def search_noalloc(vis, widths, strides, nts, nf, snr_thresh, cands, ncand, peaks=None, stream=None):
    """volks_search_noalloc: the search without plan or workspace (every intermediate in the library's static 32 MiB
    device array; no allocation inside the call).  All buffers are the caller's torch CUDA tensors: vis complex64
    [nbl][nif][nap][nchan]; cands uint8 [capacity*36]; ncand int32 [1]; peaks uint8 [nwin_total*16] or None.
    Asynchronous on `stream`.  Returns the library's code (VOLKS_OK / VOLKS_ELIMIT ...) without raising."""
    assert vis.is_cuda and vis.dtype == torch.complex64 and vis.is_contiguous()
    nbl, nif, nap, nchan = vis.shape
    n = len(widths)
    arr = lambda v: (ctypes.c_int32 * max(len(v), 1))(*[int(x) for x in v])
    w, s, t = arr(widths), arr(strides), arr(nts)
    p = volks_params(nbl, nif, nap, nchan, n, w, s, t, int(nf), float(snr_thresh))
    cap = cands.numel() * cands.element_size() // CAND_DTYPE.itemsize
    st = (stream or torch.cuda.current_stream(vis.device)).cuda_stream
    return lib().volks_search_noalloc(ctypes.byref(p), vis.data_ptr(), peaks.data_ptr() if peaks is not None else None,
                                      cands.data_ptr() if cap else None, cap, ncand.data_ptr(), st)


def measure_fp32_peak(repeats=5, stream=None):
    """volks_measure_fp32_peak -> (best TFLOP/s, mean TFLOP/s, ms per launch) on the current device."""
    best, mean, ms = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    st = (stream or torch.cuda.current_stream()).cuda_stream
    _check(lib().volks_measure_fp32_peak(int(repeats), ctypes.byref(best), ctypes.byref(mean), ctypes.byref(ms), st))
    return best.value, mean.value, ms.value


def bin_to_physical(nt, nf, rate_idx, delay_idx, ap_seconds, chan_hz):
    r, d = ctypes.c_double(), ctypes.c_double()
    _check(lib().volks_bin_to_physical(nt, nf, rate_idx, delay_idx, ap_seconds, chan_hz,
                                       ctypes.byref(r), ctypes.byref(d)))
    return r.value, d.value


def dm_shifts(dm, f_chan_mhz, f_ref_mhz, ap_seconds):
    """volks_dm_shifts: int32 AP shifts (same shape as f_chan_mhz) for one dispersion measure."""
    f = np.ascontiguousarray(f_chan_mhz, dtype=np.float64)
    out = np.zeros(f.shape, dtype=np.int32)
    _check(lib().volks_dm_shifts(float(dm), f.ctypes.data, f.size, float(f_ref_mhz), float(ap_seconds), out.ctypes.data))
    return out


def allif_search(vis, widths, strides, nfa, snr_thresh, want_peaks=False, cand_capacity=1 << 20, shifts=None,
                 options=None):
    """One-shot f2 search (volks_plan_create_allif + volks_allif_search); returns like fringe_search."""
    nbl, nif, nap, nchan = vis.shape
    plan = Plan(nbl, nif, nap, nchan, widths, strides, None, nfa, snr_thresh, allif=True, options=options)
    try:
        return fringe_search(vis, want_peaks=want_peaks, cand_capacity=cand_capacity, plan=plan, shifts=shifts)
    finally:
        plan.close()


def fringe_search(vis, widths=None, strides=None, nts=None, nf=None, snr_thresh=None, want_peaks=False,
                  cand_capacity=1 << 20, plan=None, shifts=None, options=None):
    """Convenience one-shot call: allocates workspace/outputs with torch, runs the search on the
    current stream, synchronises and returns (cands CAND_DTYPE[n], ncand_true, peaks|None)."""
    if not vis.is_cuda:
        raise RuntimeError("volks fringe_search needs a CUDA tensor (there is no CPU fallback)")
    own = plan is None
    if own:
        nbl, nif, nap, nchan = vis.shape
        plan = Plan(nbl, nif, nap, nchan, widths, strides, nts, nf, snr_thresh, options=options)
    dev = vis.device
    ws = torch.empty(plan.workspace_bytes, dtype=torch.uint8, device=dev)
    cands = torch.empty(cand_capacity * CAND_DTYPE.itemsize, dtype=torch.uint8, device=dev)
    ncand = torch.zeros(1, dtype=torch.int32, device=dev)
    peaks = torch.empty(max(plan.nwin_total, 1) * PEAK_DTYPE.itemsize, dtype=torch.uint8, device=dev) if want_peaks else None
    shift = None if shifts is None else torch.as_tensor(np.ascontiguousarray(shifts, dtype=np.int32), device=dev)
    plan.fringe_search(vis, ws, cands, ncand, peaks, shift=shift)
    torch.cuda.synchronize(dev)
    n = int(ncand.item()) & 0xFFFFFFFF
    c = cands[: min(n, cand_capacity) * CAND_DTYPE.itemsize].cpu().numpy().view(CAND_DTYPE)
    p = peaks[: plan.nwin_total * PEAK_DTYPE.itemsize].cpu().numpy().view(PEAK_DTYPE) if want_peaks else None
    if own:
        plan.close()
    return c, n, p
