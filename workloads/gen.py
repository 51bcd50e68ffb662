"""Synthetic visibility slabs shaped like BASELINE.json's five configs.

Stand-ins for the paper's EL060 VLBI data (1.024 ms APs, 8 IFs x 16 MHz, 7 stations / 21
baselines) - the dataset itself is not available here and no record of
it is reproduced.  Recipe:

  noise   re, im ~ N(0, 1/2) iid per (bl, IF, AP, channel), complex64           ("CN(0,1)")
  pulse   boxcar over APs [t_p, t_p+W_p), adds a_p * exp(i*phi) with the PLUS sign so that the
          forward transform exp(-i Phi) of PAPER.md:74-79 (Eq. 1) peaks at +delay / +rate
  RFI     per config (single-channel tones / time-varying channels / broadband bursts)

Parameter draws use numpy PCG64(seed) on the host; the noise uses a seeded torch.Generator on the
target device, so a (config, device type, torch version) triple fixes the array.  Both the oracle
and the CUDA path always consume the SAME array (tests copy it to the host for the oracle).
Nothing here computes a DFT, a power, a peak or an SNR.
"""
import math

import numpy as np
import torch

CONFIG_IDS = (0, 1, 2, 3, 4)   # BASELINE.json configs; id 5 = the paper's own EL060-shaped segment (f2 bench only)
B_IF_HZ = 16e6  # PAPER.md:173 (Table 1: 16 MHz IFs); reading A15


def next_pow2(x):
    n = 1
    while n < x:
        n *= 2
    return n


def _stations(nbl):
    s = 2
    while s * (s - 1) // 2 < nbl:
        s += 1
    pairs = [(i, j) for i in range(s) for j in range(i + 1, s)][:nbl]
    return s, pairs


def config(cfg_id, **over):
    """Search parameters + generation recipe of BASELINE.json configs[cfg_id].
    Keyword overrides (nbl, nif, nap, nchan, npulses, ...) give reduced-size variants for tests."""
    if cfg_id == 0:
        c = dict(nbl=1, nif=1, nchan=32, nap=512, widths=[8], strides=[1], nts=[16], nf=64,
                 t_ap=1e-3, seed=0, npulses=1)
    elif cfg_id == 1:
        w = [4, 8, 16, 32]
        c = dict(nbl=1, nif=8, nchan=64, nap=2000, widths=w, strides=[x // 2 for x in w],
                 nts=[2 * x for x in w], nf=128, t_ap=1e-3, seed=1, npulses=5)
    elif cfg_id == 2:
        w = [2, 4, 8, 16, 32, 64]
        c = dict(nbl=10, nif=8, nchan=128, nap=120000, widths=w, strides=[1] * 6,
                 nts=[2 * x for x in w], nf=256, t_ap=0.5e-3, seed=2, npulses=50)
    elif cfg_id == 3:
        w = [1, 2, 4, 8, 16]
        c = dict(nbl=45, nif=16, nchan=32, nap=40000, widths=w, strides=[1] * 5,
                 nts=[2 * x for x in w], nf=128, t_ap=0.25e-3, seed=3, npulses=20)
    elif cfg_id == 4:
        w = [64, 128, 256]
        c = dict(nbl=21, nif=4, nchan=1024, nap=20000, widths=w, strides=[x // 4 for x in w],
                 nts=[512] * 3, nf=2048, t_ap=1e-3, seed=4, npulses=10)
    elif cfg_id == 5:
        # the paper's benchmark segment: 4 s of EL060-shaped data, 21 baselines,
        # 1.024 ms APs, 8 IFs x 1024 points, window sizes 2, 4, 8, 16 APs; searched with f2 (nfa = 32768)
        w = [2, 4, 8, 16]
        c = dict(nbl=21, nif=8, nchan=1024, nap=3906, widths=w, strides=[1] * 4, nts=[2 * x for x in w], nf=2048,
                 t_ap=1.024e-3, seed=5, npulses=4)
    else:
        raise ValueError("config id must be 0..5")
    c["snr_thresh"] = 6.0  # PAPER.md:208 "SNR > 6"; A15
    c["id"] = cfg_id
    c.update(over)
    return c


def nwin(nap, w, s):
    return 0 if nap < w else (nap - w) // s + 1


def nwin_total(c):
    return c["nbl"] * c["nif"] * sum(nwin(c["nap"], w, s) for w, s in zip(c["widths"], c["strides"]))


def _add(vis, bl, ifq, t_lo, t_hi, k_lo, k_hi, amp, phase):
    """vis[bl, ifq, t_lo:t_hi, k_lo:k_hi] += amp * exp(i phase); phase is a float64 tensor of the
    block's shape (or broadcastable to it), amp a float or a float64 tensor like phase."""
    amp = torch.as_tensor(amp, dtype=torch.float64, device=vis.device)
    z = torch.polar(amp.expand(phase.shape).contiguous(), phase)
    vis[bl, ifq, t_lo:t_hi, k_lo:k_hi] += z.to(torch.complex64)


def generate(cfg_id, device="cpu", **over):
    """Returns (vis complex64 [nbl][nif][nap][nchan] on `device`, cfg dict, truth dict)."""
    c = config(cfg_id, **over)
    nbl, nif, nap, nchan = c["nbl"], c["nif"], c["nap"], c["nchan"]
    dev = torch.device(device)
    g = torch.Generator(device=dev)
    g.manual_seed(1000 + c["seed"])
    vis = torch.empty((nbl, nif, nap, nchan), dtype=torch.complex64, device=dev)
    vr = torch.view_as_real(vis)
    for b in range(nbl):
        for n in range(nif):
            vr[b, n].normal_(0.0, math.sqrt(0.5), generator=g)

    rng = np.random.Generator(np.random.PCG64(c["seed"]))
    nst, pairs = _stations(nbl)
    df = B_IF_HZ / nchan
    kk = torch.arange(nchan, dtype=torch.float64, device=dev)[None, :]
    truth = dict(pulses=[], rfi=[])
    npul = c["npulses"]
    wmin, wmax = {0: (8, 8), 1: (2, 32), 2: (2, 64), 3: (1, 16), 4: (64, 256), 5: (2, 16)}[cfg_id]
    alo, ahi = {0: (0.5, 0.5), 1: (0.2, 1.0), 2: (0.3, 1.0), 3: (0.1, 0.5), 4: (0.03, 0.1), 5: (0.05, 0.15)}[cfg_id]
    slot = nap // max(npul, 1)
    for p in range(npul):
        W = int(rng.integers(wmin, wmax + 1))
        W = min(W, max(slot - 1, 1), nap)
        a = float(rng.uniform(alo, ahi))
        if cfg_id == 0:
            tp = 200 if nap >= 208 else 0
        else:
            tp = p * slot + int(rng.integers(0, max(slot - W, 1)))
        tt = torch.arange(tp, tp + W, dtype=torch.float64, device=dev)[:, None]
        rec = dict(t0=tp, width=W, amp=a)
        if cfg_id == 0:
            phi0 = float(rng.uniform(0, 2 * math.pi))
            ph = 2 * math.pi * (5.0 * kk / 32.0 + 2.0 * tt / 8.0) + phi0   # t = absolute AP (A17)
            _add(vis, 0, 0, tp, tp + W, 0, nchan, a, ph)
            rec.update(delay_bin=5, rate_bin=2)
        elif cfg_id == 1:
            tau_c = float(rng.uniform(-0.5, 0.5))   # cycles / channel  (A18)
            rho_c = float(rng.uniform(-0.5, 0.5))   # cycles / AP
            phi0 = float(rng.uniform(0, 2 * math.pi))
            for n in range(nif):                    # identical delay / rate across IFs
                ph = 2 * math.pi * (tau_c * (kk + n * nchan) + rho_c * (tt - tp)) + phi0
                _add(vis, 0, n, tp, tp + W, 0, nchan, a, ph)
            rec.update(tau_c=tau_c, rho_c=rho_c)
        else:
            tau_st = rng.uniform(-50e-9, 50e-9, nst)     # per-station residual delay
            nu_st = rng.uniform(-5e-3, 5e-3, nst)        # per-station residual rate [Hz]
            phi_bl = rng.uniform(0, 2 * math.pi, nbl)
            for b, (i, j) in enumerate(pairs):
                tau, nu = tau_st[j] - tau_st[i], nu_st[j] - nu_st[i]
                for n in range(nif):
                    ph = 2 * math.pi * ((n * B_IF_HZ + kk * df) * tau + nu * (tt - tp) * c["t_ap"]) + phi_bl[b]
                    _add(vis, b, n, tp, tp + W, 0, nchan, a, ph)
            rec.update(tau_st=tau_st.tolist(), nu_st=nu_st.tolist())
        truth["pulses"].append(rec)

    ta = torch.arange(nap, dtype=torch.float64, device=dev)[:, None]
    if cfg_id == 1:      # 3 single-channel tones at 20x noise amplitude
        for _ in range(3):
            n, k = int(rng.integers(0, nif)), int(rng.integers(0, nchan))
            nu, psi = float(rng.uniform(-0.05, 0.05)), float(rng.uniform(0, 2 * math.pi))
            _add(vis, 0, n, 0, nap, k, k + 1, 20.0, 2 * math.pi * nu * ta + psi)
            truth["rfi"].append(dict(ifq=n, chan=k, amp=20.0, nu=nu))
    elif cfg_id == 2:    # 1 % of channels, time-varying, 10-50x noise, baseline 0 only
        nr = max(1, round(0.01 * nif * nchan))
        for _ in range(nr):
            n, k = int(rng.integers(0, nif)), int(rng.integers(0, nchan))
            A, P = float(rng.uniform(10, 50)), float(rng.uniform(1e2, 1e4))
            psi, nu = float(rng.uniform(0, 2 * math.pi)), float(rng.uniform(-0.01, 0.01))
            env = A * 0.5 * (1.0 + torch.sin(2 * math.pi * ta / P + psi))
            _add(vis, 0, n, 0, nap, k, k + 1, env, 2 * math.pi * nu * ta + psi)
            truth["rfi"].append(dict(bl=0, ifq=n, chan=k, amp=A, period=P))
    elif cfg_id == 3:    # bursty broadband RFI in 0.5 % of APs on 2 baselines
        nb = max(1, round(0.005 * nap))
        for b in range(min(2, nbl)):
            aps = rng.choice(nap, size=nb, replace=False)
            for t in aps.tolist():
                A, tau_c = float(rng.uniform(2, 5)), float(rng.uniform(-0.5, 0.5))
                psi = float(rng.uniform(0, 2 * math.pi))
                for n in range(nif):
                    _add(vis, b, n, t, t + 1, 0, nchan, A, 2 * math.pi * tau_c * (kk + n * nchan) + psi)
                truth["rfi"].append(dict(bl=b, ap=t, amp=A, tau_c=tau_c))
    return vis, c, truth
