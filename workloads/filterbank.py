"""Seeded synthetic filterbanks standing in for the paper's FAST PSRFITS files
(PAPER.md:176 — 8-bit, 256-4k channels, ~98 us, injected simulated pulses).

x[t][c], time-major, channel 0 = highest frequency.  Noise is Gaussian from a seeded
torch generator on the requested device, generated in fixed-size time chunks so the
bytes depend only on (seed, device type, shape).  Pulses are top-hats of `width`
samples whose arrival in channel c is delayed by the cold-plasma law relative to
channel 0 (reading A17).  uint8 samples are clip(rint(mean + sigma*g + pulses), 0, 255).
"""
from __future__ import annotations

import numpy as np
import torch

# Signal model of the injected pulses (not the library's delay-table builder):
# arrival delay in seconds = KDM_SIGNAL * DM * (f^-2 - f0^-2), f in MHz.
KDM_SIGNAL = 4.148808e3
_CHUNK_ROWS = 1 << 14


def pulse_table(cfg, seed=None, nsamp=None):
    """List of dict(dm, width, amp, t0) for a config; random ones drawn from default_rng(seed)."""
    spec = cfg.get("pulses")
    if not spec:
        return []
    if spec["kind"] == "fixed":
        return [dict(p) for p in spec["items"]]
    seed = cfg["seed"] if seed is None else seed
    nsamp = cfg["nsamp"] if nsamp is None else nsamp
    rng = np.random.default_rng(seed)
    sigma = cfg["noise"]["sigma"]
    f0 = cfg["f_top"]
    f_lo = cfg["f_top"] + (cfg["nchan"] - 1) * cfg["chan_bw"]
    out = []
    for _ in range(spec["n"]):
        dm = float(rng.uniform(*spec["dm"]))
        width = int(rng.integers(spec["width"][0], spec["width"][1] + 1))
        snr = float(rng.uniform(*spec["snr"]))
        sweep = int(np.ceil(KDM_SIGNAL * dm * (f_lo ** -2 - f0 ** -2) / cfg["dt"]))
        hi = max(1, nsamp - sweep - width - 1)
        t0 = int(rng.integers(0, hi))
        # "S/N-equivalent amplitude": summed over nchan*width samples the pulse
        # stands snr sigma above the noise of that sum.
        amp = snr * sigma / np.sqrt(cfg["nchan"] * width)
        out.append(dict(dm=dm, width=width, amp=float(amp), t0=t0))
    return out


def _pulse_starts(cfg, pulse):
    c = np.arange(cfg["nchan"], dtype=np.float64)
    f = cfg["f_top"] + c * cfg["chan_bw"]
    delay = KDM_SIGNAL * pulse["dm"] * (1.0 / (f * f) - 1.0 / (cfg["f_top"] ** 2)) / cfg["dt"]
    return pulse["t0"] + np.floor(delay + 0.5).astype(np.int64)


def make_filterbank(cfg, device="cpu", nsamp=None, seed=None, noise=True, pulses=True,
                    out=None):
    """Return x[nsamp][nchan] (torch uint8 or float32) on `device`.

    noise=False gives the noise-free pulse-only input (mean 0) used by the
    worked-example pin (reading A16).  `out` may be a preallocated tensor.
    """
    nsamp = int(cfg["nsamp"] if nsamp is None else nsamp)
    seed = int(cfg["seed"] if seed is None else seed)
    nchan = cfg["nchan"]
    dev = torch.device(device)
    tdtype = torch.uint8 if cfg["dtype"] == "u8" else torch.float32
    x = out if out is not None else torch.empty((nsamp, nchan), dtype=tdtype, device=dev)
    assert x.shape == (nsamp, nchan) and x.dtype == tdtype
    gen = torch.Generator(device=dev)
    gen.manual_seed(seed)
    plist = pulse_table(cfg, seed=seed, nsamp=nsamp) if pulses else []
    starts = [torch.from_numpy(_pulse_starts(cfg, p)).to(dev) for p in plist]
    lo = [int(s.min()) for s in starts]
    hi = [int(s.max()) + p["width"] for s, p in zip(starts, plist)]
    mean = cfg["noise"]["mean"] if noise else 0.0
    sigma = cfg["noise"]["sigma"] if noise else 0.0
    for ta in range(0, nsamp, _CHUNK_ROWS):
        tb = min(nsamp, ta + _CHUNK_ROWS)
        if noise:
            g = torch.randn((tb - ta, nchan), generator=gen, device=dev, dtype=torch.float32)
            g.mul_(sigma).add_(mean)
        else:
            g = torch.zeros((tb - ta, nchan), device=dev, dtype=torch.float32)
        rows = None
        for p, st, l, h in zip(plist, starts, lo, hi):
            if h <= ta or l >= tb:
                continue
            if rows is None:
                rows = torch.arange(ta, tb, device=dev, dtype=torch.int64)[:, None]
            m = (rows >= st[None, :]) & (rows < (st[None, :] + p["width"]))
            g.add_(m.to(torch.float32), alpha=p["amp"])
        if tdtype == torch.uint8:
            x[ta:tb] = g.round_().clamp_(0.0, 255.0).to(torch.uint8)
        else:
            x[ta:tb] = g
    return x
