"""The five workloads of BASELINE.json `configs`, as plain data.

Each config lists one or more *plans* (config 4 has four DM ranges).  Where
BASELINE.json gives no subband DM the arithmetic mean of the plan's DM list is
used (reading A5); DM ranges "lo-hi step" are half-open (reading A6).
"""
from __future__ import annotations

import numpy as np


def _dms(lo, hi, step):
    n = int(round((hi - lo) / step))
    return lo + step * np.arange(n, dtype=np.float64)


def _plan(dms, downsamp, subband_dm=None, nsub=64):
    dms = np.asarray(dms, dtype=np.float64)
    if subband_dm is None:
        subband_dm = float(dms.mean())
    return dict(dm_list=dms, downsamp=int(downsamp), subband_dm=float(subband_dm), nsub=int(nsub))


CONFIGS = {
    # configs[0]: Tiny
    "tiny": dict(
        nchan=64, f_top=1500.0, chan_bw=-7.8125, dt=98.304e-6, nsamp=8192, dtype="u8",
        noise=dict(mean=128.0, sigma=16.0), seed=0,
        pulses=dict(kind="fixed", items=[dict(dm=100.0, width=4, amp=40.0, t0=3000)]),
        plans=[_plan(np.arange(0.0, 160.0, 5.0), 1, subband_dm=77.5, nsub=8)],
    ),
    # configs[1]: CRAFTS-like single beam (the configuration the metric is quoted on)
    "crafts": dict(
        nchan=4096, f_top=1500.0, chan_bw=-0.1220703125, dt=49.152e-6, nsamp=1 << 20, dtype="u8",
        noise=dict(mean=128.0, sigma=12.0), seed=1,
        pulses=dict(kind="random", n=20, dm=(50.0, 900.0), width=(1, 32), snr=(8.0, 30.0)),
        plans=[_plan(np.arange(0.0, 1024.0, 1.0), 1, nsub=64)],
    ),
    # configs[2]: UWB-like low-frequency wideband
    "uwb": dict(
        nchan=4096, f_top=1620.0, chan_bw=-0.32958984375, dt=98.304e-6, nsamp=1 << 21, dtype="u8",
        noise=dict(mean=128.0, sigma=12.0), seed=2,
        pulses=dict(kind="random", n=10, dm=(10.0, 480.0), width=(1, 32), snr=(8.0, 30.0)),
        plans=[_plan(np.arange(0.0, 512.0, 1.0), 2, nsub=128)],
    ),
    # configs[3]: multi-stage DDplan float32, four DM ranges back to back
    "ddplan": dict(
        nchan=4096, f_top=1500.0, chan_bw=-0.1220703125, dt=49.152e-6, nsamp=1 << 21, dtype="f32",
        noise=dict(mean=0.0, sigma=1.0), seed=3,
        pulses=dict(kind="random", n=30, dm=(10.0, 2900.0), width=(1, 32), snr=(8.0, 30.0)),
        plans=[_plan(_dms(0.0, 300.0, 0.5), 1), _plan(_dms(300.0, 600.0, 1.0), 2),
               _plan(_dms(600.0, 1200.0, 2.0), 4), _plan(_dms(1200.0, 3000.0, 5.0), 8)],
    ),
    # configs[4]: 19-beam streaming; per-beam geometry of "crafts", 4 blocks of 2^19
    "stream19": dict(
        nchan=4096, f_top=1500.0, chan_bw=-0.1220703125, dt=49.152e-6, nsamp=1 << 21, dtype="u8",
        noise=dict(mean=128.0, sigma=12.0), seed=100,   # beam b uses seed 100 + b
        pulses=dict(kind="random", n=5, dm=(50.0, 900.0), width=(1, 32), snr=(8.0, 30.0)),
        plans=[_plan(np.arange(0.0, 1024.0, 1.0), 1, nsub=64)],
        nbeams=19, block=1 << 19, nblocks=4,
    ),
}


def get_config(name, **overrides):
    cfg = dict(CONFIGS[name])
    cfg.update(overrides)
    cfg["name"] = name
    return cfg


def plan_args(cfg, plan_index=0, nsamp=None):
    """Keyword arguments of gsp_plan_create / oracle.delay_tables for one plan of a config."""
    p = cfg["plans"][plan_index]
    return dict(nchan=cfg["nchan"], f_top=cfg["f_top"], chan_bw=cfg["chan_bw"], dt=cfg["dt"],
                nsamp=int(cfg["nsamp"] if nsamp is None else nsamp), nsub=p["nsub"],
                subband_dm=p["subband_dm"], dm_list=p["dm_list"], downsamp=p["downsamp"],
                dtype=cfg["dtype"])
