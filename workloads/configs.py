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


# The paper's own DDplans (Tables 2 and 3) on its two FAST-UWB bands (Table 1):
# (low DM, high DM, dDM, DownSamp, number of DMs); the DM list of a range is low + dDM * arange(number).
_TABLE2_BAND1 = [(0.0, 11.34, 0.01, 1, 1134), (11.34, 22.2, 0.03, 2, 362), (22.2, 39.05, 0.05, 4, 337),
                 (39.05, 77.15, 0.1, 8, 381), (77.15, 153.75, 0.2, 16, 383), (153.75, 343.75, 0.5, 32, 380),
                 (343.75, 687.75, 1.0, 64, 344), (687.75, 969.75, 2.0, 128, 141)]
_TABLE3_BAND2 = [(0.0, 48.77, 0.01, 1, 4877), (48.77, 93.14, 0.03, 2, 1479), (93.14, 164.74, 0.05, 4, 1432),
                 (164.74, 325.04, 0.1, 8, 1603), (325.04, 485.04, 0.2, 16, 800), (485.04, 592.84, 0.2, 16, 539)]


def _table_plans(table, nsub):
    return [_plan(lo + step * np.arange(n, dtype=np.float64), ds, nsub=nsub) for lo, hi, step, ds, n in table]


CONFIGS.update({
    # Band1 of Table 1: 512 channels over 271-398 MHz (0.25 MHz wide), 98 us, one 52 s drift
    # (2^19 samples = 51.5 s), 8-bit; Table 2's eight DM ranges, 3462 trial DMs, DownSamp 1 ... 128.
    # One subband DM per range (reading A5); 32 subbands of 16 channels.
    "band1": dict(
        nchan=512, f_top=397.875, chan_bw=-0.25, dt=98.304e-6, nsamp=1 << 19, dtype="u8",
        noise=dict(mean=128.0, sigma=12.0), seed=11,
        pulses=dict(kind="random", n=10, dm=(5.0, 900.0), width=(1, 32), snr=(8.0, 30.0)),
        plans=_table_plans(_TABLE2_BAND1, 32),
    ),
    # Band2 of Table 1: 2048 channels over 291-802 MHz, same sampling; Table 3's six ranges, 10,730 trial DMs.
    # 64 subbands of 32 channels.
    "band2": dict(
        nchan=2048, f_top=801.875, chan_bw=-0.25, dt=98.304e-6, nsamp=1 << 19, dtype="u8",
        noise=dict(mean=128.0, sigma=12.0), seed=12,
        pulses=dict(kind="random", n=10, dm=(5.0, 580.0), width=(1, 32), snr=(8.0, 30.0)),
        plans=_table_plans(_TABLE3_BAND2, 64),
    ),
})


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
