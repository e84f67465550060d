#!/usr/bin/env python
"""bench.py — throughput of the whole hot path (stage 1 + downsample + stage 2); one JSON line on stdout.

    python bench.py --gpus N --steps K --warmup W            # libgsp (CUDA) arm, BASELINE configs[1] ("crafts")
    python bench.py --config uwb|ddplan|band1|band2|stream19 # the other workloads (multi-plan configs run all
                                                             # their DM ranges in one gsp_dedisperse_multi call)
    python bench.py --gpus N --shard dm                      # one beam, DM list sharded over N GPUs (strong scaling)
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle, timed as it stands, same workload

A "step" is one pass of the whole path over one synthetic beam already resident in HBM (`value`), and the
same through gsp_dedisperse_host from pinned host buffers (`e2e`).  N > 1: one process per GPU (launched by
torchrun, or spawned by this script when it is started without one): replicas only — every rank dedisperses
its own beam, no collective on the data path; value = units of all ranks / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import socket
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "DM-trial*samples/s dedispersed"
UNIT = "GS/s"
SM_COUNT, ADD_LANES, SM_MAX_HZ = 148, 128, 1.965e9       # add-pipe peak
PEAK_TADD = SM_COUNT * ADD_LANES * SM_MAX_HZ / 1e12        # 37.2 Tadd/s


def _measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return None


def sources_sha16():
    """Hash of the CUDA/C++ sources libgsp.so is built from: ties profiles/traffic.csv to a build."""
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_2110_12749_b200", "csrc")
    for name in sorted(os.listdir(csrc)):
        if name.endswith((".cu", ".cuh", ".cpp", ".h")):
            h.update(name.encode())
            h.update(open(os.path.join(csrc, name), "rb").read())
    return h.hexdigest()[:16]


def _ncu_traffic(kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of `kernel` on the benchmark workload from the
    committed `ncu --set full` summary profiles/traffic.csv — only when that capture was made from THIS build's
    sources (first line `# sources_sha16=...`); otherwise None and a note saying so."""
    try:
        lines = open(os.path.join(ROOT, "profiles", "traffic.csv")).read().splitlines()
        tag = [l for l in lines if l.startswith("# sources_sha16=")]
        if not tag or tag[0].split("=", 1)[1].strip() != sources_sha16():
            return None, "profiles/traffic.csv was captured from other sources than this build"
        for line in lines:
            f = [t.strip() for t in line.split(",")]
            if len(f) >= 3 and f[0] == kernel:
                return float(f[1]) + float(f[2]), "profiles/traffic.csv (ncu --set full, same sources)"
    except Exception:
        pass
    return None, "no ncu capture committed"


def reduce_max(x, dist=None, device="cpu"):
    """MAX over ranks of a scalar (the multi-GPU timing rule); identity for a single process."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_seed(cfg, rank):
    """Replicas only: rank r dedisperses its own beam, seeded cfg.seed + r."""
    return int(cfg["seed"]) + int(rank)


def dm_shard(dm_list, rank, world):
    """DM-sharded multi-GPU run (the MPI-PRESTO decomposition PAPER.md:176):
    rank r takes a contiguous slice of the sorted trial-DM list (neighbouring DMs share stage-2 windows)."""
    dm_list = np.asarray(dm_list, dtype=np.float64)
    bounds = [(len(dm_list) * r) // world for r in range(world + 1)]
    return dm_list[bounds[rank]:bounds[rank + 1]], bounds[rank]


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.rows, self.proc, self.th = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            return
        self.th = threading.Thread(target=self._pump, daemon=True)
        self.th.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append([t.strip() for t in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except Exception:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def _workload_string(a, nout, name="crafts"):
    dms = a["dm_list"]
    return (f"{name}: {a['nchan']} ch, f_top {a['f_top']} MHz, chan_bw {a['chan_bw']} MHz, dt {a['dt']*1e6:.3f} us, "
            f"nsamp {a['nsamp']}, {a['dtype']} noise+pulses, {a['nsub']} subbands @DM {a['subband_dm']}, "
            f"{len(dms)} DMs {dms[0]:g}-{dms[-1]:g}, downsamp {a['downsamp']}, nout {nout}")


def _l2_policy(in_bytes, out_bytes, host_arm=False):
    return (f"inputs ({in_bytes / 2**30:.2f} GiB) and outputs ({out_bytes / 2**30:.2f} GiB) larger than the "
            f"126 MB L2: no flush between iterations" if min(in_bytes, out_bytes) > 2 * 126e6 else
            f"inputs {in_bytes / 2**20:.1f} MiB / outputs {out_bytes / 2**20:.1f} MiB: L2-resident workload, "
            + ("host arm: nothing is flushed between iterations" if host_arm else
               "a 256 MiB buffer is written between iterations"))


def cpu_oracle_rate(a, cfg, sample_nsamp, steps=1, warmup=0, x=None, nthreads=None, keep=False):
    """Time the oracle, as it stands, on a bounded sample of the workload (host cores)."""
    import oracle
    s1, s2 = oracle.delay_tables(a["nchan"], a["f_top"], a["chan_bw"], a["dt"], a["nsub"],
                                 a["subband_dm"], a["dm_list"], a["downsamp"])
    if x is None:
        x = workloads.make_filterbank(cfg, nsamp=sample_nsamp).numpy()
    nthr = oracle.max_threads() if nthreads is None else nthreads
    g = oracle.geometry(sample_nsamp, s1, s2, a["downsamp"])
    y = None
    for _ in range(warmup):
        oracle.dedisperse(x, s1, s2, a["downsamp"], nthreads=nthr)
    t0 = time.perf_counter()
    for _ in range(steps):
        y = oracle.dedisperse(x, s1, s2, a["downsamp"], nthreads=nthr)
    dt = (time.perf_counter() - t0) / steps
    units = len(a["dm_list"]) * g["nout"]
    cb = dict(value=units / dt / 1e9, unit=UNIT, cores=nthr, kind="oracle", cpu_model=cpu_model(),
              sample=f"first {sample_nsamp} of {a['nsamp']} samples, all {len(a['dm_list'])} DMs "
                     f"({units:.3e} DM-samples, {dt:.2f} s per pass, {steps} passes timed)")
    return cb, dt, units, (y if keep else None)


def run_reference(args):
    """The tier's reference arm: the oracle as it stands on the box's host cores, on the SAME workload as the
    gsp arm (the whole beam, one oracle pass per step)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = workloads.get_config(args.config)
    a = workloads.plan_args(cfg, args.plan or 0)
    if args.nsamp:
        a["nsamp"] = args.nsamp
    warm = min(args.warmup, 3)             # the same W as the gsp arm (a pass is seconds: bounded at 3)
    cb, dt, units, _ = cpu_oracle_rate(a, cfg, a["nsamp"], steps=args.steps, warmup=warm)
    import oracle
    g = oracle.geometry(a["nsamp"], *oracle.delay_tables(a["nchan"], a["f_top"], a["chan_bw"], a["dt"], a["nsub"],
                                                         a["subband_dm"], a["dm_list"], a["downsamp"]), a["downsamp"])
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT,
            "n_gpus": args.gpus, "steps": args.steps, "warmup": warm, "ms_per_step": dt * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int64",
            "data": "synthetic",
            # the same `config` as the gsp arm prints for this workload, key for key
            "config": {"workload": _workload_string(a, g["nout"], args.config),
                       "l2_policy": _l2_policy(a["nsamp"] * a["nchan"] * (1 if a["dtype"] == "u8" else 4),
                                               len(a["dm_list"]) * g["nout"] * 4, host_arm=True)},
            "parallelism": f"host cores, OpenMP x{cb['cores']}",
            "cpu_baseline": cb,
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def _dist_setup():
    import torch
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libgsp has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    return world, rank, local, dist


def run_gsp(args):
    import torch

    import paper_2110_12749_b200 as gsp

    world, rank, local, dist = _dist_setup()
    cfg = workloads.get_config(args.config)
    a = workloads.plan_args(cfg, args.plan or 0)
    if args.nsamp:
        a["nsamp"] = args.nsamp
    shard = args.shard == "dm" and world > 1
    dm_off = 0
    if shard:
        a["dm_list"], dm_off = dm_shard(a["dm_list"], rank, world)
    plan = gsp.Plan(a["nchan"], a["f_top"], a["chan_bw"], a["dt"], a["nsamp"], a["nsub"],
                    a["subband_dm"], a["dm_list"], a["downsamp"], a["dtype"])
    stream = torch.cuda.current_stream().cuda_stream
    bcast_ms = None
    if shard:
        # one beam for the whole job: generated on rank 0, broadcast over NVLink (the only collective; it is
        # not on the per-step path and is timed on its own)
        tdtype = torch.uint8 if a["dtype"] == "u8" else torch.float32
        x = (workloads.make_filterbank(cfg, device="cuda", nsamp=a["nsamp"]) if rank == 0
             else torch.empty((a["nsamp"], a["nchan"]), dtype=tdtype, device="cuda"))
        torch.cuda.synchronize()
        dist.barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        dist.broadcast(x, src=0)
        e1.record()
        torch.cuda.synchronize()
        bcast_ms = reduce_max(e0.elapsed_time(e1), dist, "cuda")
    else:
        x = workloads.make_filterbank(cfg, device="cuda", nsamp=a["nsamp"], seed=replica_seed(cfg, rank))
    out = torch.empty((plan.ndm, plan.out_pitch), dtype=torch.float32, device="cuda")
    units = plan.ndm * plan.nout
    in_bytes = x.numel() * x.element_size()
    out_bytes = plan.ndm * plan.nout * 4
    flush = None
    if min(in_bytes, out_bytes) <= 2 * 126e6:
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    # ---- device-resident timing ------------------------------------------------------------
    for _ in range(args.warmup):
        plan.dedisperse(x, out, stream)
    barrier()
    plan.enable_stage_timing(True)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.2)
    barrier()
    ms_total = 0.0
    if flush is None:
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        for _ in range(args.steps):
            plan.dedisperse(x, out, stream)
        ev1.record()
        barrier()
        ms_total = ev0.elapsed_time(ev1)
    else:
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        for e0, e1 in evs:
            flush.fill_(1)                       # evict the workload from L2 (outside the timed events)
            e0.record()
            plan.dedisperse(x, out, stream)
            e1.record()
        barrier()
        ms_total = sum(e0.elapsed_time(e1) for e0, e1 in evs)
    ms1, ms2, ncalls = plan.stage_ms_total()
    plan.enable_stage_timing(False)
    ms_step = reduce_max(ms_total, dist, "cuda") / args.steps
    total_units = units
    if dist is not None:
        t = torch.tensor([float(units)], dtype=torch.float64, device="cuda")
        dist.all_reduce(t)
        total_units = float(t.item())
    value = total_units / (ms_step * 1e-3) / 1e9

    # ---- the step after the path, on the device: single-pulse search on d_out (gsp_search_*) ----
    search = None
    if not args.no_search and plan.out_pitch % 4 == 0 and plan.ndm <= 65535:
        cap = 1 << 20
        with gsp.Search(plan.ndm, plan.nout, plan.out_pitch, 1024, 6, 7.0, cap) as srch:
            bufs = [torch.empty(cap, dtype=torch.int32, device="cuda") for _ in range(3)]
            snr = torch.empty(cap, dtype=torch.float32, device="cuda")
            cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
            for _ in range(2):
                srch.run(out, bufs[0], bufs[1], bufs[2], snr, cnt, None, stream)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(5):
                srch.run(out, bufs[0], bufs[1], bufs[2], snr, cnt, None, stream)
            e1.record()
            torch.cuda.synchronize()
            s_ms = e0.elapsed_time(e1) / 5
            search = {"api": "gsp_search_run on d_out (block 1024, widths 1-32, threshold 7.0)", "ms": s_ms,
                      "candidates": int(cnt.item()), "achieved_GBps": out_bytes / (s_ms * 1e-3) / 1e9,
                      "d2h_bytes_instead_of_output": int(cnt.item()) * 16 + 8}

    # ---- the step before the path, fused into stage 1: RFI prologue on (channel mask + zero-DM clip) ----
    # (reported beside the headline, never part of it: the timed steps above run without a prologue)
    rfi = None
    if not args.no_rfi and a["dtype"] == "u8" and 1024 * a["nchan"] * 255 < (1 << 31):
        import numpy as np
        rng = np.random.default_rng(12)
        mask = (rng.random(a["nchan"]) < 0.05).astype(np.uint8)
        pad = np.full(a["nchan"], 128, dtype=np.uint8)
        plan.set_rfi(mask, pad, 3.0, 1024)
        for _ in range(2):
            plan.dedisperse(x, out, stream)
        plan.enable_stage_timing(True)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(5):
            plan.dedisperse(x, out, stream)
        e1.record()
        torch.cuda.synchronize()
        r1, r2, rn = plan.stage_ms_total()
        plan.enable_stage_timing(False)
        rfi = {"api": "gsp_plan_set_rfi (5% of channels masked, zero-DM clip 3 sigma over blocks of 1024 rows)",
               "ms_per_step": e0.elapsed_time(e1) / 5, "stage1_ms": r1 / max(rn, 1), "stage2_ms": r2 / max(rn, 1),
               "stage1_impl": plan.get_impl(1), "launches_per_step": plan.launches_per_call,
               "l2": "warm (back-to-back steps)" }
        plan.set_rfi(None, None)

    # ---- end to end: host buffers through gsp_dedisperse_host -------------------------------
    e2e = None
    if not args.no_e2e:
        h_in = torch.empty(x.shape, dtype=x.dtype, pin_memory=True)
        h_in.copy_(x)
        h_out = torch.empty((plan.ndm, plan.nout), dtype=torch.float32, pin_memory=True)
        e2e_steps = max(1, min(args.steps, args.e2e_steps))
        for _ in range(min(args.warmup, 2)):
            plan.dedisperse_host(h_in, h_out, plan.nout, stream)
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            plan.dedisperse_host(h_in, h_out, plan.nout, stream)
        torch.cuda.synchronize()
        te = reduce_max((time.perf_counter() - t0) / e2e_steps, dist, "cuda")
        e2e = {"value": total_units / te / 1e9, "unit": UNIT,
               "h2d_bytes_per_step": in_bytes, "d2h_bytes_per_step": out_bytes,
               "ms_per_step": te * 1e3, "steps": e2e_steps,
               "api": "gsp_dedisperse_host (pinned host in/out, chunked H2D/kernels/D2H pipeline)"}
        del h_out
        # ---- end to end for the pipeline the paper runs (dedispersion -> single-pulse search):
        # host input through gsp_dedisperse_host_in (series stay on the device), gsp_search_run on them, and only
        # the candidate list copied back
        if search is not None:
            cap = 1 << 20
            with gsp.Search(plan.ndm, plan.nout, plan.out_pitch, 1024, 6, 7.0, cap) as srch:
                bufs = [torch.empty(cap, dtype=torch.int32, device="cuda") for _ in range(3)]
                snr = torch.empty(cap, dtype=torch.float32, device="cuda")
                cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
                h_cnt = torch.zeros(1, dtype=torch.int64, pin_memory=True)
                h_c = [torch.empty(cap, dtype=torch.int32, pin_memory=True) for _ in range(3)]
                h_snr = torch.empty(cap, dtype=torch.float32, pin_memory=True)

                def pipeline_step():
                    plan.dedisperse_host_in(h_in, out, plan.out_pitch, stream)
                    srch.run(out, bufs[0], bufs[1], bufs[2], snr, cnt, None, stream)
                    h_cnt.copy_(cnt, non_blocking=True)
                    torch.cuda.synchronize()
                    n = min(int(h_cnt.item()), cap)
                    for hb, db in zip(h_c + [h_snr], bufs + [snr]):
                        hb[:n].copy_(db[:n], non_blocking=True)
                    torch.cuda.synchronize()
                    return n

                pipeline_step()
                barrier()
                t0 = time.perf_counter()
                for _ in range(e2e_steps):
                    ncand = pipeline_step()
                ts = reduce_max((time.perf_counter() - t0) / e2e_steps, dist, "cuda")
            e2e["search"] = {"value": total_units / ts / 1e9, "unit": UNIT, "ms_per_step": ts * 1e3,
                             "h2d_bytes_per_step": in_bytes, "d2h_bytes_per_step": 8 + 16 * ncand,
                             "candidates": ncand,
                             "api": "gsp_dedisperse_host_in (pinned host in, series left on the device) + "
                                    "gsp_search_run + copy of the candidate list"}
        del h_in
    # the sampler covers both timed regions (device-resident steps and the end-to-end steps)
    clocks = sampler.stop() if rank == 0 else None

    if rank != 0:
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (stage 2) -------------------------------------------
    k2_ms = ms2 / max(ncalls, 1)
    k1_ms = ms1 / max(ncalls, 1)
    k2_adds = float(plan.ndm) * plan.nsub * plan.nout            # one add per (DM, subband, sample)
    k1_adds = float(plan.nchan) * plan.n1
    achieved = k2_adds / (k2_ms * 1e-3) / 1e12
    peaks = _measured_peaks()
    hbm = (peaks or {}).get("hbm_gbs", 6650.0)
    t_hbm = (in_bytes + out_bytes) / (hbm * 1e9)
    t_add = (k1_adds + k2_adds) / (PEAK_TADD * 1e12)
    ws_bytes = plan.nsub * plan.n1d * 4                          # subband intermediate, written then read
    k2_bytes = ws_bytes + out_bytes
    k1_bytes = in_bytes + ws_bytes
    f32 = a["dtype"] == "f32"
    packed = (not f32) and (a["nchan"] // a["nsub"]) * 255 * a["downsamp"] <= 65535
    smem_feed_tadd = SM_COUNT * (64 if packed else 32) * SM_MAX_HZ / 1e12   # operands per 32-bit LDS lane: 2 u16 / 1 word
    split = plan.stage1_split
    k1_name = ("stage1_f32_stream_kernel (TMA-fed time-major ring, lanes = channels)" if f32 and split[4] else
               "stage1_f32_kernel (de-skewing tile)" if f32 else
               "stage1_stream_u8_kernel (TMA-fed channel->subband + downsample)" +
               (" (+ its long-ring instantiation)" if split[5] + split[6] else "") +
               (" + stage1_u8_wide_kernel" if split[1] + split[2] else "") +
               (" + stage1_tiled_u8_kernel" if split[3] else ""))
    tr2, note2 = _ncu_traffic("stage2") if args.config == "crafts" and not args.nsamp else (None, "not captured for this workload")
    tr1, _ = _ncu_traffic("stage1") if args.config == "crafts" and not args.nsamp else (None, None)
    roofline = {"bound": "alu", "kernel": "stage2_tiled_kernel (subband->DM shift-and-sum + store)",
                "achieved": achieved, "peak": PEAK_TADD, "unit": "Tadd/s", "frac": achieved / PEAK_TADD,
                "traffic": tr2, "traffic_source": note2,
                "peak_source": "148 SMs x 128 add lanes x 1.965 GHz (DESIGN.md §7; unit counts and clock from the B200 "
                               "guides; issue rates measured by the committed microbenchmark, profiles/r2_microbench.md)",
                "kernel_ms": k2_ms, "algorithmic_adds": k2_adds, "algorithmic_bytes": k2_bytes,
                "smem_operand_feed_peak": smem_feed_tadd,
                "frac_of_smem_operand_feed": achieved / smem_feed_tadd,
                "stage1": {"bound": "hbm", "kernel": k1_name,
                           "kernel_ms": k1_ms, "algorithmic_bytes": k1_bytes,
                           "achieved": k1_bytes / (k1_ms * 1e-3) / 1e9 if k1_ms > 0 else None,
                           "peak": hbm, "unit": "GB/s",
                           "frac": k1_bytes / (k1_ms * 1e-3) / 1e9 / hbm if k1_ms > 0 else None,
                           "peak_source": "MEASURED_PEAKS.json hbm_gbs (of measured)" if peaks
                                          else "6650 GB/s (of fallback)",
                           "traffic": tr1},
                "path_roofline_ms": max(t_hbm, t_add) * 1e3,
                "path_roofline_frac": max(t_hbm, t_add) * 1e3 / ms_step}

    cb = None
    if not args.no_cpu:
        # bounded sample, about 10-30 s of host work: the whole beam once when it is the 2^20-sample uint8
        # workload — and then EVERY output of the GPU run is compared with it — else the first 2^19 samples
        whole = a["dtype"] == "u8" and a["nsamp"] <= (1 << 20)
        ns = a["nsamp"] if whole else min(a["nsamp"], 1 << 19)
        cb, _, _, y_or = cpu_oracle_rate(a, cfg, ns, steps=1, x=x[:ns].cpu().numpy(), keep=whole)
        if whole:
            plan.dedisperse(x, out, stream)
            torch.cuda.synchronize()
            nbad = 0
            for d0 in range(0, plan.ndm, 128):
                nbad += int((out[d0:d0 + 128, : plan.nout].cpu().numpy() != y_or[d0:d0 + 128]).sum())
            cb["gpu_output_equals_oracle"] = (nbad == 0)
            cb["outputs_compared"] = int(y_or.size)
            if nbad:
                print(json.dumps({"error": f"{nbad} GPU outputs differ from the oracle"}))
                raise SystemExit(3)
            del y_or
        # one thread, on a 2^16-sample slice (the whole beam would take minutes)
        n1t = min(a["nsamp"], max(1 << 16, plan.halo + 16384))
        c1, _, _, _ = cpu_oracle_rate(a, cfg, n1t, steps=1, x=x[:n1t].cpu().numpy(), nthreads=1)
        cb["value_1thread"] = c1["value"]
        cb["sample_1thread"] = c1["sample"]

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "strong" if shard else "weak",
            "vs_baseline": None, "dtype": "int32" if a["dtype"] == "u8" else "f32", "data": "synthetic",
            "config": {"workload": _workload_string(a, plan.nout, args.config),
                       "l2_policy": _l2_policy(in_bytes, out_bytes)},
            "parallelism": (f"one beam broadcast from rank 0, DM list sharded x{world}" if shard
                            else f"replicas x{world}"),
            "kernels": {"stage1_impl": plan.get_impl(1), "stage2_impl": plan.get_impl(2),
                        "stage1_split": list(plan.stage1_split)},
            "realtime_factor": (1 if shard else world) * a["nsamp"] * a["dt"] / (ms_step * 1e-3),
            "clocks": clocks, "e2e": e2e, "gpu_launches": plan.launches_per_call * args.steps,
            "roofline": roofline, "cpu_baseline": cb, "search": search, "rfi": rfi}
    if shard:
        line["input_broadcast_ms"] = bcast_ms
    print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def run_multi(args):
    """Multi-plan configs (ddplan: BASELINE configs[3]; band1 / band2: the paper's Tables 2-3): every DM range
    over the same beam in ONE gsp_dedisperse_multi call per step (shared stage-1 launches)."""
    import torch

    import paper_2110_12749_b200 as gsp

    world, rank, local, dist = _dist_setup()
    cfg = workloads.get_config(args.config)
    nsamp = args.nsamp or cfg["nsamp"]
    plans, outs, A = [], [], []
    for pi in range(len(cfg["plans"])):
        a = workloads.plan_args(cfg, pi, nsamp=nsamp)
        A.append(a)
        p = gsp.Plan(a["nchan"], a["f_top"], a["chan_bw"], a["dt"], a["nsamp"], a["nsub"], a["subband_dm"],
                     a["dm_list"], a["downsamp"], a["dtype"])
        plans.append(p)
        outs.append(torch.empty((p.ndm, p.out_pitch), dtype=torch.float32, device="cuda"))
    x = workloads.make_filterbank(cfg, device="cuda", nsamp=nsamp, seed=replica_seed(cfg, rank))
    stream = torch.cuda.current_stream().cuda_stream
    units = sum(p.ndm * p.nout for p in plans)
    in_bytes = x.numel() * x.element_size()
    out_bytes = sum(p.ndm * p.nout * 4 for p in plans)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        gsp.dedisperse_multi(plans, x, outs, stream)
    barrier()
    plans[0].enable_stage_timing(True)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.2)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(args.steps):
        gsp.dedisperse_multi(plans, x, outs, stream)
    ev1.record()
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms_step = reduce_max(ev0.elapsed_time(ev1), dist, "cuda") / args.steps
    ms1, ms2, ncalls = plans[0].stage_ms_total()
    plans[0].enable_stage_timing(False)
    # the ranges one after the other, each in its own gsp_dedisperse call (what the shared launches save)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for p, o in zip(plans, outs):
        p.dedisperse(x, o, stream)
    e1.record()
    torch.cuda.synchronize()
    ms_separate = e0.elapsed_time(e1)
    # ---- end to end: the beam from pinned host memory, every range's series back to pinned host memory ----
    # (one copy in, one gsp_dedisperse_multi call, one copy out per range; not pipelined.  Only when both sides
    # fit 8 GiB of pinned memory: the 32 GiB float32 beam of the ddplan config does not)
    e2e = None
    if not args.no_e2e and in_bytes <= (8 << 30) and out_bytes <= (8 << 30):
        h_in = torch.empty(x.shape, dtype=x.dtype, pin_memory=True)
        h_in.copy_(x)
        h_outs = [torch.empty((p.ndm, p.out_pitch), dtype=torch.float32, pin_memory=True) for p in plans]
        e2e_steps = max(1, min(args.steps, args.e2e_steps))

        def e2e_step():
            x.copy_(h_in, non_blocking=True)
            gsp.dedisperse_multi(plans, x, outs, stream)
            for ho, o in zip(h_outs, outs):
                ho.copy_(o, non_blocking=True)
            torch.cuda.synchronize()

        e2e_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            e2e_step()
        te = reduce_max((time.perf_counter() - t0) / e2e_steps, dist, "cuda")
        e2e = {"value": world * units / te / 1e9, "unit": UNIT, "h2d_bytes_per_step": in_bytes,
               "d2h_bytes_per_step": sum(o.numel() * 4 for o in outs), "ms_per_step": te * 1e3, "steps": e2e_steps,
               "api": "pinned host beam -> device, gsp_dedisperse_multi, every range's rows -> pinned host (not pipelined)"}
        del h_in, h_outs
    if rank != 0:
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return
    peaks = _measured_peaks()
    hbm = (peaks or {}).get("hbm_gbs", 6650.0)
    adds2 = sum(float(p.ndm) * p.nsub * p.nout for p in plans)
    adds1 = sum(float(p.nchan) * p.n1 for p in plans)
    t_hbm_once = (in_bytes + out_bytes) / (hbm * 1e9)                       # input read once for all ranges
    t_hbm_each = (in_bytes * len(plans) + out_bytes) / (hbm * 1e9)          # input read per range
    t_add = (adds1 + adds2) / (PEAK_TADD * 1e12)
    k2_ms = ms2 / max(ncalls, 1)
    k1_ms = ms1 / max(ncalls, 1)
    cb = None
    if not args.no_cpu:
        ns = min(nsamp, 1 << 17 if A[0]["dtype"] == "f32" else 1 << 18)
        ns = max(ns, plans[0].halo + 4096)
        cb, _, _, _ = cpu_oracle_rate(A[0], cfg, ns, steps=1, x=x[:ns].cpu().numpy())
        cb["sample"] = "range 1 of the plan: " + cb["sample"]
    line = {"metric": METRIC, "value": world * units / (ms_step * 1e-3) / 1e9, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "int32" if cfg["dtype"] == "u8" else "f32",
            "data": "synthetic",
            "config": {"workload": f"{args.config}: {cfg['nchan']} ch, f_top {cfg['f_top']} MHz, chan_bw {cfg['chan_bw']} MHz, "
                                   f"dt {cfg['dt']*1e6:.3f} us, nsamp {nsamp}, {cfg['dtype']}, {len(plans)} DM ranges "
                                   f"(DMs, downsamp, subband DM) = "
                                   + "; ".join(f"({p.ndm}, {a['downsamp']}, {a['subband_dm']:g})" for p, a in zip(plans, A))
                                   + f", {sum(p.ndm for p in plans)} trial DMs in all",
                       "parallelism": f"replicas x{world}", "l2_policy": _l2_policy(in_bytes, out_bytes),
                       "stage_impls": [[p.get_impl(1), p.get_impl(2)] for p in plans],
                       "stage1_splits": [list(p.stage1_split) for p in plans]},
            "realtime_factor": world * nsamp * cfg["dt"] / (ms_step * 1e-3),
            "ms_as_separate_calls": ms_separate,
            "clocks": clocks, "e2e": e2e,
            "gpu_launches": gsp.dedisperse_multi_launches(plans) * args.steps,
            "roofline": {"bound": "hbm" if t_hbm_once > t_add else "alu",
                         "kernel": "whole gsp_dedisperse_multi call (all ranges)",
                         "stage1_ms": k1_ms, "stage2_ms": k2_ms,
                         "achieved": (in_bytes + out_bytes) / (ms_step * 1e-3) / 1e9 if t_hbm_once > t_add
                                     else (adds1 + adds2) / (ms_step * 1e-3) / 1e12,
                         "peak": hbm if t_hbm_once > t_add else PEAK_TADD,
                         "unit": "GB/s" if t_hbm_once > t_add else "Tadd/s",
                         "frac": max(t_hbm_once, t_add) * 1e3 / ms_step, "traffic": None,
                         "path_roofline_ms_input_read_once": max(t_hbm_once, t_add) * 1e3,
                         "path_roofline_ms_input_read_per_range": max(t_hbm_each, t_add) * 1e3,
                         "path_roofline_frac_input_read_per_range": max(t_hbm_each, t_add) * 1e3 / ms_step},
            "cpu_baseline": cb}
    print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def run_stream19(args):
    """BASELINE configs[4]: 19 independent beams, each dedispersed in 4 consecutive blocks of 2^19
    samples with the max-delay overlap (H = H1 + ds*H2 rows) carried device-to-device; the H2D copy
    of block k+1 runs on a side stream under the kernels of block k.  Every step processes all 19
    beams from pinned host memory; the result read back per block is the per-DM maximum."""
    import torch

    import paper_2110_12749_b200 as gsp

    cfg = workloads.get_config("stream19")
    a = workloads.plan_args(cfg)
    B, nblk, nbeams, nchan = cfg["block"], cfg["nblocks"], cfg["nbeams"], cfg["nchan"]
    if args.beams:
        nbeams = args.beams
    torch.cuda.set_device(0)
    mk = lambda n: gsp.Plan(a["nchan"], a["f_top"], a["chan_bw"], a["dt"], n, a["nsub"], a["subband_dm"],
                            a["dm_list"], a["downsamp"], a["dtype"])
    first = mk(B)
    H = first.halo
    blk = mk(B + H)
    assert blk.nout == B
    ndistinct = min(nbeams, args.host_beams)        # distinct beams held in pinned memory, cycled
    host = []
    for b in range(ndistinct):
        xb = workloads.make_filterbank(cfg, device="cuda", seed=cfg["seed"] + b)
        hb = torch.empty(xb.shape, dtype=xb.dtype, pin_memory=True)
        hb.copy_(xb)
        host.append(hb)
        del xb
    d_in = [torch.empty((H + B, nchan), dtype=torch.uint8, device="cuda") for _ in range(2)]
    d_out = [torch.empty((blk.ndm, blk.out_pitch), dtype=torch.float32, device="cuda") for _ in range(2)]
    h_res = torch.empty((nbeams * nblk, blk.ndm), dtype=torch.float32, pin_memory=True)
    s_k, s_in = torch.cuda.Stream(), torch.cuda.Stream()
    ev_in = [torch.cuda.Event() for _ in range(2)]
    ev_k = [torch.cuda.Event() for _ in range(2)]
    ev_c = [torch.cuda.Event() for _ in range(2)]     # block using buffer i has taken its carry from buffer i^1

    def one_pass():
        n = 0
        for b in range(nbeams):
            hb = host[b % ndistinct]
            for k in range(nblk):
                i = n & 1
                with torch.cuda.stream(s_in):
                    s_in.wait_event(ev_k[i])                       # buffer i: kernels of block n-2 done
                    s_in.wait_event(ev_c[i ^ 1])                   # ... and block n-1 has copied its halo out of it
                    d_in[i][H:].copy_(hb[k * B:(k + 1) * B], non_blocking=True)
                    ev_in[i].record(s_in)
                with torch.cuda.stream(s_k):
                    s_k.wait_event(ev_in[i])
                    if k == 0:
                        first.dedisperse(d_in[i][H:], d_out[i], s_k.cuda_stream)
                        nv = first.nout
                    else:
                        d_in[i][:H].copy_(d_in[i ^ 1][B:], non_blocking=True)   # the carried halo
                    ev_c[i].record(s_k)
                    if k > 0:
                        blk.dedisperse(d_in[i], d_out[i], s_k.cuda_stream)
                        nv = B
                    h_res[n].copy_(d_out[i][:, :nv].amax(dim=1), non_blocking=True)
                    ev_k[i].record(s_k)
                n += 1
        torch.cuda.synchronize()

    for _ in range(max(1, min(args.warmup, 1))):
        one_pass()
    sampler = ClockSampler(0)
    sampler.start()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        one_pass()
    wall = (time.perf_counter() - t0) / args.steps
    clocks = sampler.stop()
    units = nbeams * blk.ndm * (first.nout + (nblk - 1) * B)
    span = B * nblk * a["dt"]
    line = {"metric": METRIC, "value": units / wall / 1e9, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": 1, "ms_per_step": wall * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": {"workload": f"stream19: {nbeams} beams x {nblk} blocks of {B} samples, {nchan} ch uint8, "
                                   f"{blk.ndm} DMs, halo {H} rows carried; {ndistinct} distinct beams in pinned "
                                   f"host memory, cycled", "parallelism": "one GPU, beams in sequence"},
            "realtime_factor": span / wall,
            "input_rate_GBps": nbeams * B * nblk * nchan / wall / 1e9,
            "realtime_input_rate_GBps": nbeams * nchan / a["dt"] / 1e9,
            "clocks": clocks,
            "e2e": {"value": units / wall / 1e9, "unit": UNIT, "h2d_bytes_per_step": nbeams * nblk * B * nchan,
                    "d2h_bytes_per_step": nbeams * nblk * blk.ndm * 4},
            "gpu_launches": nbeams * nblk * 2 * args.steps}
    print(json.dumps(line))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def spawn_ranks(args):
    """`python bench.py --gpus N` started WITHOUT torchrun: launch the N ranks ourselves, one per GPU, the way
    the driver does (torch.distributed.run, 127.0.0.1 rendezvous), and relay rank 0's JSON line."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), os.path.abspath(__file__)] + sys.argv[1:]
    r = subprocess.run(cmd)
    raise SystemExit(r.returncode)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="gsp", choices=["gsp", "reference"])
    ap.add_argument("--config", default="crafts")
    ap.add_argument("--plan", type=int, default=None, help="one plan (DM range) of a multi-plan config such as ddplan")
    ap.add_argument("--shard", default="none", choices=["none", "dm"],
                    help="dm: ONE beam broadcast from rank 0, the DM list sharded over the ranks (strong scaling)")
    ap.add_argument("--nsamp", type=int, default=0, help="override the workload length (debugging)")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-search", action="store_true")
    ap.add_argument("--no-rfi", action="store_true", help="skip the RFI-prologue timing reported beside the headline")
    ap.add_argument("--beams", type=int, default=0, help="stream19: number of beams (default 19)")
    ap.add_argument("--host-beams", type=int, default=4, help="stream19: distinct beams kept in pinned memory")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "gsp" else args.warmup
    if args.impl == "reference":
        run_reference(args)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.config != "stream19":
        spawn_ranks(args)
    if args.config == "stream19":
        run_stream19(args)
    elif args.plan is None and len(workloads.get_config(args.config)["plans"]) > 1:
        run_multi(args)
    else:
        run_gsp(args)


if __name__ == "__main__":
    main()
