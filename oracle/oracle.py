"""ctypes front-end of ``gsp_oracle.cpp`` (plain C++17 CPU oracle; test infrastructure).

Every function here only marshals numpy arrays into the C++ routines; the
arithmetic lives in ``gsp_oracle.cpp`` where each step cites the passage of
PAPER.md / BASELINE.json / DESIGN.md reading that it follows.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gsp_oracle.cpp")
_LIB = os.path.join(_HERE, "libgsp_oracle.so")
_SRC_X = os.path.join(_HERE, "gsp_extras_oracle.cpp")
_LIB_X = os.path.join(_HERE, "libgsp_extras_oracle.so")
_lib = None
_libx = None


def build_oracle(force: bool = False) -> str:
    """Compile the oracle with the host C++ compiler (no CUDA involved)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-shared", "-fPIC", _SRC, "-o", _LIB]
        subprocess.run(cmd, check=True)
    if force or not os.path.exists(_LIB_X) or os.path.getmtime(_LIB_X) < os.path.getmtime(_SRC_X):
        # RFI prologue + single-pulse search: every float decision in a stated order, no fused multiply-add
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-shared", "-fPIC", _SRC_X, "-o", _LIB_X]
        subprocess.run(cmd, check=True)
    return _LIB


def _loadx():
    global _libx
    if _libx is None:
        build_oracle()
        lib = ctypes.CDLL(_LIB_X)
        c = ctypes
        lib.gsp_oracle_rfi_prologue.argtypes = [c.c_void_p, c.c_longlong, c.c_int, c.c_void_p, c.c_void_p,
                                                c.c_double, c.c_int, c.c_void_p, c.c_void_p, c.c_void_p]
        lib.gsp_oracle_rfi_prologue.restype = c.c_int
        lib.gsp_oracle_search.argtypes = [c.c_void_p, c.c_int, c.c_longlong, c.c_longlong, c.c_int, c.c_int,
                                          c.c_float, c.c_longlong, c.c_void_p, c.c_void_p, c.c_void_p,
                                          c.c_void_p, c.c_void_p]
        lib.gsp_oracle_search.restype = c.c_longlong
        _libx = lib
    return _libx


def _load():
    global _lib
    if _lib is None:
        build_oracle()
        lib = ctypes.CDLL(_LIB)
        i32p = ctypes.POINTER(ctypes.c_int32)
        i64p = ctypes.POINTER(ctypes.c_longlong)
        f32p = ctypes.POINTER(ctypes.c_float)
        f64p = ctypes.POINTER(ctypes.c_double)
        lib.gsp_oracle_tables.argtypes = [ctypes.c_int, ctypes.c_double, ctypes.c_double,
                                          ctypes.c_double, ctypes.c_int, ctypes.c_double, f64p,
                                          ctypes.c_int, ctypes.c_int, i32p, i32p]
        for name in ("gsp_oracle_dedisperse_u8", "gsp_oracle_dedisperse_f32"):
            getattr(lib, name).argtypes = [ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int,
                                           ctypes.c_int, i32p, i32p, ctypes.c_int, ctypes.c_int,
                                           f32p, ctypes.c_longlong, ctypes.c_int]
        for name in ("gsp_oracle_points_u8", "gsp_oracle_points_f32"):
            getattr(lib, name).argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, i32p, i32p,
                                           ctypes.c_int, i32p, i64p, ctypes.c_longlong, f32p]
        _lib = lib
    return _lib


def _ptr(a, ctype):
    return a.ctypes.data_as(ctypes.POINTER(ctype))


def max_threads() -> int:
    return int(_load().gsp_oracle_max_threads())


def delay_tables(nchan, f_top, chan_bw, dt, nsub, subband_dm, dm_list, downsamp):
    """(s1[nchan], s2[ndm][nsub]) int32 — O1-O3, rule R3 (gsp_oracle_tables)."""
    dm = np.ascontiguousarray(dm_list, dtype=np.float64)
    s1 = np.empty(nchan, dtype=np.int32)
    s2 = np.empty((dm.size, nsub), dtype=np.int32)
    rc = _load().gsp_oracle_tables(nchan, f_top, chan_bw, dt, nsub, subband_dm,
                                   _ptr(dm, ctypes.c_double), dm.size, downsamp,
                                   _ptr(s1, ctypes.c_int32), _ptr(s2, ctypes.c_int32))
    if rc:
        raise ValueError(f"gsp_oracle_tables rc={rc}")
    return s1, s2


def geometry(nsamp, s1, s2, downsamp):
    """H1, H2, n1, n1d, nout (O4-O6 extents)."""
    H1 = int(s1.max())
    H2 = int(s2.max())
    n1 = nsamp - H1
    n1d = n1 // downsamp
    return dict(H1=H1, H2=H2, n1=n1, n1d=n1d, nout=n1d - H2)


def dedisperse(x, s1, s2, downsamp, nthreads=1):
    """Full two-stage result y[ndm][nout] float32 for x[nsamp][nchan] (uint8 or float32)."""
    x = np.ascontiguousarray(x)
    nsamp, nchan = x.shape
    ndm, nsub = s2.shape
    g = geometry(nsamp, s1, s2, downsamp)
    if g["nout"] <= 0:
        raise ValueError("input too short for the delay tables")
    y = np.empty((ndm, g["nout"]), dtype=np.float32)
    fn = {np.dtype(np.uint8): _load().gsp_oracle_dedisperse_u8,
          np.dtype(np.float32): _load().gsp_oracle_dedisperse_f32}[x.dtype]
    s1c = np.ascontiguousarray(s1, dtype=np.int32)
    s2c = np.ascontiguousarray(s2, dtype=np.int32)
    rc = fn(x.ctypes.data, nsamp, nchan, nsub, _ptr(s1c, ctypes.c_int32),
            _ptr(s2c, ctypes.c_int32), ndm, downsamp, _ptr(y, ctypes.c_float), g["nout"],
            int(nthreads))
    if rc:
        raise ValueError(f"gsp_oracle_dedisperse rc={rc}")
    return y


def points(x, s1, s2, downsamp, d_idx, u_idx):
    """y_d[u] for listed (d, u) pairs, each straight from the definition."""
    x = np.ascontiguousarray(x)
    _, nchan = x.shape
    _, nsub = s2.shape
    d = np.ascontiguousarray(d_idx, dtype=np.int32)
    u = np.ascontiguousarray(u_idx, dtype=np.int64)
    out = np.empty(d.size, dtype=np.float32)
    fn = {np.dtype(np.uint8): _load().gsp_oracle_points_u8,
          np.dtype(np.float32): _load().gsp_oracle_points_f32}[x.dtype]
    s1c = np.ascontiguousarray(s1, dtype=np.int32)
    s2c = np.ascontiguousarray(s2, dtype=np.int32)
    fn(x.ctypes.data, nchan, nsub, _ptr(s1c, ctypes.c_int32), _ptr(s2c, ctypes.c_int32),
       downsamp, _ptr(d, ctypes.c_int32), _ptr(u, ctypes.c_longlong), d.size,
       _ptr(out, ctypes.c_float))
    return out


def rfi_prologue(x, chan_mask, chan_pad, clip_sigma=0.0, clip_block=0):
    """RFI prologue F1-F4 (gsp_extras_oracle.cpp) on a uint8 filterbank x[nsamp][nchan].
    Returns (x2, z, clipped): the cleaned filterbank, the zero-DM series (after the channel mask)
    and the per-row clip flags."""
    x = np.ascontiguousarray(x, dtype=np.uint8)
    nsamp, nchan = x.shape
    pad = np.ascontiguousarray(chan_pad, dtype=np.uint8)
    assert pad.shape == (nchan,)
    mask = None if chan_mask is None else np.ascontiguousarray(chan_mask, dtype=np.uint8)
    x2 = np.empty_like(x)
    z = np.empty(nsamp, dtype=np.int64)
    clipped = np.empty(nsamp, dtype=np.uint8)
    rc = _loadx().gsp_oracle_rfi_prologue(x.ctypes.data, nsamp, nchan,
                                          None if mask is None else mask.ctypes.data, pad.ctypes.data,
                                          float(clip_sigma), int(clip_block), x2.ctypes.data,
                                          z.ctypes.data, clipped.ctypes.data)
    if rc:
        raise ValueError(f"gsp_oracle_rfi_prologue rc={rc}")
    return x2, z, clipped


def search(y, nout=None, block=1024, nwidths=6, threshold=6.0, max_cand=None, return_stats=False):
    """Single-pulse search S1-S6 (gsp_extras_oracle.cpp) on y[ndm][pitch] float32 (nout valid samples
    per row).  Returns a dict of arrays dm, sample, width, snr (candidates in (DM, block) order) and the
    total count; with return_stats also stats[ndm][nblk][2] = (mu_f, r_f)."""
    y = np.ascontiguousarray(y, dtype=np.float32)
    ndm, pitch = y.shape
    nout = pitch if nout is None else int(nout)
    nblk = (nout + block - 1) // block
    cap = ndm * nblk if max_cand is None else int(max_cand)
    dm = np.empty(cap, dtype=np.int32)
    u = np.empty(cap, dtype=np.int32)
    w = np.empty(cap, dtype=np.int32)
    snr = np.empty(cap, dtype=np.float32)
    stats = np.empty((ndm, nblk, 2), dtype=np.float32) if return_stats else None
    n = _loadx().gsp_oracle_search(y.ctypes.data, ndm, nout, pitch, int(block), int(nwidths),
                                   float(threshold), cap, dm.ctypes.data, u.ctypes.data, w.ctypes.data,
                                   snr.ctypes.data, None if stats is None else stats.ctypes.data)
    if n < 0:
        raise ValueError("gsp_oracle_search: bad arguments")
    k = min(int(n), cap)
    out = dict(count=int(n), dm=dm[:k], sample=u[:k], width=w[:k], snr=snr[:k])
    if return_stats:
        out["stats"] = stats
    return out
