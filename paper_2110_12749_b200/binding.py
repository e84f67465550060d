"""ctypes binding of libgsp.so — same entry points as include/gsp.h, marshalling only."""
from __future__ import annotations

import ctypes
import os
import re

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_PKG)
_LIB_PATH = os.path.join(_PKG, "libgsp.so")
_HEADER = os.path.join(_ROOT, "include", "gsp.h")

GSP_U8, GSP_F32 = 0, 1
GSP_IMPL_AUTO, GSP_IMPL_GENERIC, GSP_IMPL_TILED, GSP_IMPL_WINDOWED = 0, 1, 2, 3
_STATUS = {0: "GSP_OK", 1: "GSP_ERR_INVALID_ARG", 2: "GSP_ERR_TOO_SHORT", 3: "GSP_ERR_ALLOC",
           4: "GSP_ERR_CUDA", 5: "GSP_ERR_TOO_LARGE"}


class GspError(RuntimeError):
    def __init__(self, status, where):
        self.status = int(status)
        super().__init__(f"{where}: {_STATUS.get(int(status), status)}")


def library_path() -> str:
    return _LIB_PATH


def declared_symbols(header: str = _HEADER):
    """Names of every function include/gsp.h declares (used by the ABI test)."""
    text = open(header).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gsp_[a-z0-9_]+)\s*\(", text)))


_lib = None


def lib():
    """Load libgsp.so (built in-tree by paper_2110_12749_b200.build); fail loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise GspError(4, f"libgsp.so not built ({_LIB_PATH}); run __graft_entry__.build()")
    L = ctypes.CDLL(_LIB_PATH)
    c = ctypes
    vp, i32, i64, dbl = c.c_void_p, c.c_int32, c.c_int64, c.c_double
    L.gsp_plan_create.argtypes = [c.POINTER(vp), c.c_int, dbl, dbl, dbl, i64, c.c_int, dbl,
                                  c.POINTER(dbl), c.c_int, c.c_int, c.c_int]
    L.gsp_plan_create.restype = c.c_int
    L.gsp_dedisperse.argtypes = [vp, vp, vp, vp]
    L.gsp_dedisperse.restype = c.c_int
    L.gsp_dedisperse_host.argtypes = [vp, vp, vp, i64, vp]
    L.gsp_dedisperse_host.restype = c.c_int
    L.gsp_dedisperse_host_in.argtypes = [vp, vp, vp, i64, vp]
    L.gsp_dedisperse_host_in.restype = c.c_int
    L.gsp_plan_destroy.argtypes = [vp]
    L.gsp_plan_destroy.restype = c.c_int
    for name in ("gsp_plan_nout", "gsp_plan_out_pitch", "gsp_plan_halo", "gsp_plan_n1",
                 "gsp_plan_n1d", "gsp_plan_workspace_bytes"):
        getattr(L, name).argtypes = [vp]
        getattr(L, name).restype = i64
    for name in ("gsp_plan_h1", "gsp_plan_h2", "gsp_plan_ndm", "gsp_plan_launches_per_call"):
        getattr(L, name).argtypes = [vp]
        getattr(L, name).restype = i32
    for name in ("gsp_plan_stage1_shifts", "gsp_plan_stage2_shifts"):
        getattr(L, name).argtypes = [vp]
        getattr(L, name).restype = c.POINTER(i32)
    L.gsp_plan_set_impl.argtypes = [vp, c.c_int, c.c_int]
    L.gsp_plan_set_impl.restype = c.c_int
    L.gsp_plan_get_impl.argtypes = [vp, c.c_int]
    L.gsp_plan_get_impl.restype = i32
    L.gsp_plan_enable_stage_timing.argtypes = [vp, c.c_int]
    L.gsp_plan_enable_stage_timing.restype = c.c_int
    L.gsp_plan_last_stage_ms.argtypes = [vp, c.POINTER(c.c_float), c.POINTER(c.c_float)]
    L.gsp_plan_last_stage_ms.restype = c.c_int
    L.gsp_plan_stage_ms_total.argtypes = [vp, c.POINTER(dbl), c.POINTER(dbl), c.POINTER(i32)]
    L.gsp_plan_stage_ms_total.restype = c.c_int
    L.gsp_dedisperse_multi.argtypes = [c.POINTER(vp), c.c_int, vp, c.POINTER(vp), vp]
    L.gsp_dedisperse_multi.restype = c.c_int
    L.gsp_plan_reserve_multi.argtypes = [vp]
    L.gsp_plan_reserve_multi.restype = c.c_int
    L.gsp_dedisperse_multi_launches.argtypes = [c.POINTER(vp), c.c_int]
    L.gsp_dedisperse_multi_launches.restype = i32
    L.gsp_plan_stage1_split.argtypes = [vp, c.POINTER(i32)]
    L.gsp_plan_stage1_split.restype = c.c_int
    L.gsp_plan_stage1_split_n.argtypes = [vp, c.POINTER(i32), i32, c.POINTER(i32)]
    L.gsp_plan_stage1_split_n.restype = c.c_int
    L.gsp_delay_tables.argtypes = [c.c_int, dbl, dbl, dbl, c.c_int, dbl, c.POINTER(dbl), c.c_int,
                                   c.c_int, c.POINTER(i32), c.POINTER(i32)]
    L.gsp_delay_tables.restype = c.c_int
    L.gsp_plan_set_rfi.argtypes = [vp, vp, vp, dbl, i32]
    L.gsp_plan_set_rfi.restype = c.c_int
    L.gsp_plan_rfi_last.argtypes = [vp, vp, vp]
    L.gsp_plan_rfi_last.restype = c.c_int
    L.gsp_search_create.argtypes = [c.POINTER(vp), c.c_int, i64, i64, c.c_int, c.c_int, c.c_float, i64]
    L.gsp_search_create.restype = c.c_int
    L.gsp_search_run.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp]
    L.gsp_search_run.restype = c.c_int
    L.gsp_search_nblocks.argtypes = [vp]
    L.gsp_search_nblocks.restype = i64
    L.gsp_search_destroy.argtypes = [vp]
    L.gsp_search_destroy.restype = c.c_int
    L.gsp_dedisperse_static.argtypes = [vp, c.c_int, i64, c.c_int, c.c_int, c.c_int, c.c_int, vp, vp, i32, i32,
                                        vp, i64, vp]
    L.gsp_dedisperse_static.restype = c.c_int
    L.gsp_static_workspace_bytes.argtypes = []
    L.gsp_static_workspace_bytes.restype = i64
    L.gsp_status_string.argtypes = [c.c_int]
    L.gsp_status_string.restype = c.c_char_p
    L.gsp_version.argtypes = []
    L.gsp_version.restype = c.c_char_p
    _lib = L
    return L


def _check(status, where):
    if status != 0:
        raise GspError(status, where)


def _dev_ptr(t):
    """Device (or host) address of a torch tensor / numpy array / int."""
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    return t.ctypes.data


def delay_tables(nchan, f_top, chan_bw, dt, nsub, subband_dm, dm_list, downsamp=1):
    """gsp_delay_tables: the library's own table builder, host only -> (s1, s2)."""
    dms = np.ascontiguousarray(dm_list, dtype=np.float64)
    s1 = np.empty(max(int(nchan), 1), dtype=np.int32)
    s2 = np.empty((max(int(dms.size), 1), max(int(nsub), 1)), dtype=np.int32)
    st = lib().gsp_delay_tables(int(nchan), float(f_top), float(chan_bw), float(dt), int(nsub),
                                float(subband_dm),
                                dms.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), int(dms.size),
                                int(downsamp), s1.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)),
                                s2.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)))
    _check(st, "gsp_delay_tables")
    return s1, s2


def static_workspace_bytes():
    """gsp_static_workspace_bytes: size of the fixed subband workspace gsp_dedisperse_static works in."""
    return int(lib().gsp_static_workspace_bytes())


def dedisperse_static(d_in, dtype, nsamp, nchan, nsub, ndm, downsamp, d_s1, d_s2, h1, h2, d_out, out_pitch,
                      stream=0):
    """gsp_dedisperse_static: the plan-free call for callers that cannot allocate device memory (no
    cudaMalloc anywhere inside; the subband intermediate sits in a 16 MiB array of the library image).
    Every pointer is a CUDA tensor (or raw device address) the caller owns; h1 / h2 are the host maxima of
    the two shift tables.  Raises GspError(GSP_ERR_TOO_LARGE) when nsub * n1d * 4 bytes exceed the array."""
    dt = {"u8": GSP_U8, "f32": GSP_F32, GSP_U8: GSP_U8, GSP_F32: GSP_F32}[dtype]
    _check(lib().gsp_dedisperse_static(_dev_ptr(d_in), dt, int(nsamp), int(nchan), int(nsub), int(ndm),
                                       int(downsamp), _dev_ptr(d_s1), _dev_ptr(d_s2), int(h1), int(h2),
                                       _dev_ptr(d_out), int(out_pitch), int(stream)), "gsp_dedisperse_static")


def dedisperse_multi_launches(plans):
    """gsp_dedisperse_multi_launches: kernels one dedisperse_multi call launches for these plans."""
    n = len(plans)
    hp = (ctypes.c_void_p * n)(*[p._h for p in plans])
    return int(lib().gsp_dedisperse_multi_launches(hp, n))


def dedisperse_multi(plans, d_in, d_outs, stream=0):
    """gsp_dedisperse_multi: every plan of `plans` over the same input `d_in`, d_outs[i] = output of plans[i]."""
    n = len(plans)
    hp = (ctypes.c_void_p * n)(*[p._h for p in plans])
    op = (ctypes.c_void_p * n)(*[_dev_ptr(o) for o in d_outs])
    _check(lib().gsp_dedisperse_multi(hp, n, _dev_ptr(d_in), op, int(stream)), "gsp_dedisperse_multi")


class Plan:
    """gsp_plan_create / gsp_dedisperse / gsp_plan_destroy with tensors instead of pointers."""

    def __init__(self, nchan, f_top, chan_bw, dt, nsamp, nsub, subband_dm, dm_list, downsamp=1,
                 dtype="u8"):
        L = lib()
        dms = np.ascontiguousarray(dm_list, dtype=np.float64)
        self._dtype = {"u8": GSP_U8, "f32": GSP_F32, GSP_U8: GSP_U8, GSP_F32: GSP_F32}[dtype]
        self._h = ctypes.c_void_p()
        st = L.gsp_plan_create(ctypes.byref(self._h), int(nchan), float(f_top), float(chan_bw),
                               float(dt), int(nsamp), int(nsub), float(subband_dm),
                               dms.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), int(dms.size),
                               int(downsamp), self._dtype)
        _check(st, "gsp_plan_create")
        self.nchan, self.nsub, self.nsamp, self.downsamp = int(nchan), int(nsub), int(nsamp), int(downsamp)
        self.ndm = int(L.gsp_plan_ndm(self._h))
        self.nout = int(L.gsp_plan_nout(self._h))
        self.out_pitch = int(L.gsp_plan_out_pitch(self._h))
        self.halo = int(L.gsp_plan_halo(self._h))
        self.n1 = int(L.gsp_plan_n1(self._h))
        self.n1d = int(L.gsp_plan_n1d(self._h))
        self.H1 = int(L.gsp_plan_h1(self._h))
        self.H2 = int(L.gsp_plan_h2(self._h))

    # -- tables ---------------------------------------------------------------
    @property
    def stage1_shifts(self):
        p = lib().gsp_plan_stage1_shifts(self._h)
        return np.ctypeslib.as_array(p, shape=(self.nchan,)).copy()

    @property
    def stage2_shifts(self):
        p = lib().gsp_plan_stage2_shifts(self._h)
        return np.ctypeslib.as_array(p, shape=(self.ndm, self.nsub)).copy()

    @property
    def workspace_bytes(self):
        return int(lib().gsp_plan_workspace_bytes(self._h))

    @property
    def launches_per_call(self):
        return int(lib().gsp_plan_launches_per_call(self._h))

    # -- implementation control ----------------------------------------------
    @property
    def stage1_split(self):
        """(ring groups, wide subbands 2 CTA/SM, wide subbands 1 CTA/SM, windowed groups, float32 streams,
        long-ring subbands 2 CTA/SM, long-ring subbands 1 CTA/SM)."""
        n = ctypes.c_int32(0)
        buf = (ctypes.c_int32 * 16)()
        _check(lib().gsp_plan_stage1_split_n(self._h, buf, 16, ctypes.byref(n)), "gsp_plan_stage1_split_n")
        return tuple(int(v) for v in buf[: n.value])

    def set_impl(self, stage, impl):
        _check(lib().gsp_plan_set_impl(self._h, int(stage), int(impl)), "gsp_plan_set_impl")

    def get_impl(self, stage):
        return int(lib().gsp_plan_get_impl(self._h, int(stage)))

    def enable_stage_timing(self, on=True):
        _check(lib().gsp_plan_enable_stage_timing(self._h, int(bool(on))), "gsp_plan_enable_stage_timing")

    def last_stage_ms(self):
        a, b = ctypes.c_float(), ctypes.c_float()
        _check(lib().gsp_plan_last_stage_ms(self._h, ctypes.byref(a), ctypes.byref(b)),
               "gsp_plan_last_stage_ms")
        return a.value, b.value

    def stage_ms_total(self):
        """(total stage-1 ms, total stage-2 ms, calls) since timing was enabled."""
        a, b, n = ctypes.c_double(), ctypes.c_double(), ctypes.c_int32()
        _check(lib().gsp_plan_stage_ms_total(self._h, ctypes.byref(a), ctypes.byref(b),
                                             ctypes.byref(n)), "gsp_plan_stage_ms_total")
        return a.value, b.value, n.value

    def reserve_multi(self):
        """gsp_plan_reserve_multi: allocate the shared-ring scratch of dedisperse_multi now (float32 plans)."""
        _check(lib().gsp_plan_reserve_multi(self._h), "gsp_plan_reserve_multi")

    # -- RFI prologue -----------------------------------------------------------
    def set_rfi(self, chan_mask, chan_pad, clip_sigma=0.0, clip_block=0):
        """gsp_plan_set_rfi: host arrays chan_mask[nchan] (or None) and chan_pad[nchan] (None clears)."""
        if chan_pad is None:
            _check(lib().gsp_plan_set_rfi(self._h, None, None, 0.0, 0), "gsp_plan_set_rfi")
            return
        pad = np.ascontiguousarray(chan_pad, dtype=np.uint8)
        mask = None if chan_mask is None else np.ascontiguousarray(chan_mask, dtype=np.uint8)
        _check(lib().gsp_plan_set_rfi(self._h, None if mask is None else mask.ctypes.data, pad.ctypes.data,
                                      float(clip_sigma), int(clip_block)), "gsp_plan_set_rfi")

    def rfi_last(self):
        """(zero-DM series, clip flags) of the last call of a clipping plan."""
        z = np.empty(self.nsamp, dtype=np.int64)
        cl = np.empty(self.nsamp, dtype=np.uint8)
        _check(lib().gsp_plan_rfi_last(self._h, z.ctypes.data, cl.ctypes.data), "gsp_plan_rfi_last")
        return z, cl

    # -- execution ------------------------------------------------------------
    def dedisperse(self, d_in, d_out, stream=0):
        """Enqueue on `stream` (a cudaStream_t handle as int, 0 = default).  d_in/d_out are
        CUDA tensors (or raw device addresses): x[nsamp][nchan], y[ndm][out_pitch] float32."""
        _check(lib().gsp_dedisperse(self._h, _dev_ptr(d_in), _dev_ptr(d_out), int(stream)),
               "gsp_dedisperse")

    def dedisperse_host(self, h_in, h_out, h_out_pitch=None, stream=0):
        """Host buffers in, host buffers out (H2D / kernels / D2H pipelined inside the library)."""
        if h_out_pitch is None:
            h_out_pitch = h_out.shape[-1]
        _check(lib().gsp_dedisperse_host(self._h, _dev_ptr(h_in), _dev_ptr(h_out), int(h_out_pitch),
                                         int(stream)), "gsp_dedisperse_host")

    def dedisperse_host_in(self, h_in, d_out, d_out_pitch=None, stream=0):
        """Host input, DEVICE output (gsp_dedisperse_host_in): only the input crosses PCIe."""
        if d_out_pitch is None:
            d_out_pitch = d_out.shape[-1]
        _check(lib().gsp_dedisperse_host_in(self._h, _dev_ptr(h_in), _dev_ptr(d_out), int(d_out_pitch),
                                            int(stream)), "gsp_dedisperse_host_in")

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h:
            lib().gsp_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()


class Search:
    """gsp_search_create / gsp_search_run / gsp_search_destroy: single-pulse search on d_out (marshalling only)."""

    def __init__(self, ndm, nout, pitch, block=1024, nwidths=6, threshold=6.0, max_cand=0):
        self._h = ctypes.c_void_p()
        st = lib().gsp_search_create(ctypes.byref(self._h), int(ndm), int(nout), int(pitch), int(block),
                                     int(nwidths), float(threshold), int(max_cand))
        _check(st, "gsp_search_create")
        self.ndm, self.nout, self.pitch, self.block = int(ndm), int(nout), int(pitch), int(block)
        self.max_cand = int(max_cand)
        self.nblocks = int(lib().gsp_search_nblocks(self._h))

    def run(self, d_y, d_dm, d_sample, d_width, d_snr, d_count, d_stats=None, stream=0):
        """Enqueue on `stream`; every argument is a CUDA tensor (or raw device address) owned by the caller."""
        p = lambda t: None if t is None else _dev_ptr(t)
        _check(lib().gsp_search_run(self._h, _dev_ptr(d_y), p(d_dm), p(d_sample), p(d_width), p(d_snr),
                                    _dev_ptr(d_count), p(d_stats), int(stream)), "gsp_search_run")

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h:
            lib().gsp_search_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()
