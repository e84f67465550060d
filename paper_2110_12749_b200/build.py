"""Build libgsp.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libgsp.so")
SOURCES = ["gsp_tables.cpp", "gsp_kernels.cu", "gsp_stage1.cu", "gsp_stage1_ring.cu", "gsp_stage1_f32.cu", "gsp_stage1_wide.cu", "gsp_api.cu", "gsp_host.cu", "gsp_search.cu", "gsp_rfi.cu", "gsp_static.cu"]
HEADERS = [os.path.join(CSRC, "gsp_internal.h"), os.path.join(CSRC, "gsp_device.cuh"), os.path.join(ROOT, "include", "gsp.h")]

NVCC_FLAGS = [
    "-std=c++17", "-O3", "-lineinfo",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-Xcompiler", "-fPIC",
    "-I", os.path.join(ROOT, "include"), "-I", CSRC,
]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps if os.path.exists(d))


def build(force=False, verbose=False, extra=()):
    """Compile every CUDA source of the package into paper_2110_12749_b200/libgsp.so
    (one nvcc per translation unit, in parallel, objects under build/; then one link)."""
    if not force and not needs_build():
        return LIB
    from concurrent.futures import ThreadPoolExecutor
    objdir = os.path.join(PKG, "build")
    os.makedirs(objdir, exist_ok=True)
    hdr_t = max(os.path.getmtime(h) for h in HEADERS + [os.path.abspath(__file__)])
    jobs = []
    for s in SOURCES:
        src = os.path.join(CSRC, s)
        obj = os.path.join(objdir, os.path.splitext(s)[0] + ".o")
        jobs.append((src, obj))

    def compile_one(job):
        src, obj = job
        if (not force and os.path.exists(obj) and os.path.getmtime(obj) > os.path.getmtime(src)
                and os.path.getmtime(obj) > hdr_t):
            return
        cmd = [_nvcc(), *NVCC_FLAGS, *extra, "-x", "cu", "-c", "-o", obj, src]
        if verbose:
            cmd[1:1] = ["-Xptxas", "-v"]
            print(" ".join(cmd))
        subprocess.run(cmd, check=True)

    with ThreadPoolExecutor(max_workers=min(8, len(jobs))) as ex:
        list(ex.map(compile_one, jobs))
    subprocess.run([_nvcc(), "-arch=sm_100a", "-shared", "-o", LIB, *[o for _, o in jobs]], check=True)
    return LIB


def build_microbench():
    """Compile the roofline microbenchmark (microbench/gsp_peaks.cu) into paper_2110_12749_b200/gsp_peaks."""
    src = os.path.join(PKG, "microbench", "gsp_peaks.cu")
    exe = os.path.join(PKG, "gsp_peaks")
    if not os.path.exists(exe) or os.path.getmtime(exe) < os.path.getmtime(src):
        subprocess.run([_nvcc(), "-std=c++17", "-O3", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a",
                        "-o", exe, src], check=True)
    return exe


if __name__ == "__main__":
    build(force=True, verbose="-v" in sys.argv)
    build_microbench()
    print(LIB)
