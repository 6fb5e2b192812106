"""Build libef.so (the product) and, on request, libef_diag.so (the diagnostic build) in-tree with nvcc for sm_100a
(cross-compiles without a GPU).

    python -m paper_2410_17954_b200.build [--force] [--verbose] [--diag]

libef.so      : csrc/{ef_api,ffn_tc,route,permute,combine,token_sched}.cu -- everything include/ef.h declares.
libef_diag.so : the same sources compiled with -DEF_DIAG, plus csrc/{ffn_simt,diag,diag_api}.cu -- additionally exports
                include/ef_diag.h (plain-FMA FFN backend for bring-up, TMA fill-rate probe, per-CTA wait-cycle counters
                with EF_KPROF=1 in the environment).  Tests and bench.py opt into it; the product never loads it.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libef.so")
LIB_DIAG = os.path.join(PKG, "libef_diag.so")

PRODUCT_SRCS = ["ef_api.cu", "ffn_tc.cu", "route.cu", "permute.cu", "combine.cu", "token_sched.cu"]
DIAG_ONLY_SRCS = ["ffn_simt.cu", "diag.cu", "diag_api.cu"]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-I", os.path.join(ROOT, "include"), "-I", CSRC]


def _newer(src_list, target):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in src_list)


def _build(lib, srcs, obj_dir, flags, force, verbose):
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(obj_dir, exist_ok=True)
    srcs = [os.path.join(CSRC, s) for s in srcs]
    hdrs = [os.path.join(CSRC, "ef_internal.h"), os.path.join(ROOT, "include", "ef.h"), os.path.join(ROOT, "include", "ef_diag.h")]
    jobs = []
    for s in srcs:
        o = os.path.join(obj_dir, os.path.basename(s)[:-3] + ".o")
        if force or _newer([s] + hdrs, o):
            extra = ["-Xptxas", "-v"] if verbose else []
            jobs.append(([nvcc] + flags + extra + ["-c", s, "-o", o], s))

    def run(job):
        cmd, s = job
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {s}:\n{r.stdout}\n{r.stderr}")
        if verbose:
            sys.stderr.write(r.stderr)
        return s

    if jobs:
        with ThreadPoolExecutor(max_workers=min(8, len(jobs))) as ex:
            list(ex.map(run, jobs))
    objs = [os.path.join(obj_dir, os.path.basename(s)[:-3] + ".o") for s in srcs]
    if force or jobs or _newer(objs, lib):
        cmd = [nvcc, "-shared", "-o", lib] + objs + ["-gencode", "arch=compute_100a,code=sm_100a", "-cudart", "static"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    return lib


def build(force: bool = False, verbose: bool = False) -> str:
    """The product library."""
    flags = NVCC_FLAGS + os.environ.get("EF_NVCC_EXTRA", "").split()      # e.g. an A/B macro for an experiment
    return _build(LIB, PRODUCT_SRCS, os.path.join(PKG, "build"), flags, force, verbose)


def build_diag(force: bool = False, verbose: bool = False) -> str:
    """The diagnostic library (never loaded by the product path)."""
    flags = NVCC_FLAGS + ["-DEF_DIAG"] + (["-DEF_KPROF"] if os.environ.get("EF_KPROF") else [])
    flags += os.environ.get("EF_NVCC_EXTRA", "").split()
    return _build(LIB_DIAG, PRODUCT_SRCS + DIAG_ONLY_SRCS, os.path.join(PKG, "build_diag"), flags, force, verbose)


if __name__ == "__main__":
    force, verbose = "--force" in sys.argv, "--verbose" in sys.argv
    print(build(force, verbose))
    if "--diag" in sys.argv:
        print(build_diag(force, verbose))
