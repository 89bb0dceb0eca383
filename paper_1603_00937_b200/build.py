"""Builds csrc/*.cu into paper_1603_00937_b200/libgbe.so for sm_100a (in-tree; the .so is git-ignored).

    python -m paper_1603_00937_b200.build [--force] [--verbose]
    python -m paper_1603_00937_b200.build --stamps     the instrumented copy libgbe_stamps.so (-DGBE_STAMPS: %globaltimer
                                                       stamps in k_sp2_packed and k_x2_tma; read by bench.py --timeline).
                                                       libgbe.so holds none of it.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libgbe.so")
LIB_STAMPS = os.path.join(HERE, "libgbe_stamps.so")
SOURCES = sorted(glob.glob(os.path.join(HERE, "csrc", "*.cu")))
HEADERS = sorted(glob.glob(os.path.join(HERE, "csrc", "*.cuh"))) + [os.path.join(ROOT, "include", "gbe.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC,-O3,-Wall", "-Xptxas", "-v" if os.environ.get("GBE_PTXAS_V") else "-warn-spills",
    "-cudart", "static",
]


def _stale(obj: str, src: str) -> bool:
    if not os.path.exists(obj):
        return True
    t = os.path.getmtime(obj)
    return any(os.path.getmtime(f) > t for f in [src] + HEADERS + [os.path.abspath(__file__)])


def build(force: bool = False, verbose: bool = False, stamps: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "nvcc")
    objdir = os.path.join(HERE, "build", "stamps") if stamps else os.path.join(HERE, "build")
    lib = LIB_STAMPS if stamps else LIB
    extra = ["-DGBE_STAMPS"] if stamps else []
    # (the stamps cost k_sp2_packed a few spilled registers at its 64-register cap: expected there, not warned about)
    flags = [f for f in NVCC_FLAGS if not (stamps and f == "-warn-spills")]
    if stamps and "-warn-spills" in NVCC_FLAGS:
        flags.remove("-Xptxas")
    os.makedirs(objdir, exist_ok=True)
    objs, procs = [], []
    for src in SOURCES:
        obj = os.path.join(objdir, os.path.basename(src)[:-3] + ".o")
        objs.append(obj)
        if force or _stale(obj, src):
            cmd = [nvcc, *flags, *extra, "-I", os.path.join(ROOT, "include"), "-I", os.path.join(HERE, "csrc"), "-c", src, "-o", obj]
            if verbose:
                print(" ".join(cmd))
            procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    failed = False
    for src, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0 or verbose or "warning" in out.lower():
            sys.stderr.write(out)
        failed |= p.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed")
    if procs or not os.path.exists(lib) or force:
        cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-cudart", "static", "-o", lib, *objs]
        if verbose:
            print(" ".join(cmd))
        subprocess.check_call(cmd)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, stamps="--stamps" in sys.argv))
