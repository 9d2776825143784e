"""Builds libanm.so (the CUDA path) in-tree with nvcc for sm_100a.  `python -m paper_2111_11687_b200.build`"""
from __future__ import annotations

import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libanm.so")
SOURCES = [os.path.join(CSRC, "anm_api.cu"), os.path.join(CSRC, "anm_static.cu")]
DEPENDS = SOURCES + [os.path.join(CSRC, "anm_kernels.cuh"), os.path.join(CSRC, "anm_alias.cuh"), os.path.join(CSRC, "anm_frontend.cuh"), os.path.join(CSRC, "anm_peaks.cuh"), os.path.join(os.path.dirname(PKG), "include", "anm.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-fmad=false", "-ftz=true", "-prec-div=false", "-prec-sqrt=false",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPENDS)


def build(force: bool = False, verbose: bool = False, out: str | None = None, extra: list | None = None) -> str:
    """Builds libanm.so in-tree; or, with `out`, a variant (e.g. extra = ["-DANM_BOUNDS_CHECK"]) into another file."""
    if out is not None:
        cmd = [nvcc()] + NVCC_FLAGS + list(extra or []) + ["-o", out] + SOURCES
        subprocess.check_call(cmd)
        return out
    if force or needs_build():
        tmp = LIB + ".tmp.%d" % os.getpid()
        extra = os.environ.get("ANM_NVCC_EXTRA", "").split()      # e.g. -DANM_POOL_THREADS=768 -DANM_CHUNK=64 (tuning experiments)
        cmd = [nvcc()] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
