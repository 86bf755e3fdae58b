"""Builds libafqmc.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

PKG_DIR = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(PKG_DIR, "csrc")
LIB = os.path.join(PKG_DIR, "libafqmc.so")
OZAKI_LIB = os.path.join(PKG_DIR, "libafqmc_ozaki.so")       # the Ozaki-scheme experiment (include/afqmc_ozaki.h)
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared"]


def _sources():
    out = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith((".cu", ".cuh")) and f != "ozaki_i8.cu"]
    out.append(os.path.join(os.path.dirname(PKG_DIR), "include", "afqmc.h"))
    return out


def _nvcc():
    nvcc = os.environ.get("NVCC") or "/usr/local/cuda/bin/nvcc"
    return nvcc if os.path.exists(nvcc) else "nvcc"


def build_ozaki_library(force: bool = False) -> str:
    """Compile csrc/ozaki_i8.cu -> libafqmc_ozaki.so (tcgen05 kind::i8 experiment) if missing or stale."""
    srcs = [os.path.join(CSRC, "ozaki_i8.cu"), os.path.join(os.path.dirname(PKG_DIR), "include", "afqmc_ozaki.h")]
    if not force and os.path.exists(OZAKI_LIB) and all(os.path.getmtime(s) <= os.path.getmtime(OZAKI_LIB) for s in srcs):
        return OZAKI_LIB
    cmd = [_nvcc(), *NVCC_FLAGS, "-o", OZAKI_LIB, srcs[0]]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + res.stdout + res.stderr)
    return OZAKI_LIB


def build_library(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/afqmc.cu -> libafqmc.so if missing or older than any source.  Returns the path.
    AFQMC_NVCC_EXTRA adds compiler flags for diagnostic builds (-DAFQMC_K1_PHASE_CLOCKS, -DAFQMC_K2_ABLATE=n: see the
    kernels' headers); such a build must be forced and must be replaced by a plain one afterwards."""
    if not force and os.path.exists(LIB):
        t = os.path.getmtime(LIB)
        if all(os.path.getmtime(s) <= t for s in _sources()):
            return LIB
    cmd = [_nvcc(), *NVCC_FLAGS, *os.environ.get("AFQMC_NVCC_EXTRA", "").split(), "-o", LIB, os.path.join(CSRC, "afqmc.cu")]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + res.stdout + res.stderr)
    if verbose:
        print(res.stderr)
    return LIB
