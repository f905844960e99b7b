"""Build steps: the sm_100a CUDA library (nvcc, in-tree) and the oracle's plain-C helper (gcc)."""
from __future__ import annotations

import os
import shutil
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_1501_01752_b200", "csrc")
LIB = os.path.join(ROOT, "paper_1501_01752_b200", "libgsm_b200.so")
ORACLE_SRC = os.path.join(ROOT, "oracle", "toeplitz_oracle.c")
ORACLE_LIB = os.path.join(ROOT, "oracle", "libtoeplitz_oracle.so")


def _stale(target, sources):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in sources)


def _nvcc():
    return shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"


def build_cuda(force=False, verbose=False):
    srcs = sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cpp")))
    deps = srcs + [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    deps.append(os.path.join(ROOT, "include", "gsm.h"))
    if not force and not _stale(LIB, deps):
        return LIB
    cmd = [_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
           "-shared", "-Xcompiler", "-fPIC", "-I", os.path.join(ROOT, "include"), "-I", CSRC,
           "-o", LIB] + srcs
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.run(cmd, check=True)
    return LIB


def build_oracle(force=False):
    if not force and not _stale(ORACLE_LIB, [ORACLE_SRC]):
        return ORACLE_LIB
    subprocess.run(["gcc", "-O3", "-fopenmp", "-fcx-limited-range", "-shared", "-fPIC",
                    "-o", ORACLE_LIB, ORACLE_SRC], check=True)
    return ORACLE_LIB
