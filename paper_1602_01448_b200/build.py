"""Builds the C-ABI library `libsharp_b200.so` in-tree with nvcc for sm_100a (no JIT cache, no torch extension:
the library has no torch types in its interface)."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libsharp_b200.so")
SOURCES = ["sharp_b200.cu"]
HEADERS = ["fft_regs.cuh", "frame_common.cuh", "frame_r.cuh", "frame_s.cuh", "object_kernels.cuh", "probe_kernels.cuh", os.path.join("..", "..", "include", "sharp_b200.h")]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    """nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo ... -> paper_1602_01448_b200/libsharp_b200.so"""
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "nvcc")
        cmd = [nvcc, "-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
               "-shared", "-Xcompiler", "-fPIC", "-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        subprocess.check_call(cmd)
    return LIB
