"""Measurement support (not on the product path): the resident-operand int8 tensor issue-rate probe.

``libxcorr_probe.so`` is a separate library (bench_support/int8_issue_probe.cu, built here beside bench.py); libxcorr.so does
not contain it and the product package does not import it.  It shares only the inline-PTX wrappers of csrc/ptx.cuh.  bench.py
calls ``int8_issue_ceiling`` to fix the roofline denominator of xengine_kernel on the box it runs on.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

HERE = Path(__file__).resolve().parent
PKG = HERE.parent / "paper_1503_06189_b200"
SRC = HERE / "int8_issue_probe.cu"
LIB = HERE / "libxcorr_probe.so"
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-shared", "-Xcompiler", "-fPIC"]
OPS_PER_MMA = 2 * 256 * 256 * 32

_lib = None


def needs_build() -> bool:
    deps = [SRC, PKG / "csrc" / "ptx.cuh"]
    return not LIB.exists() or any(d.stat().st_mtime > LIB.stat().st_mtime for d in deps)


def build(force: bool = False) -> Path:
    if not force and not needs_build():
        return LIB
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    subprocess.check_call([os.environ.get("NVCC", "nvcc"), *NVCC_FLAGS, "-o", str(tmp), str(SRC)])
    os.replace(tmp, LIB)
    return LIB


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        if needs_build():
            build()
        L = ctypes.CDLL(str(LIB))
        L.xcorr_probe_int8_issue.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_double),
                                             ctypes.POINTER(ctypes.c_double)]
        L.xcorr_probe_int8_issue.restype = ctypes.c_int
        _lib = L
    return _lib


def int8_issue(mma_per_pair: int, launches: int, pattern: int = 1) -> tuple[float, float]:
    """-> (int8 TOP/s, elapsed ms) of `launches` probe launches of `mma_per_pair` M256 N256 K32 MMAs per CTA pair."""
    tops, ms = ctypes.c_double(), ctypes.c_double()
    rc = lib().xcorr_probe_int8_issue(int(mma_per_pair), int(launches), int(pattern), ctypes.byref(tops), ctypes.byref(ms))
    if rc != 0:
        raise RuntimeError(f"xcorr_probe_int8_issue failed with code {rc}")
    return tops.value, ms.value


def int8_issue_ceiling(pattern: int = 1, sustained_seconds: float = 4.0) -> dict:
    """Burst (best of 10 single launches of about 1 ms after an idle gap; also of about 0.1 ms, the length of one C2 kernel,
    where launch, TMEM allocation and drain are not amortised) and sustained (back-to-back launches for at least
    `sustained_seconds`, power-capped) issue rate.  pattern 1 = operand bytes uniform in [0, 15], like the product's operands."""
    per = 1400                                   # MMAs per pair and launch: 1400 x 128 clk = 179 k clk, about one C2 xengine_kernel
    long_per = 14000                             # ~1 ms: launch, TMEM allocation and drain amortised
    int8_issue(per, 3, pattern)
    burst_short = max(int8_issue(per, 1, pattern)[0] for _ in range(10))
    burst = max(int8_issue(long_per, 1, pattern)[0] for _ in range(10))
    t1, ms1 = int8_issue(long_per, 20, pattern)
    n = max(20, int(20 * sustained_seconds * 1e3 / ms1))
    sustained, ms = int8_issue(long_per, n, pattern)
    return {"burst_tops": burst, "burst_tops_single_0p1ms_launch": burst_short, "sustained_tops": sustained, "sustained_seconds": ms * 1e-3,
            "pattern": pattern, "mma_per_pair_per_launch": long_per, "shape": "cta_group::2 M256 N256 K32 kind::i8, MN-major SWIZZLE_128B, resident operands"}
