"""Test-support CUDA code, built in-tree into tests/support/libxcorr_testsupport.so.  Nothing in the product imports it.

simt_xcorr: a standalone one-thread-per-visibility kernel (simt_xcorr.cu) used by the GPU tests as an on-device second
opinion beside the oracle comparisons; it shares no code with libxcorr.so.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

HERE = Path(__file__).resolve().parent
LIB = HERE / "libxcorr_testsupport.so"
SOURCES = [HERE / "simt_xcorr.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-shared", "-Xcompiler", "-fPIC"]

_lib = None


def needs_build() -> bool:
    return not LIB.exists() or any(s.stat().st_mtime > LIB.stat().st_mtime for s in SOURCES)


def build(force: bool = False) -> Path:
    if not force and not needs_build():
        return LIB
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    subprocess.check_call([os.environ.get("NVCC", "nvcc"), *NVCC_FLAGS, "-o", str(tmp), *map(str, SOURCES)])
    os.replace(tmp, LIB)
    return LIB


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        if needs_build():
            build()
        L = ctypes.CDLL(str(LIB))
        L.simt_xcorr.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
        L.simt_xcorr.restype = ctypes.c_int
        _lib = L
    return _lib


def simt_xcorr(frame_dev, stream=None):
    """frame_dev: CUDA uint8 tensor [T][F][N] -> CUDA int32 tensor [F][P][2] computed by the SIMT second-opinion kernel."""
    import torch
    t, f, n = frame_dev.shape
    out = torch.empty((f, n * (n + 1) // 2, 2), dtype=torch.int32, device="cuda")
    st = torch.cuda.current_stream().cuda_stream if stream is None else stream.cuda_stream
    rc = lib().simt_xcorr(frame_dev.data_ptr(), n, f, t, out.data_ptr(), st)
    if rc != 0:
        raise RuntimeError(f"simt_xcorr failed: {rc}")
    return out
