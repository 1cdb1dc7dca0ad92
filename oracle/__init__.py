"""CPU ORACLE for the X-engine correlation path -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares nothing with the CUDA path in
``paper_1503_06189_b200/`` (no code, headers, tables, helpers) and never imports it.

Contents
--------
* ``naive`` / ``planar`` / ``pairs``: ctypes front ends to ``xcorr_oracle.c`` (plain C, the
  definition written out; see that file's header for the passages followed: PAPER.md:25, :65-67,
  :93, :99 and the readings R1..R5 in DESIGN.md).
* ``brute_full``: an independent numpy statement of the same definition that builds the *full*
  N x N complex matrix ``sum_t x x^H`` with int64 ``einsum`` (tiny inputs only).  Used to pin the C.
* ``identity_total_power`` / ``freivalds_rhs`` / ``hermitian_from_triangle``: O(N*T) exact integer
  identities that any correct V satisfies; they check whole matrices at sizes where the full
  triangle costs minutes.
* ``unpack``: the nibble decode (R2, R3) in numpy.

Every function here is pinned in ``tests/test_oracle_pins.py``; nothing is "parity unpinned".
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "xcorr_oracle.c"
_LIB = _HERE / "liboracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile xcorr_oracle.c with gcc -O2 -fopenmp (building the checker is not using it)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-o", str(tmp), str(_SRC)]
        )
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(str(_LIB))
        u8p = ctypes.POINTER(ctypes.c_uint8)
        i32p = ctypes.POINTER(ctypes.c_int32)
        i64p = ctypes.POINTER(ctypes.c_int64)
        ci = ctypes.c_int
        lib.xcorr_oracle_naive.argtypes = [u8p, ci, ci, ci, i32p]
        lib.xcorr_oracle_naive.restype = ci
        lib.xcorr_oracle_planar.argtypes = [u8p, ci, ci, ci, i32p]
        lib.xcorr_oracle_planar.restype = ci
        lib.xcorr_oracle_planar_range.argtypes = [u8p, ci, ci, ci, ci, ci, i32p]
        lib.xcorr_oracle_planar_range.restype = ci
        lib.xcorr_oracle_pairs.argtypes = [u8p, ci, ci, ci, i32p, ctypes.c_int64, i64p]
        lib.xcorr_oracle_pairs.restype = ci
        lib.xcorr_oracle_pair_index.argtypes = [ci, ci, ci]
        lib.xcorr_oracle_pair_index.restype = ctypes.c_int64
        lib.xcorr_oracle_threads.argtypes = []
        lib.xcorr_oracle_threads.restype = ci
        _lib = lib
    return _lib


def threads() -> int:
    """OpenMP threads the C oracle will use (what bench.py reports as ``cores``)."""
    return int(_load().xcorr_oracle_threads())


def n_pairs(n_inputs: int) -> int:
    return n_inputs * (n_inputs + 1) // 2


def pair_index(n_inputs: int, i: int, j: int) -> int:
    """R4: p(i,j) = i(2N-i+1)/2 + (j-i), i <= j (row-major upper triangle incl. diagonal)."""
    return int(_load().xcorr_oracle_pair_index(n_inputs, i, j))


def _check_frame(frame: np.ndarray) -> tuple[int, int, int]:
    if frame.dtype != np.uint8 or frame.ndim != 3 or not frame.flags.c_contiguous:
        raise ValueError("frame must be a C-contiguous uint8 array of shape [T][F][N]")
    t, f, n = frame.shape
    return n, f, t


def _u8(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8))


def _i32(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))


def naive(frame: np.ndarray) -> np.ndarray:
    """Literal (f, i<=j, t) loop nest.  Returns int32[F][P][2]."""
    n, f, t = _check_frame(frame)
    out = np.zeros((f, n_pairs(n), 2), dtype=np.int32)
    rc = _load().xcorr_oracle_naive(_u8(frame), n, f, t, _i32(out))
    if rc:
        raise OverflowError("a visibility does not fit int32")
    return out


def planar(frame: np.ndarray, f_begin: int = 0, f_end: int | None = None) -> np.ndarray:
    """Planar-storage form of the same loop nest (OpenMP).  Returns int32[F][P][2]; with a channel
    range, channels outside it are zero."""
    n, f, t = _check_frame(frame)
    f_end = f if f_end is None else f_end
    if not (0 <= f_begin <= f_end <= f):
        raise ValueError("bad channel range")
    out = np.zeros((f, n_pairs(n), 2), dtype=np.int32)
    rc = _load().xcorr_oracle_planar_range(_u8(frame), n, f, t, f_begin, f_end, _i32(out))
    if rc == 3:
        raise MemoryError("oracle scratch allocation failed")
    if rc:
        raise OverflowError("a visibility does not fit int32")
    return out


def pairs(frame: np.ndarray, idx: np.ndarray) -> np.ndarray:
    """Exact sums for listed (f, i, j) triples (i <= j).  idx int32[K][3] -> int64[K][2]."""
    n, f, t = _check_frame(frame)
    idx = np.ascontiguousarray(idx, dtype=np.int32)
    if idx.ndim != 2 or idx.shape[1] != 3:
        raise ValueError("idx must be [K][3] = (f, i, j)")
    out = np.zeros((idx.shape[0], 2), dtype=np.int64)
    rc = _load().xcorr_oracle_pairs(
        _u8(frame), n, f, t, _i32(idx), idx.shape[0],
        out.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)),
    )
    if rc:
        raise ValueError("bad (f,i,j) triple")
    return out


# ----------------------------------------------------------------------------------------------
# numpy statements of the same definition (independent of the C above)
# ----------------------------------------------------------------------------------------------
def unpack(frame: np.ndarray) -> tuple[np.ndarray, np.ndarray]:
    """R2/R3: (re, im) int64 arrays, re = sext4(high nibble), im = sext4(low nibble)."""
    b = frame.astype(np.int64)
    hi = b >> 4
    lo = b & 15
    return np.where(hi >= 8, hi - 16, hi), np.where(lo >= 8, lo - 16, lo)


def brute_full(frame: np.ndarray) -> tuple[np.ndarray, np.ndarray]:
    """Full N x N matrices (Re, Im) of V_f = sum_t x x^H, int64, shape [F][N][N].  Tiny inputs only.

    (a+bi)(c-di) = (ac+bd) + i(bc-ad), written with four real einsums."""
    re, im = unpack(frame)  # [T][F][N]
    vre = np.einsum("tfi,tfj->fij", re, re) + np.einsum("tfi,tfj->fij", im, im)
    vim = np.einsum("tfi,tfj->fij", im, re) - np.einsum("tfi,tfj->fij", re, im)
    return vre, vim


def triangle_from_full(vre: np.ndarray, vim: np.ndarray) -> np.ndarray:
    """Pack [F][N][N] full matrices into int64[F][P][2] in the R4 order."""
    f, n, _ = vre.shape
    iu = np.triu_indices(n)  # row-major upper triangle incl. diagonal == R4 order
    return np.stack([vre[:, iu[0], iu[1]], vim[:, iu[0], iu[1]]], axis=-1)


def hermitian_from_triangle(tri_f: np.ndarray, n_inputs: int) -> np.ndarray:
    """One channel's [P][2] triangle -> full complex128-free representation: (Re, Im) int64 [N][N]
    with V[j,i] = conj(V[i,j])."""
    iu = np.triu_indices(n_inputs)
    vre = np.zeros((n_inputs, n_inputs), dtype=np.int64)
    vim = np.zeros((n_inputs, n_inputs), dtype=np.int64)
    vre[iu] = tri_f[:, 0]
    vim[iu] = tri_f[:, 1]
    il = np.tril_indices(n_inputs, -1)
    vre[il] = vre.T[il]
    vim[il] = -vim.T[il]
    return vre, vim


def identity_total_power(frame: np.ndarray) -> np.ndarray:
    """int64[F]:  sum_t |sum_n x_n|^2, which must equal  sum_i V_ii + 2 sum_{i<j} Re V_ij."""
    re, im = unpack(frame)
    sr = re.sum(axis=2)
    si = im.sum(axis=2)
    return (sr * sr + si * si).sum(axis=0)


def lhs_total_power(tri: np.ndarray, n_inputs: int) -> np.ndarray:
    """int64[F]: sum_i V_ii + 2 sum_{i<j} Re V_ij from a [F][P][2] triangle."""
    iu = np.triu_indices(n_inputs)
    w = np.where(iu[0] == iu[1], 1, 2).astype(np.int64)
    return (tri[:, :, 0].astype(np.int64) * w[None, :]).sum(axis=1)


def freivalds_rhs(frame_f: np.ndarray, u: np.ndarray, w: np.ndarray) -> tuple[int, int]:
    """For one channel's bytes [T][N] and integer vectors u, w (real): the exact value of
    u^T V w = sum_t (u . x_t) * conj(w . x_t), as (Re, Im) Python ints.  O(N*T)."""
    b = frame_f.astype(np.int64)
    hi = b >> 4
    lo = b & 15
    re = np.where(hi >= 8, hi - 16, hi)
    im = np.where(lo >= 8, lo - 16, lo)
    ar, ai = re @ u, im @ u  # a_t = u . x_t
    br, bi = re @ w, im @ w  # b_t = w . x_t
    return int((ar * br + ai * bi).sum()), int((ai * br - ar * bi).sum())


def freivalds_lhs(tri_f: np.ndarray, n_inputs: int, u: np.ndarray, w: np.ndarray) -> tuple[int, int]:
    """u^T V w from one channel's triangle, V completed Hermitian-ly.  O(N^2)."""
    vre, vim = hermitian_from_triangle(tri_f.astype(np.int64), n_inputs)
    return int(u @ vre @ w), int(u @ vim @ w)
