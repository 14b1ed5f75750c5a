"""Seeded synthetic inputs for the out-of-core DGEMM path (shared by oracle tests, GPU tests, bench).

Holds none of the method's arithmetic: it maps (seed, matrix_id, i, j) to one double with a
counter-based hash, so any element or sub-block can be regenerated (DESIGN.md
"Input recipe").  Two implementations of the same recipe live here -- `fill` (C + OpenMP, for the
multi-GB configs) and `fill_numpy` (vectorised numpy, small sizes) -- and a test checks they agree
bit for bit.  matrix_id: A = 1, B = 2, C = 3.  dist: "uniform" [-1,1), "int" {-4..4}, "normal" (0,1).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "synthgen.c")
_LIB = os.path.join(_HERE, "libsynthgen.so")

DIST = {"uniform": 0, "int": 1, "normal": 2}
MATRIX_ID = {"A": 1, "B": 2, "C": 3}
BASE_SEED = 180805056  # + config index


def build(force: bool = False) -> str:
    """Compile libsynthgen.so with gcc if missing or older than its source."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.synth_fill.restype = ctypes.c_int
        lib.synth_fill.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_int64, ctypes.c_int64,
                                   ctypes.c_uint64, ctypes.c_int, ctypes.c_int, ctypes.c_int64,
                                   ctypes.c_int64, ctypes.c_int64]
        lib.synth_fill_const.restype = ctypes.c_int
        lib.synth_fill_const.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_double]
        _lib = lib
    return _lib


def fill_ptr(ptr: int, rows: int, cols: int, ld: int, seed: int, matrix: str, dist: str,
             row0: int = 0, col0: int = 0, logical_cols: int | None = None) -> None:
    """Fill raw host memory at address `ptr` (rows x cols doubles, leading dimension ld)."""
    rc = _load().synth_fill(ptr, rows, cols, ld, seed, MATRIX_ID[matrix], DIST[dist], row0, col0,
                            cols if logical_cols is None else logical_cols)
    if rc != 0:
        raise ValueError("synth_fill: bad argument")


def fill(arr: np.ndarray, seed: int, matrix: str, dist: str, cols: int | None = None,
         row0: int = 0, col0: int = 0, logical_cols: int | None = None) -> np.ndarray:
    """Fill a C-contiguous float64 2-D array in place; arr.shape[1] is the leading dimension and
    `cols` (default: all) the logical width, columns beyond it are left untouched."""
    assert arr.dtype == np.float64 and arr.ndim == 2 and arr.flags.c_contiguous
    ncols = arr.shape[1] if cols is None else cols
    fill_ptr(arr.ctypes.data, arr.shape[0], ncols, arr.shape[1], seed, matrix, dist, row0, col0,
             ncols if logical_cols is None else logical_cols)
    return arr


def fill_const_ptr(ptr: int, n: int, value: float) -> None:
    if _load().synth_fill_const(ptr, n, value) != 0:
        raise ValueError("synth_fill_const: bad argument")


_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        x = x + np.uint64(0x9E3779B97F4A7C15)
        x = (x ^ (x >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        x = (x ^ (x >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return x ^ (x >> np.uint64(31))


def fill_numpy(rows: int, cols: int, seed: int, matrix: str, dist: str, row0: int = 0,
               col0: int = 0, logical_cols: int | None = None) -> np.ndarray:
    """Same recipe in numpy (small sizes); returns a new dense rows x cols array."""
    lc = cols if logical_cols is None else logical_cols
    i = np.arange(row0, row0 + rows, dtype=np.uint64)[:, None]
    j = np.arange(col0, col0 + cols, dtype=np.uint64)[None, :]
    with np.errstate(over="ignore"):
        lin = i * np.uint64(lc) + j
        key = np.uint64(seed) ^ (np.uint64(MATRIX_ID[matrix]) * np.uint64(0x9E3779B97F4A7C15))
        h = _splitmix64(key ^ _splitmix64(lin))
    if dist == "uniform":
        return (h >> np.uint64(11)).astype(np.float64) * 2.0 ** -52 - 1.0
    if dist == "int":
        return ((h % np.uint64(9)).astype(np.int64) - 4).astype(np.float64)
    if dist == "normal":
        u1 = ((h >> np.uint64(11)).astype(np.float64) + 1.0) * 2.0 ** -53
        u2 = (_splitmix64(h) >> np.uint64(11)).astype(np.float64) * 2.0 ** -53
        return np.sqrt(-2.0 * np.log(u1)) * np.cos(6.283185307179586476925286766559 * u2)
    raise ValueError(dist)


def shape_triangular(A: np.ndarray, dist: str) -> None:
    """Input recipe for the triangular solves: turn a filled square matrix into a WELL CONDITIONED
    triangular operand in place -- off-diagonal entries divided by M (absolute row and column sums below 1), diagonal
    moved to magnitude [1, 2) keeping its sign; for the integer distribution the off-diagonal entries stay as drawn and the
    diagonal becomes +-1 (divisions exact).  Both triangles are shaped; callers poison the one they do not pass.
    Input shaping only: none of the solver's arithmetic lives here."""
    M = A.shape[0]
    assert A.shape[1] >= M
    d = A[np.arange(M), np.arange(M)].copy()
    sign = np.where(d < 0, -1.0, 1.0)
    if dist == "int":
        A[np.arange(M), np.arange(M)] = sign
    else:
        A[:, :M] /= float(max(M, 1))
        A[np.arange(M), np.arange(M)] = sign * (1.0 + np.minimum(np.abs(d), 0.999999))
