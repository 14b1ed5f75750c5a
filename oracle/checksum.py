"""TEST INFRASTRUCTURE ONLY -- whole-matrix checksum identities for sizes where the full oracle is hours.

For C = alpha*A*B + beta*C0 and any vectors x (length N) and y (length M):

    C x   = alpha * A (B x) + beta * (C0 x)          y^T C = alpha * (y^T A) B + beta * (y^T C0)

at O(MN + MK + KN) cost instead of O(MNK).  With small-integer A, B, C0, x, y and alpha, beta multiples of
1/2 every term is an integer or half-integer below 2^53, so both identities hold EXACTLY and any single
wrong element of C changes one row sum and one column sum (SURVEY 8(c) "V-large" (2)).  On float inputs
the same identities hold within the summed element gate  sum_j RTOL * D_ij * |x_j|  (V-large (3)).
numpy only; shares nothing with the CUDA path.
"""
from __future__ import annotations

import numpy as np


def _chunks(n: int, chunk: int):
    return [(r, min(n, r + chunk)) for r in range(0, n, chunk)]


def _pool():
    from concurrent.futures import ThreadPoolExecutor
    import os
    return ThreadPoolExecutor(max_workers=min(16, os.cpu_count() or 1))


def _abs_mv(X: np.ndarray, v: np.ndarray, chunk: int = 256) -> np.ndarray:
    """|X| @ |v| in row chunks (bounded temporaries for multi-GB X; the chunks run on a thread pool -- every output element
    is still one dot product of its own row, so the values do not depend on the chunking)."""
    av = np.abs(v)
    out = np.empty(X.shape[0])

    def one(rr):
        out[rr[0]:rr[1]] = np.abs(X[rr[0]:rr[1]]) @ av

    with _pool() as ex:
        list(ex.map(one, _chunks(X.shape[0], chunk)))
    return out


def _abs_vm(v: np.ndarray, X: np.ndarray, chunk: int = 256) -> np.ndarray:
    """|v| @ |X| in row chunks: the chunk partials are computed on a thread pool and added up in chunk order."""
    av = np.abs(v)
    out = np.zeros(X.shape[1])
    rows = _chunks(X.shape[0], chunk)
    with _pool() as ex:
        for base in range(0, len(rows), 64):          # bounded number of partials alive
            parts = list(ex.map(lambda rr: av[rr[0]:rr[1]] @ np.abs(X[rr[0]:rr[1]]), rows[base:base + 64]))
            for p in parts:
                out += p
    return out


def before(C0: np.ndarray, x: np.ndarray, y: np.ndarray):
    """The C0-dependent terms; call while C still holds C0 (C is updated in place afterwards)."""
    return {"C0x": C0 @ x, "yC0": y @ C0, "absC0x": _abs_mv(C0, x), "yabsC0": _abs_vm(y, C0)}


def expected(alpha, A, B, beta, pre, x, y):
    """(C x, y^T C) predicted from A, B and the saved C0 terms, plus the summed gate denominators."""
    Cx = alpha * (A @ (B @ x)) + beta * pre["C0x"]
    yC = alpha * ((y @ A) @ B) + beta * pre["yC0"]
    Dx = abs(alpha) * _abs_mv(A, _abs_mv(B, x)) + abs(beta) * pre["absC0x"]
    yD = abs(alpha) * _abs_vm(_abs_vm(y, A), B) + abs(beta) * pre["yabsC0"]
    return Cx, yC, Dx, yD
