"""GPU parity at full BASELINE.json sizes for configs[2] and configs[3] (SURVEY 8(c) "V-large").

The full oracle would take hours here (7e13 / 1.4e14 flops), so the updated C is checked on
  (1) complete rows and columns computed by the oracle one by one -- first, last, both sides of slab
      boundaries of the plan, and random ones -- bit-exact on the {-4..4} integer variant, within
      1e-13 * D on the float inputs, and
  (2) whole-matrix checksum identities C x and y^T C (oracle/checksum.py): exact on the integer variant,
      within the summed gate on float inputs.
C0 is regenerated from the counter-based generator (C is overwritten in place).
"""
import numpy as np
import pytest

import oracle
import oracle.checksum as cks
import synthgen

pytestmark = pytest.mark.gpu
RTOL = 1e-13
GiB = 1 << 30

CASES = {
    # name: M, N, K, alpha, beta, budget, dist (BASELINE.json configs[2], configs[3])
    "cfg3": (32768, 32768, 32768, 1.0, 0.0, 4 * GiB, "uniform", 3),
    "cfg4": (65536, 65536, 16384, 2.0, -1.0, 16 * GiB, "normal", 4),
}


def band_indices(n, blk, count, rng):
    idx = {0, n - 1} | {int(v) for v in rng.integers(0, n, count)}
    nblk = -(-n // blk)
    for b in sorted({1, nblk // 2, nblk - 1} - {0}):
        if b * blk < n:
            idx |= {b * blk - 1, b * blk}
    return np.array(sorted(idx))


@pytest.mark.parametrize("name", ["cfg3", "cfg4"])
@pytest.mark.parametrize("variant", ["float", "int"])
def test_full_size_bands_and_checksums(name, variant):
    import paper_1808_05056_b200 as H
    M, N, K, alpha, beta, budget, dist, idx = CASES[name]
    dist = "int" if variant == "int" else dist
    seed = synthgen.BASE_SEED + idx
    A, B, C = H.HostMatrix(M, K), H.HostMatrix(K, N), H.HostMatrix(M, N)
    try:
        synthgen.fill(A.array, seed, "A", dist); synthgen.fill(B.array, seed, "B", dist)
        if beta == 0.0:
            synthgen.fill_const_ptr(C.ptr, M * N, float("nan"))      # beta == 0: C must not be read (G8)
        else:
            synthgen.fill(C.array, seed, "C", dist)
        x = synthgen.fill_numpy(N, 1, 77, "A", "int")[:, 0]
        y = synthgen.fill_numpy(1, M, 77, "B", "int")[0]
        zero = np.zeros(1)
        pre = cks.before(C.view, x, y) if beta != 0.0 else {"C0x": zero, "yC0": zero, "absC0x": zero, "yabsC0": zero}
        plan = H.hclooc_plan(M, N, K, beta != 0.0, 0, budget)
        rng = np.random.default_rng(11)
        rows, cols = band_indices(M, plan.mb, 3, rng), band_indices(N, plan.nb, 3, rng)
        # C0 on the bands, regenerated (not copied) from the generator
        if beta != 0.0:
            C0_rows = np.vstack([synthgen.fill(np.empty((1, N)), seed, "C", dist, row0=int(r), logical_cols=N) for r in rows])
            C0_cols = C.view[:, cols].copy()
        st = H.hclooc_dgemm_ex(None, M, N, K, alpha, A, A.ld, B, B.ld, beta, C, C.ld, budget)
        assert st.plan.workspace_bytes <= budget
        assert st.bytes_h2d == st.plan.bytes_h2d and st.bytes_d2h == M * N * 8
        assert not np.isnan(C.view[rows]).any() and not np.isnan(C.view[:, cols]).any()
        # (1) bands: the oracle on complete rows / columns
        ref_r, D_r = _oracle_rows(alpha, A.view, B.view, beta, C0_rows if beta != 0.0 else None, rows)
        ref_c, D_c = _oracle_cols(alpha, A.view, B.view, beta, C0_cols if beta != 0.0 else None, cols)
        got_r, got_c = C.view[rows], C.view[:, cols]
        if variant == "int":
            assert np.array_equal(got_r, ref_r) and np.array_equal(got_c, ref_c)
        else:
            ok, worst = oracle.within_gate(got_r, ref_r, D_r, RTOL)
            assert ok, f"rows: worst |err|/D = {worst:.3e}"
            ok, worst = oracle.within_gate(got_c, ref_c, D_c, RTOL)
            assert ok, f"cols: worst |err|/D = {worst:.3e}"
        # (2) checksums over the whole matrix
        Cx, yC, Dx, yD = cks.expected(alpha, A.view, B.view, beta, pre, x, y)
        gx, gy = C.view @ x, y @ C.view
        assert not np.isnan(gx).any() and not np.isnan(gy).any()
        if variant == "int":
            assert np.array_equal(gx, Cx) and np.array_equal(gy, yC)
        else:
            assert (np.abs(gx - Cx) <= RTOL * Dx).all() and (np.abs(gy - yC) <= RTOL * yD).all()
    finally:
        for X in (A, B, C):
            X.free()


def _oracle_rows(alpha, A, B, beta, C0_rows, rows):
    """Rows `rows` of alpha*A*B + beta*C0 with C0 given only on those rows (dense len(rows) x N)."""
    Asub = np.ascontiguousarray(A[rows])
    return oracle.dgemm_sub(alpha, Asub, B, beta, C0_rows, rows=None, cols=None)


def _oracle_cols(alpha, A, B, beta, C0_cols, cols):
    """Columns `cols` with C0 given only on those columns (dense M x len(cols))."""
    Bsub = np.ascontiguousarray(B[:, cols])
    return oracle.dgemm_sub(alpha, A, Bsub, beta, C0_cols, rows=None, cols=None)
