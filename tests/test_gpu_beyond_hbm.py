"""GPU parity for a problem whose matrices do not fit the GPU's memory (BASELINE.json configs[4], scaled).

configs[4] (M = N = 163840, K = 8192: 236 GB pinned) needs more host memory than the GPU box has (196 GiB), so the same
shape is scaled to the host exactly as bench.py's default workload is (bench.cfg5_scaled: the largest M = N, a multiple of
2048, whose matrices leave 14 GiB of MemTotal unpinned -- 147456 on the 196 GiB boxes: A + B + C = 193.3 GB, more than the
B200's 191.5 GB of HBM, so no part of the call can be in-core); K = 8192, alpha = 1, beta = 0.5, device budget "all free HBM".
Checked like the other full-size cases (SURVEY 8(c) "V-large"): oracle rows and columns on bands on both sides of slab
boundaries, and whole-matrix checksums (oracle/checksum.py), C0 regenerated from the counter-based generator.

The three matrices are pinned ONCE for both variants (pinning 180 GiB takes about a minute); the test runs whenever the host
has the memory and skips itself otherwise.  HCLOOC_BEYOND_HBM_N=<n> forces another size (experiments).
"""
import json
import os
import sys
import time

import numpy as np
import pytest

import oracle
import oracle.checksum as cks
import synthgen

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
pytestmark = pytest.mark.gpu
RTOL = 1e-13
GiB = 1 << 30
K, ALPHA, BETA = 8192, 1.0, 0.5


def _size():
    sys.path.insert(0, ROOT)
    import bench
    forced = os.environ.get("HCLOOC_BEYOND_HBM_N")
    return int(forced) if forced else bench.cfg5_scaled()["M"]


@pytest.fixture(scope="module")
def big():
    """(H, A, B, C, t_pin): the three pinned host matrices, shared by the variants."""
    import torch
    import paper_1808_05056_b200 as H
    import bench
    assert torch.cuda.is_available()
    M = N = _size()
    total = 8 * (M * K + K * N + M * N)
    avail = bench.meminfo("MemAvailable")
    if avail < total + 8 * GiB:
        pytest.skip(f"host has {avail / GiB:.0f} GiB available, the case pins {total / GiB:.0f} GiB")
    t0 = time.perf_counter()
    A, B, C = H.HostMatrix(M, K), H.HostMatrix(K, N), H.HostMatrix(M, N)
    t_pin = time.perf_counter() - t0
    yield H, A, B, C, t_pin
    for X in (A, B, C):
        X.free()


@pytest.mark.parametrize("variant", ["int", "float"])
def test_matrices_larger_than_hbm(big, variant):
    import torch
    from test_gpu_large import band_indices, _oracle_rows, _oracle_cols
    H, A, B, C, t_pin = big
    M, N = C.rows, C.cols
    total = 8 * (M * K + K * N + M * N)
    hbm = torch.cuda.get_device_properties(0).total_memory
    dist = "int" if variant == "int" else "uniform"
    seed = synthgen.BASE_SEED + 5
    t0 = time.perf_counter()
    synthgen.fill(A.array, seed, "A", dist); synthgen.fill(B.array, seed, "B", dist); synthgen.fill(C.array, seed, "C", dist)
    t_fill = time.perf_counter() - t0
    x = synthgen.fill_numpy(N, 1, 77, "A", "int")[:, 0]
    y = synthgen.fill_numpy(1, M, 77, "B", "int")[0]
    t0 = time.perf_counter()
    if variant == "int":      # exact equality needs no gate denominators: two passes over C0 instead of four
        pre = {"C0x": C.view @ x, "yC0": y @ C.view, "absC0x": np.zeros(M), "yabsC0": np.zeros(N)}
    else:
        pre = cks.before(C.view, x, y)
    t_pre = time.perf_counter() - t0
    plan = H.hclooc_plan(M, N, K, 1, 0, H.hclGetMemSize(0) - GiB)
    rng = np.random.default_rng(13)
    rows, cols = band_indices(M, plan.mb, 2, rng), band_indices(N, plan.nb, 2, rng)
    C0_rows = np.vstack([synthgen.fill(np.empty((1, N)), seed, "C", dist, row0=int(r), logical_cols=N) for r in rows])
    C0_cols = C.view[:, cols].copy()
    st = H.hclooc_dgemm_ex(None, M, N, K, ALPHA, A, A.ld, B, B.ld, BETA, C, C.ld, 0)     # budget 0 = all free HBM
    assert st.bytes_d2h == M * N * 8 and st.bytes_h2d == st.plan.bytes_h2d
    assert total > hbm or os.environ.get("HCLOOC_BEYOND_HBM_N"), "the case no longer exceeds this GPU's memory"
    # (1) bands
    ref_r, D_r = _oracle_rows(ALPHA, A.view, B.view, BETA, C0_rows, rows)
    ref_c, D_c = _oracle_cols(ALPHA, A.view, B.view, BETA, C0_cols, cols)
    got_r, got_c = C.view[rows], C.view[:, cols]
    if variant == "int":
        assert np.array_equal(got_r, ref_r) and np.array_equal(got_c, ref_c)
    else:
        ok, worst = oracle.within_gate(got_r, ref_r, D_r, RTOL)
        assert ok, f"rows: worst |err|/D = {worst:.3e}"
        ok, worst = oracle.within_gate(got_c, ref_c, D_c, RTOL)
        assert ok, f"cols: worst |err|/D = {worst:.3e}"
    # (2) checksums over the whole matrix
    t0 = time.perf_counter()
    Cx, yC, Dx, yD = cks.expected(ALPHA, A.view, B.view, BETA, pre, x, y)
    gx, gy = C.view @ x, y @ C.view
    t_post = time.perf_counter() - t0
    assert not np.isnan(gx).any() and not np.isnan(gy).any()
    if variant == "int":
        assert np.array_equal(gx, Cx) and np.array_equal(gy, yC)
    else:
        assert (np.abs(gx - Cx) <= RTOL * Dx).all() and (np.abs(gy - yC) <= RTOL * yD).all()
    flops = 2.0 * M * N * K
    rec = {"workload": f"cfg5s: {M}x{N}x{K} FP64, alpha=1 beta=0.5, budget = all free HBM", "variant": variant,
           "matrices_bytes": total, "hbm_total_bytes": hbm, "exceeds_hbm": total > hbm,
           "plan": {k: getattr(st.plan, k) for k in ("mb", "nb", "h", "w", "n_steps", "n_sets", "n_abuf", "n_bbuf", "workspace_bytes")},
           "bytes_h2d": int(st.bytes_h2d), "bytes_d2h": int(st.bytes_d2h), "t_total_s": st.t_total_s,
           "tflops_e2e": flops / st.t_total_s / 1e12, "frac_of_fp64_roofline_at_37.2": flops / 37.2e12 / st.t_total_s,
           "t_pin_s": t_pin, "t_fill_s": t_fill, "t_checksums_s": [t_pre, t_post],
           "bands": {"rows": len(rows), "cols": len(cols)}, "parity": "bit-exact" if variant == "int" else "within 1e-13*D"}
    os.makedirs("gpurun_out", exist_ok=True)
    with open("gpurun_out/beyond_hbm.json", "a") as f:
        f.write(json.dumps(rec) + "\n")
