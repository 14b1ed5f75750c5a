"""Times the out-of-core DSYRK (hclooc_dsyrk) beside the DGEMM it replaces (C = alpha*A*A^T + beta*C through hclooc_dgemm_t with
op(B) = A^T, which computes and moves both triangles), on pinned host matrices under a device budget.

    python -m paper_1808_05056_b200.dsyrk_bench [--n N] [--k K] [--budget BYTES] [--reps R]

Prints one JSON line: times, TFLOP/s counted on the flops each operation must do (DSYRK: N(N+1)K, DGEMM: 2 N^2 K), host-link bytes.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main() -> None:
    import synthgen
    import paper_1808_05056_b200 as H
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=32768)
    ap.add_argument("--k", type=int, default=8192)
    ap.add_argument("--budget", type=int, default=4 << 30)
    ap.add_argument("--reps", type=int, default=3)
    ap.add_argument("--beta", type=float, default=1.0)
    args = ap.parse_args()
    N, K = args.n, args.k
    A, C = H.HostMatrix(N, K), H.HostMatrix(N, N)
    synthgen.fill(A.array, synthgen.BASE_SEED + 7, "A", "uniform")
    synthgen.fill(C.array, synthgen.BASE_SEED + 7, "C", "uniform")
    ctx = H.hclooc_ctx_create(0)
    out = {"N": N, "K": K, "budget_bytes": args.budget, "beta": args.beta}
    try:
        for label, call, flops in (
                ("dsyrk_lower", lambda: H.hclooc_dsyrk(ctx, H.HCL_UPLO_LOWER, H.HCL_OP_N, N, K, 1.0, A, K, args.beta, C, N, args.budget), float(N) * (N + 1) * K),
                ("dgemm_nt", lambda: H.hclooc_dgemm_t(ctx, 0, 1, N, N, K, 1.0, A, K, A, K, args.beta, C, N, args.budget), 2.0 * N * N * K)):
            ts, st = [], None
            for _ in range(max(2, args.reps)):
                st = call()
                ts.append(st.t_total_s)
            t = float(np.mean(ts[1:]))
            out[label] = {"t_s": t, "tflops": flops / t / 1e12, "flops": flops, "h2d_GB": st.bytes_h2d / 1e9, "d2h_GB": st.bytes_d2h / 1e9,
                          "kernels": int(st.n_kernels), "t_flop_s_at_37.2": flops / 37.2e12}
        out["dsyrk_time_over_dgemm_time"] = out["dsyrk_lower"]["t_s"] / out["dgemm_nt"]["t_s"]
    finally:
        H.hclooc_ctx_destroy(ctx)
    print(json.dumps(out))


if __name__ == "__main__":
    main()
