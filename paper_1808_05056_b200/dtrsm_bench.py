"""Times the out-of-core DTRSM (hclooc_dtrsm: op(T) X = alpha B, T and B in pinned host memory) under a device budget.

    python -m paper_1808_05056_b200.dtrsm_bench [--m M] [--n N] [--budget BYTES] [--reps R] [--uplo 0|1] [--trans 0|1]

Prints one JSON line: time, TFLOP/s on the M*M*N flops of the solve, host-link bytes, and the roofline of the call as
bench.py defines it (the slower of the flops at 37.2 TFLOP/s and the call's own bytes at the measured link rates).
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

FP64_PEAK = 37.2e12                      # DMMA issue rate measured by hclooc_probe_fp64 (profiles/r01_box_probe.md)
H2D, D2H, DUPLEX = 55.5e9, 51.5e9, 88e9  # link rates of DESIGN.md section 10


def main() -> None:
    import synthgen
    import paper_1808_05056_b200 as H
    ap = argparse.ArgumentParser()
    ap.add_argument("--m", type=int, default=32768)
    ap.add_argument("--n", type=int, default=32768)
    ap.add_argument("--budget", type=int, default=4 << 30)
    ap.add_argument("--reps", type=int, default=3)
    ap.add_argument("--uplo", type=int, default=0)
    ap.add_argument("--trans", type=int, default=0)
    args = ap.parse_args()
    M, N = args.m, args.n
    A, B = H.HostMatrix(M, M), H.HostMatrix(M, N)
    synthgen.fill(A.array, synthgen.BASE_SEED + 9, "A", "uniform")
    synthgen.shape_triangular(A.view, "uniform")
    synthgen.fill(B.array, synthgen.BASE_SEED + 9, "B", "uniform")
    ctx = H.hclooc_ctx_create(0)
    try:
        ts, st = [], None
        for _ in range(max(2, args.reps)):
            st = H.hclooc_dtrsm(ctx, args.uplo, args.trans, 0, M, N, 1.0, A, M, B, N, args.budget)
            ts.append(st.t_total_s)
    finally:
        H.hclooc_ctx_destroy(ctx)
    t = float(np.mean(ts[1:]))
    flops = float(M) * M * N
    t_flop = flops / FP64_PEAK
    t_link = max(st.bytes_h2d / H2D, st.bytes_d2h / D2H, (st.bytes_h2d + st.bytes_d2h) / DUPLEX)
    print(json.dumps({"M": M, "N": N, "uplo": args.uplo, "trans": args.trans, "budget_bytes": args.budget, "t_s": t, "t_all_s": ts,
                      "tflops": flops / t / 1e12, "flops": flops, "NB": int(st.plan.mb), "chunk": int(st.plan.nb),
                      "block_rows": int(st.plan.h), "h2d_GB": st.bytes_h2d / 1e9, "d2h_GB": st.bytes_d2h / 1e9,
                      "kernels": int(st.n_kernels), "workspace_bytes": int(st.plan.workspace_bytes),
                      "t_flop_s": t_flop, "t_link_s": t_link, "bound": "fp64" if t_flop >= t_link else "link",
                      "frac_of_roofline": max(t_flop, t_link) / t}))


if __name__ == "__main__":
    main()
