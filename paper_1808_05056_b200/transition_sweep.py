"""The paper's own experiment shape on one B200:

square FP64 DGEMM, N swept across the point where A, B and C stop fitting the device budget, end-to-end
TFLOP/s = 2 N^3 / t with the host<->device transfers inside t (:368), for

  tuned : hclooc_dgemm_ex   -- this library's scheduler (serpentine order, cached A slices, B prefetch, several
                               compute streams) and
  fig2  : hclooc_dgemm_fig2 -- the paper's Figure 2 pipeline (two round-robin streams, five event families,
                               single B buffer) written over the exported hcl* runtime calls,

both on the same pinned host matrices and with the same device budget (default 12.2e9 bytes: the paper's
12 GB cards switched to out-of-core above N = 22528, :368).  What the paper reports for its own two codes is
"0 % loss at the transition" (:372, :396) and 4-10 % between the abstraction and the hand-tuned code (:15).

    python -m paper_1808_05056_b200.transition_sweep [--budget BYTES] [--sizes N,N,...] [--reps R] [--out FILE]

Prints one JSON line per size and a Markdown table at the end (also written to --out).
"""
from __future__ import annotations

import argparse
import ctypes
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

DEFAULT_SIZES = [4096, 8192, 12288, 16384, 20480, 22528, 23552, 24576, 28672, 32768, 36864, 40960, 46080]


def main() -> None:
    import synthgen
    import paper_1808_05056_b200 as H
    ap = argparse.ArgumentParser()
    ap.add_argument("--budget", type=int, default=12_200_000_000)
    ap.add_argument("--sizes", default=",".join(str(n) for n in DEFAULT_SIZES))
    ap.add_argument("--reps", type=int, default=3, help="timed calls per size and pipeline (the first is discarded)")
    ap.add_argument("--alpha", type=float, default=1.0)
    ap.add_argument("--beta", type=float, default=1.0)
    ap.add_argument("--out", default="")
    args = ap.parse_args()
    sizes = sorted(int(x) for x in args.sizes.split(","))
    nmax = sizes[-1]
    # one pinned allocation per matrix, reused for every size as a dense N x N matrix (ld = N)
    bufs = [H.HostMatrix(nmax, nmax) for _ in range(3)]
    ctx = H.hclooc_ctx_create(0)
    rows = []
    try:
        for n in sizes:
            A, B, C = (np.frombuffer((ctypes.c_double * (n * n)).from_address(X.ptr), dtype=np.float64).reshape(n, n)
                       for X in bufs)
            for arr, name in ((A, "A"), (B, "B"), (C, "C")):
                synthgen.fill(arr, synthgen.BASE_SEED + 9, name, "uniform")
            in_core = 24 * n * n <= args.budget
            rec = {"N": n, "in_core": in_core, "budget_bytes": args.budget, "flops": 2.0 * n ** 3}
            for label, call in (("tuned", lambda: H.hclooc_dgemm_ex(ctx, n, n, n, args.alpha, A, n, B, n, args.beta, C, n, args.budget)),
                                ("fig2", lambda: H.hclooc_dgemm_fig2(n, n, n, args.alpha, A, n, B, n, args.beta, C, n, args.budget))):
                ts, st = [], None
                for _ in range(max(2, args.reps)):
                    st = call()
                    ts.append(st.t_total_s)
                t = float(np.mean(ts[1:]))
                rec[label] = {"t_s": t, "tflops": 2.0 * n ** 3 / t / 1e12, "h": st.plan.h, "w": st.plan.w, "steps": st.plan.n_steps,
                              "h2d_GB": st.bytes_h2d / 1e9, "d2h_GB": st.bytes_d2h / 1e9}
            rec["fig2_over_tuned"] = rec["fig2"]["tflops"] / rec["tuned"]["tflops"]
            rows.append(rec)
            print(json.dumps(rec), flush=True)
    finally:
        H.hclooc_ctx_destroy(ctx)
        for X in bufs:
            X.free()
    lines = ["| N | fits budget | tuned TFLOP/s (h x w) | Figure-2 TFLOP/s (h x w) | Figure-2 / tuned |", "|---|---|---|---|---|"]
    for r in rows:
        lines.append(f"| {r['N']} | {'yes' if r['in_core'] else 'no'} | {r['tuned']['tflops']:.2f} ({r['tuned']['h']} x {r['tuned']['w']}) | "
                     f"{r['fig2']['tflops']:.2f} ({r['fig2']['h']} x {r['fig2']['w']}) | {r['fig2_over_tuned']:.3f} |")
    table = "\n".join(lines)
    print(table)
    if args.out:
        with open(args.out, "w") as f:
            f.write(table + "\n\n" + "\n".join(json.dumps(r) for r in rows) + "\n")


if __name__ == "__main__":
    main()
