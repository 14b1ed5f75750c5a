"""Direct mode against the staged pipeline on small problems (BASELINE config 1).

For square FP64 problems N x N x N under a small device budget, times hclooc_dgemm_ex three ways on the same
pinned host matrices:

  staged : slices streamed through device buffers (hclooc_ctx_set_direct(ctx, 0)) -- the paper's pipeline shape,
  direct : no device buffer, one launch whose TMA loads read A and B from host memory and whose epilogue updates C
           in host memory (hclooc_ctx_set_direct(ctx, 1)),
  auto   : what the cost model picks (-1),

and prints the measured times beside the planner's model of each (plan.t_model_s), which is how the constants of
the direct-mode model (50 GB/s for SM-initiated reads of pinned host memory, 30 us fixed) were set.

    python -m paper_1808_05056_b200.direct_sweep [--budget BYTES] [--sizes N,N,...] [--reps R] [--out FILE]
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

DEFAULT_SIZES = [128, 256, 512, 768, 1024, 1536, 2048]


def main() -> None:
    import synthgen
    import paper_1808_05056_b200 as H
    ap = argparse.ArgumentParser()
    ap.add_argument("--budget", type=int, default=1 << 20)
    ap.add_argument("--sizes", default=",".join(str(n) for n in DEFAULT_SIZES))
    ap.add_argument("--reps", type=int, default=8, help="timed calls per size and mode (the first two are discarded)")
    ap.add_argument("--alpha", type=float, default=1.0)
    ap.add_argument("--beta", type=float, default=0.5)
    ap.add_argument("--out", default="")
    args = ap.parse_args()
    ctx = H.hclooc_ctx_create(0)
    rows = []
    try:
        for n in sorted(int(x) for x in args.sizes.split(",")):
            A, B, C = H.HostMatrix(n, n), H.HostMatrix(n, n), H.HostMatrix(n, n)
            for X, name in ((A, "A"), (B, "B"), (C, "C")):
                synthgen.fill(X.array, synthgen.BASE_SEED + 1, name, "uniform")
            rec = {"N": n, "budget_bytes": args.budget, "flops": 2.0 * n ** 3}
            for label, mode in (("staged", 0), ("direct", 1), ("auto", -1)):
                H.hclooc_ctx_set_direct(ctx, mode)
                ts, st = [], None
                for _ in range(max(3, args.reps)):
                    st = H.hclooc_dgemm_ex(ctx, n, n, n, args.alpha, A, n, B, n, args.beta, C, n, args.budget)
                    ts.append(st.t_total_s)
                t = float(np.median(ts[2:]))
                rec[label] = {"t_ms": 1e3 * t, "tflops": 2.0 * n ** 3 / t / 1e12, "direct": int(st.plan.direct), "steps": int(st.plan.n_steps),
                              "copies": int(st.n_copies_h2d + st.n_copies_d2h), "h2d_MB": st.bytes_h2d / 1e6, "d2h_MB": st.bytes_d2h / 1e6,
                              "model_ms": 1e3 * st.plan.t_model_s, "link_GBps": (st.bytes_h2d + st.bytes_d2h) / t / 1e9}
            rows.append(rec)
            print(json.dumps(rec), flush=True)
            for X in (A, B, C):
                X.free()
    finally:
        H.hclooc_ctx_destroy(ctx)
    lines = ["| N | staged ms (steps, copies; model) | direct ms (MB read over the link; model) | auto picks | direct / staged speed |",
             "|---|---|---|---|---|"]
    for r in rows:
        s, d, a = r["staged"], r["direct"], r["auto"]
        lines.append(f"| {r['N']} | {s['t_ms']:.3f} ({s['steps']}, {s['copies']}; {s['model_ms']:.3f}) | {d['t_ms']:.3f} ({d['h2d_MB']:.1f}; {d['model_ms']:.3f}) | "
                     f"{'direct' if a['direct'] else 'staged'} ({a['t_ms']:.3f} ms) | {s['t_ms'] / d['t_ms']:.2f} |")
    table = "\n".join(lines)
    print(table)
    if args.out:
        with open(args.out, "w") as f:
            f.write(table + "\n\n" + "\n".join(json.dumps(r) for r in rows) + "\n")


if __name__ == "__main__":
    main()
