"""Measures, through the library's own runtime calls, the machine figures the planner's cost model and bench.py's
roofline use (DESIGN.md sections 6, 7, 10; `machine_model()` in csrc/planner.cpp; FP64_PEAK_TFLOPS and LINK in bench.py):

  * FP64 issue rate of register-resident DMMA (mma.sync.m8n8k4.f64) and DFMA chains  -- hclooc_probe_fp64
  * host link: pinned H2D and D2H copies alone at several chunk sizes, both directions at once, and 2-D (strided)
    copies at several row widths                                                      -- hclMemcpyAsync / hclMemcpy2DAsync

    python -m paper_1808_05056_b200.box_probe [--out FILE]

Prints a Markdown table (also written to --out).
"""
from __future__ import annotations

import argparse
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

MiB = 1 << 20


def main() -> None:
    import paper_1808_05056_b200 as H
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default="")
    ap.add_argument("--total-mib", type=int, default=2048, help="bytes moved per link measurement")
    args = ap.parse_args()
    rows = []

    for kind, name in ((0, "FP64 DMMA (mma.sync.m8n8k4.f64 -> DMMA.8x8x4), register chains"), (1, "FP64 DFMA, 16 chains per thread")):
        vals = [H.hclooc_probe_fp64(kind, c, 1.0) for c in (1, 2, 4)]
        rows.append((name, " / ".join(f"{v:.2f}" for v in vals) + " TFLOP/s at 1 / 2 / 4 CTAs of 256 threads per SM"))

    total = args.total_mib * MiB
    host_a, host_b = H.hclooc_host_alloc(total), H.hclooc_host_alloc(total)
    dev_a, dev_b = H.hclMalloc(total), H.hclMalloc(total)
    s0, s1 = H.hclStreamCreate(), H.hclStreamCreate()

    def rate(fn, nbytes):
        fn()                                   # warm-up
        H.hclStreamSynchronize(s0); H.hclStreamSynchronize(s1)
        t0 = time.perf_counter()
        fn()
        H.hclStreamSynchronize(s0); H.hclStreamSynchronize(s1)
        return nbytes / (time.perf_counter() - t0) / 1e9

    def chunks(direction, stream, chunk, host, dev):
        def run():
            for off in range(0, total, chunk):
                if direction == H.HCL_H2D:
                    H.hclMemcpyAsync(dev + off, host + off, chunk, H.HCL_H2D, stream)
                else:
                    H.hclMemcpyAsync(host + off, dev + off, chunk, H.HCL_D2H, stream)
        return run

    sizes = (64 * 1024, 1 * MiB, 8 * MiB, 256 * MiB)
    h2d = [rate(chunks(H.HCL_H2D, s0, c, host_a, dev_a), total) for c in sizes]
    d2h = [rate(chunks(H.HCL_D2H, s0, c, host_a, dev_a), total) for c in sizes]
    label = " / ".join("64 KiB" if c < MiB else f"{c // MiB} MiB" for c in sizes)
    rows.append(("H2D, pinned, 1-D copies back to back", " / ".join(f"{v:.1f}" for v in h2d) + f" GB/s at {label} chunks"))
    rows.append(("D2H, pinned, 1-D copies back to back", " / ".join(f"{v:.1f}" for v in d2h) + f" GB/s at {label} chunks"))

    def both():
        chunks(H.HCL_H2D, s0, 256 * MiB, host_a, dev_a)()
        chunks(H.HCL_D2H, s1, 256 * MiB, host_b, dev_b)()
    duplex = rate(both, 2 * total)
    rows.append(("both directions at once (256 MiB chunks, two streams)", f"{duplex:.1f} GB/s in total, {duplex / 2:.1f} per direction"))

    # 2-D copies: rows of `width` bytes out of a host matrix whose pitch is 64 KiB (an 8192-column FP64 matrix)
    pitch = 64 * 1024
    nrows = total // pitch
    for direction, name in ((H.HCL_H2D, "H2D"), (H.HCL_D2H, "D2H")):
        vals = []
        widths = (128, 1024, 2048, 4096, 16384)
        for w in widths:
            def run(w=w):
                if direction == H.HCL_H2D:
                    H.hclMemcpy2DAsync(dev_a, w, host_a, pitch, w, nrows, H.HCL_H2D, s0)
                else:
                    H.hclMemcpy2DAsync(host_a, pitch, dev_a, w, w, nrows, H.HCL_D2H, s0)
            vals.append(rate(run, w * nrows))
        rows.append((f"{name}, 2-D copy of {nrows} rows, host pitch 64 KiB", " / ".join(f"{v:.1f}" for v in vals) + " GB/s at row widths " +
                     " / ".join(f"{w} B" if w < 1024 else f"{w // 1024} KiB" for w in widths)))

    for p in (dev_a, dev_b):
        H.hclFree(p)
    for p in (host_a, host_b):
        H.hclooc_host_free(p)
    for s in (s0, s1):
        H.hclStreamDestroy(s)

    lines = ["| quantity | measured |", "|---|---|"] + [f"| {a} | {b} |" for a, b in rows]
    table = "\n".join(lines)
    print(table)
    if args.out:
        with open(args.out, "w") as f:
            f.write(table + "\n")


if __name__ == "__main__":
    main()
