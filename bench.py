#!/usr/bin/env python
"""bench.py -- end-to-end out-of-core DGEMM TFLOP/s on one B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path (S0 validate, S1 plan, S2-S4 uploads, S5 DGEMM tile kernel,
S6 download, S7 events) over one synthetic problem: hclooc_dgemm(M,N,K,alpha,A,lda,B,ldb,beta,C,ldc,budget).

  value : the same call with A, B, C already resident in HBM (device pointers): the library's in-core case,
          one DGEMM launch on the caller's matrices with nothing staged, i.e. whole-job
          throughput with inputs resident when the timed region starts.
  e2e   : the same call through the C ABI with pinned HOST buffers (the product path): host->device and
          device->host copies inside the timed region.  Its roofline is max(flops / FP64 peak, link time).
  roofline : the FP64 DMMA kernel timed alone with CUDA events on its launch stream at a GPU-filling launch of the
          plan's B-slice shape (M x nb x K; hclDgemmAsync picks the persistent stream-K variant for it);
          `pipeline_step` inside it is one step of the plan launched exactly as the pipeline launches it
          (mb x nb x K with plan.ksplit CTAs per tile), against the peak of the SMs that launch occupies.
  cpu_baseline : the oracle, as it stands, on the host cores, on a bounded row sample of the same workload.

`--impl reference` times the oracle (the reference arm of this tier).  Under torchrun the problem grows to
world*M rows cut into one row band of C per GPU (independent bands, B on every rank, no collective: weak
scaling).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

MiB, GiB = 1 << 20, 1 << 30
# BASELINE.json configs (index = position in the list); cfg2 (index 1) is the one the metric is quoted on.
WORKLOADS = {
    "cfg1": dict(M=512, N=512, K=512, alpha=1.0, beta=0.5, budget=1 * MiB, dist="uniform", seed_idx=1,
                 desc="512^3 FP64, budget 1 MiB"),
    "cfg2": dict(M=8192, N=8192, K=8192, alpha=1.0, beta=1.0, budget=256 * MiB, dist="uniform", seed_idx=2,
                 desc="8192^3 FP64, alpha=1 beta=1, budget 256 MiB"),
    "cfg3": dict(M=32768, N=32768, K=32768, alpha=1.0, beta=0.0, budget=4 * GiB, dist="uniform", seed_idx=3,
                 desc="32768^3 FP64, beta=0, budget 4 GiB"),
    "cfg4": dict(M=65536, N=65536, K=16384, alpha=2.0, beta=-1.0, budget=16 * GiB, dist="normal", seed_idx=4,
                 desc="65536x65536x16384 FP64, alpha=2 beta=-1, budget 16 GiB"),
}
FP64_PEAK_TFLOPS = 37.2   # 148 SMs x 4 SMSPs x 32 flop/clk (DMMA.8x8x4: 512 flop / 16 clk) x 1.965 GHz; measured 37.17
# fallback (the first box probed, profiles/r01_box_probe.md); bench.py measures the link of the box it runs on (measure_link)
LINK = dict(h2d_GBps=55.5, d2h_GBps=51.5, duplex_GBps=88.0, source="profiles/r01_box_probe.md")


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.rows, self.proc, self.gpu = [], None, gpu_index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            self.proc.terminate()
            self.t.join(timeout=2)

    def summary(self):
        t0 = time.time()
        while self.proc and not self.rows and time.time() - t0 < 3.0:      # a run shorter than the first sample (config 1)
            time.sleep(0.05)
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        reasons = set()
        for r in self.rows:
            if len(r) >= 7:
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def ncu_traffic(launch):
    """dram__bytes_read.sum + dram__bytes_write.sum of the roofline-leg launch from the committed ncu capture
    (profiles/r01_traffic.json, written from `ncu --set full`), or None if that capture is of another launch."""
    try:
        with open(os.path.join(ROOT, "profiles", "r01_traffic.json")) as f:
            t = json.load(f)
        return t["dram_bytes"] if t.get("launch") == launch else None
    except (OSError, ValueError, KeyError):
        return None


def measure_link(H, total=1 << 30, chunk=256 << 20):
    """Host-link peaks of THIS box, measured through the library's runtime calls right before the timed legs (boxes of the
    pool differ: 51.5-57 GB/s D2H, 88-100 GB/s duplex): pinned 256 MiB copies, each direction alone and both at once."""
    try:
        host_a, host_b = H.hclooc_host_alloc(total), H.hclooc_host_alloc(total)
        dev_a, dev_b = H.hclMalloc(total), H.hclMalloc(total)
        s0, s1 = H.hclStreamCreate(), H.hclStreamCreate()
    except Exception:
        return None

    def run(up, down):
        for off in range(0, total, chunk):
            if up:
                H.hclMemcpyAsync(dev_a + off, host_a + off, chunk, H.HCL_H2D, s0)
            if down:
                H.hclMemcpyAsync(host_b + off, dev_b + off, chunk, H.HCL_D2H, s1)
        H.hclStreamSynchronize(s0); H.hclStreamSynchronize(s1)

    out = {}
    for key, up, down in (("h2d_GBps", True, False), ("d2h_GBps", False, True), ("duplex_GBps", True, True)):
        run(up, down)
        best = 0.0
        for _ in range(2):
            t0 = time.perf_counter()
            run(up, down)
            best = max(best, (int(up) + int(down)) * total / (time.perf_counter() - t0) / 1e9)
        out[key] = best
    for p in (dev_a, dev_b):
        H.hclFree(p)
    for p in (host_a, host_b):
        H.hclooc_host_free(p)
    for s in (s0, s1):
        H.hclStreamDestroy(s)
    out["source"] = "measured live on this box (1 GiB in 256 MiB pinned copies per direction, best of 2)"
    return out


def link_roofline_s(flops, bytes_h2d, bytes_d2h):
    """Lower bound on the time of the host-resident path: FP64 at peak vs the scheduler's actual bytes
    at the measured link rates (each direction alone, and their sum at the duplex rate)."""
    t_flop = flops / (FP64_PEAK_TFLOPS * 1e12)
    t_link = max(bytes_h2d / (LINK["h2d_GBps"] * 1e9), bytes_d2h / (LINK["d2h_GBps"] * 1e9),
                 (bytes_h2d + bytes_d2h) / (LINK["duplex_GBps"] * 1e9))
    return max(t_flop, t_link), t_flop, t_link


def oracle_sample(wl, rows, seed):
    """Inputs for the oracle on a bounded sample: the first `rows` rows of C (all N columns, whole K)."""
    import synthgen
    M, N, K = rows, wl["N"], wl["K"]
    A = synthgen.fill(np.empty((M, K)), seed, "A", wl["dist"], logical_cols=K)
    B = synthgen.fill(np.empty((K, N)), seed, "B", wl["dist"])
    C = synthgen.fill(np.empty((M, N)), seed, "C", wl["dist"], logical_cols=N)
    return A, B, C


def time_oracle(wl, rows, seed, steps, warmup):
    import oracle
    A, B, C = oracle_sample(wl, rows, seed)
    times = []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        oracle.dgemm(wl["alpha"], A, B, wl["beta"], C)
        dt = time.perf_counter() - t0
        if it >= warmup:
            times.append(dt)
    flops = 2.0 * rows * wl["N"] * wl["K"]
    return flops, times


def run_reference(args, wl, name):
    """Reference arm of this tier: the CPU oracle, as it stands, on the host cores."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cores = os.cpu_count() or 1
    rows = min(wl["M"], max(32, args.ref_rows))
    flops, times = time_oracle(wl, rows, 180805056 + wl["seed_idx"], args.steps, max(1, min(args.warmup, 1)))
    ms = 1e3 * float(np.mean(times))
    val = flops / (ms * 1e-3) / 1e12
    sample = f"first {rows} rows of C (all {wl['N']} columns, K={wl['K']}) per step, oracle.dgemm, OpenMP"
    out = {"impl": "reference", "metric": "end-to-end out-of-core DGEMM TFLOP/s (host-resident A,B,C)", "value": val,
           "unit": "TFLOP/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": f"{name}: {wl['desc']}", "sample": sample},
           "cpu_baseline": {"value": val, "unit": "TFLOP/s", "cores": cores, "kind": "oracle", "sample": sample},
           "e2e": {"value": val, "unit": "TFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


def run_ours(args, wl, name):
    import torch
    import synthgen
    import paper_1808_05056_b200 as H
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback for the product path")
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    M, N, K, alpha, beta, budget = wl["M"], wl["N"], wl["K"], wl["alpha"], wl["beta"], wl["budget"]
    seed = synthgen.BASE_SEED + wl["seed_idx"]
    flops = 2.0 * M * N * K
    # N > 1: ONE problem of world*M rows cut into row bands of C (hclooc_shard_rows): rank r owns rows r*M .. of A
    # and C, every rank holds all of B; the bands are independent, so no collective is on
    # the data path and per-GPU work is fixed as N grows (weak scaling).
    row0, rows = H.hclooc_shard_rows(world * M, world, rank, 128)
    assert (row0, rows) == (rank * M, M) or M % 128

    # ---- inputs: pinned host matrices (the product path) and HBM-resident copies (the `value` leg)
    A, B, C = H.HostMatrix(M, K), H.HostMatrix(K, N), H.HostMatrix(M, N)
    synthgen.fill(A.array, seed, "A", wl["dist"], row0=rank * M); synthgen.fill(B.array, seed, "B", wl["dist"])
    synthgen.fill(C.array, seed, "C", wl["dist"], row0=rank * M)
    dA, dB, dC = (torch.from_numpy(X.array).cuda() for X in (A, B, C))
    torch.cuda.synchronize()      # the library's streams do not wait for PyTorch's: device operands must be complete

    # ---- PyTorch owns device memory and streams; the library carves its buffers from this workspace
    ws = torch.empty(budget, dtype=torch.uint8, device="cuda")
    streams = [torch.cuda.Stream() for _ in range(10)]
    ctx = H.hclooc_ctx_create(local, ws, ws.numel(), streams[0], streams[1], streams[2:])

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def ci95_rel(xs):
        """Half-width of the 95 % confidence interval of the mean over the mean (Student t; PAPER.md:362 asks
        for 2.5 %)."""
        n = len(xs)
        if n < 2:
            return None
        t95 = {2: 12.71, 3: 4.303, 4: 3.182, 5: 2.776, 6: 2.571, 7: 2.447, 8: 2.365, 9: 2.306, 10: 2.262}.get(n, 2.0 if n > 30 else 2.2)
        return float(t95 * np.std(xs, ddof=1) / np.sqrt(n) / np.mean(xs))

    per_call = []

    def timed(fn, steps, warmup):
        st = None
        per_call.clear()
        for _ in range(warmup):
            st = fn()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            st = fn()
            per_call.append(st.t_total_s)
        e1.record()
        barrier()
        ms = e0.elapsed_time(e1)
        if world > 1:
            t = torch.tensor([ms], device="cuda", dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        return ms / steps, (st, ci95_rel(list(per_call)), 1e3 * float(np.mean(per_call)), 1e3 * float(np.min(per_call)))

    def resident():
        if ta or tb:
            return H.hclooc_dgemm_t(ctx, ta, tb, M, N, K, alpha, dA, M if ta else K, dB, K if tb else N, beta, dC, N, budget)
        return H.hclooc_dgemm_ex(ctx, M, N, K, alpha, dA, K, dB, N, beta, dC, N, budget)

    ta, tb = int(args.trans[0] == "T"), int(args.trans[1] == "T")

    def host():
        if ta or tb:     # the M*K (K*N) doubles of A (B) read as the stored K x M (N x K) matrix
            return H.hclooc_dgemm_t(ctx, ta, tb, M, N, K, alpha, A, M if ta else K, B, K if tb else N, beta, C, C.ld, budget)
        return H.hclooc_dgemm_ex(ctx, M, N, K, alpha, A, A.ld, B, B.ld, beta, C, C.ld, budget)

    if not args.kernel_only:
        live = measure_link(H)
        if live:
            LINK.update(live)
    with ClockSampler(local) as clk:
        if args.kernel_only:
            plan = H.hclooc_plan(M, N, K, beta != 0.0, 0, budget)
        else:
            ms_res, (st_res, ci_res, _, _) = timed(resident, args.steps, max(args.warmup, 3))
            ms_e2e, (st_e2e, ci_e2e, call_mean_ms, call_min_ms) = timed(host, args.steps, max(args.warmup, 3))
            plan = st_e2e.plan
        # ---- roofline leg: the tile kernel alone, one GPU-filling launch of the plan's B-slice shape
        nb = min(plan.nb, N)
        cur = torch.cuda.current_stream()
        kt = []
        for it in range(max(args.warmup, 3) + args.steps):
            k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            k0.record(cur)
            if ta or tb:
                H.hclDgemmAsyncT(ta, tb, M, nb, K, alpha, dA, M if ta else K, dB, K if tb else N, beta, dC, N, cur)
            else:
                H.hclDgemmAsync(M, nb, K, alpha, dA, K, dB, N, beta, dC, N, cur)
            k1.record(cur)
            k1.synchronize()
            if it >= max(args.warmup, 3):
                kt.append(k0.elapsed_time(k1))
        # ---- one pipeline step, launched as the executor launches it (it need not fill the GPU: steps overlap)
        mb = min(plan.mb, M)
        stt = []
        for it in range(max(args.warmup, 3) + max(args.steps, 10)):
            k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            k0.record(cur)
            H.hclDgemmAsyncT(ta, tb, mb, nb, K, alpha, dA, M if ta else K, dB, K if tb else N, beta, dC, N, cur, variant=max(1, plan.ksplit))
            k1.record(cur)
            k1.synchronize()
            if it >= max(args.warmup, 3):
                stt.append(k0.elapsed_time(k1))
        clocks = clk.summary()
    ms_step = float(np.mean(stt))
    step_ctas = min(148, -(-mb // 128) * -(-nb // 128) * max(1, plan.ksplit))
    step_achieved = 2.0 * mb * nb * K / (ms_step * 1e-3) / 1e12
    step_peak = FP64_PEAK_TFLOPS * step_ctas / 148.0
    ms_kernel = float(np.mean(kt))
    kflops = 2.0 * M * nb * K
    achieved = kflops / (ms_kernel * 1e-3) / 1e12
    if args.kernel_only:
        if rank == 0:
            print(json.dumps({"kernel_only": True, "launch": f"{M}x{nb}x{K}", "ms_per_launch": ms_kernel, "achieved_tflops": achieved,
                              "frac": achieved / FP64_PEAK_TFLOPS, "clocks": clocks}))
        H.hclooc_ctx_destroy(ctx)
        return

    t_roof, t_flop, t_link = link_roofline_s(flops, st_e2e.bytes_h2d, st_e2e.bytes_d2h)
    out = {
        "metric": "end-to-end out-of-core DGEMM TFLOP/s (host-resident A,B,C) and % of roofline",
        "value": world * flops / (ms_res * 1e-3) / 1e12, "unit": "TFLOP/s", "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_res, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "ci95_rel": ci_res,
        "config": {"workload": f"{name}: {wl['desc']}", "M": M, "N": N, "K": K, "alpha": alpha, "beta": beta,
                   "device_budget_bytes": budget, "dist": wl["dist"], "trans": args.trans, "parallelism": (f"{world} row bands of C of {M} rows each, one per GPU (hclooc_shard_rows), B on every rank, no collective"
                                   if world > 1 else "1 GPU"), "M_global": world * M,
                   "plan": {k: getattr(plan, k) for k in ("mb", "nb", "kb", "h", "w", "kpanels", "n_steps", "n_sets", "n_bbuf", "workspace_bytes")},
                   "l2": "inputs (A+B+C = %.2f GB) exceed the 126 MB L2; no flush needed" % ((M * K + K * N + M * N) * 8 / 1e9),
                   "value_leg": "A,B,C resident in HBM: in-core case, one tile-kernel launch over the whole problem, nothing staged"},
        "e2e": {"value": world * flops / (ms_e2e * 1e-3) / 1e12, "unit": "TFLOP/s", "ms_per_step": ms_e2e,
                "h2d_bytes_per_step": int(st_e2e.bytes_h2d), "d2h_bytes_per_step": int(st_e2e.bytes_d2h),
                "roofline_s": t_roof, "t_flop_s": t_flop, "t_link_s": t_link, "bound": "link" if t_link > t_flop else "fp64",
                "frac_of_roofline": t_roof / (ms_e2e * 1e-3), "link_peaks": LINK, "ci95_rel": ci_e2e,
                "call_ms_mean": call_mean_ms, "call_ms_min": call_min_ms},
        "gpu_launches": int((st_res.n_kernels + st_e2e.n_kernels) * args.steps + len(kt) + len(stt)),
        "clocks": clocks,
        "roofline": {"bound": "alu", "achieved": achieved, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s",
                     "frac": achieved / FP64_PEAK_TFLOPS, "traffic": ncu_traffic(f"{M}x{nb}x{K}"),
                     "kernel": "hclooc_dgemm_streamk_kernel" if -(-M // 128) * -(-nb // 128) >= 148 else "hclooc_dgemm_tile_kernel",
                     "launch": f"{M}x{nb}x{K} (one B slice of the plan, all rows)", "ms_per_launch": ms_kernel,
                     "peak_source": "derived 148 SM x 128 FP64 flop/clk x 1.965 GHz; DMMA microbenchmark measured 37.17",
                     "pipeline_step": {"kernel": f"hclooc_dgemm_tile_kernel<{max(1, plan.ksplit)}>", "launch": f"{mb}x{nb}x{K}",
                                       "ctas": step_ctas, "ms_per_launch": ms_step, "achieved": step_achieved,
                                       "peak": step_peak, "frac": step_achieved / step_peak,
                                       "note": "peak = 37.2 TFLOP/s x CTAs/148: a step occupies only its own CTAs, other steps run beside it"}},
    }
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        rows = min(M, args.cpu_rows if args.cpu_rows > 0 else max(128, int(1.0e12 / (2.0 * N * K)) // 128 * 128))
        cflops, times = time_oracle(wl, rows, seed, 1, 0)
        out["cpu_baseline"] = {"value": cflops / times[0] / 1e12, "unit": "TFLOP/s", "cores": os.cpu_count(), "kind": "oracle",
                               "sample": f"first {rows} rows of C (all {N} columns, K={K}), {times[0]:.1f} s of oracle.dgemm"}
    H.hclooc_ctx_destroy(ctx)
    if world > 1:
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=sorted(WORKLOADS))
    ap.add_argument("--ref-rows", type=int, default=512, help="rows of C per oracle step (reference arm)")
    ap.add_argument("--cpu-rows", type=int, default=0, help="rows of C in the cpu_baseline sample (0 = about 1e12 flop, 10-30 s)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--trans", default="NN", choices=["NN", "TN", "NT", "TT"],
                    help="e2e leg through hclooc_dgemm_t with op(A), op(B) transposed (the same buffers read as the stored K x M / N x K matrices)")
    ap.add_argument("--kernel-only", action="store_true", help="only the roofline leg (for ncu captures of the tile kernel)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    wl, name = WORKLOADS[args.workload], args.workload
    if args.impl == "reference":
        return run_reference(args, wl, name)
    run_ours(args, wl, name)


if __name__ == "__main__":
    main()
