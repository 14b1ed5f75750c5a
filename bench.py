#!/usr/bin/env python
"""bench.py -- end-to-end out-of-core DGEMM TFLOP/s on one B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path (S0 validate, S1 plan, S2-S4 uploads, S5 DGEMM tile kernel,
S6 download, S7 events) over one synthetic problem: hclooc_dgemm(M,N,K,alpha,A,lda,B,ldb,beta,C,ldc,budget)
with A, B, C in pinned HOST memory.

Workload (`--workload auto`, the default): the LARGEST configuration the host can pin -- BASELINE.json
configs[4] (beyond-HBM: M = N = 163840, K = 8192, budget = all free HBM) scaled to this host's memory
("cfg5s": M = N = 147456 on a 196 GiB host, A+B+C = 193 GB > the GPU's memory), else configs[3], [2], [1].

  value : device-timed (CUDA events around the K calls) throughput of that call.  Nothing of such a problem can
          be resident in HBM, so the timed region is the host-resident call itself.
  e2e   : the same K calls timed by the host clock (call entry to return, G16), with the scheduler's actual
          host<->device bytes; its roofline is max(flops / FP64 peak, link time at the link rates measured
          on this box right before).
  in_core : the library's in-core case (all three operands device-resident: one stream-K launch, nothing
          staged) on a problem that fits -- the kernel-only rate, NOT the metric.
  per_config : BASELINE configs[0..3] (cfg1-cfg4) end to end in the same run, each with its bytes, bound,
          fraction of its roofline and plan.
  roofline : the FP64 DMMA tile kernel AS THE PIPELINE LAUNCHES IT: a traced call brackets every kernel with
          events on its own compute stream; achieved = flops of all launches / time during which at least one
          of them was running.  `solo_step` is one step's launch timed alone, `streamk` a GPU-filling launch of
          the persistent kernel; `peak_measured` is hclooc_probe_fp64 run live.
  cpu_baseline : the oracle, as it stands, on the host cores, on a bounded sample of the same workload.

`--impl reference` times the oracle (the reference arm of this tier) under the same metric string and
workload name.  Under torchrun the problem grows to world*M rows cut into one row band of C per GPU
(independent bands, B on every rank, no collective: weak scaling).
`--op dsyrk|dtrsm|dpotrf|dgetrf` (and the `_dev` device phases) and `--sweep transition` time the other product paths (one JSON line each).
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
METRIC = "end-to-end out-of-core DGEMM TFLOP/s (host-resident A,B,C) and % of roofline"
# BASELINE.json configs (index + 1 = cfg number); budget 0 = all free HBM
WORKLOADS = {
    "cfg1": dict(M=512, N=512, K=512, alpha=1.0, beta=0.5, budget=1 * MiB, dist="uniform", seed_idx=1,
                 desc="512^3 FP64, alpha=1 beta=0.5, budget 1 MiB"),
    "cfg2": dict(M=8192, N=8192, K=8192, alpha=1.0, beta=1.0, budget=256 * MiB, dist="uniform", seed_idx=2,
                 desc="8192^3 FP64, alpha=1 beta=1, budget 256 MiB"),
    "cfg3": dict(M=32768, N=32768, K=32768, alpha=1.0, beta=0.0, budget=4 * GiB, dist="uniform", seed_idx=3,
                 desc="32768^3 FP64, beta=0, budget 4 GiB"),
    "cfg4": dict(M=65536, N=65536, K=16384, alpha=2.0, beta=-1.0, budget=16 * GiB, dist="normal", seed_idx=4,
                 desc="65536x65536x16384 FP64, alpha=2 beta=-1, budget 16 GiB"),
}
FP64_PEAK_TFLOPS = 37.2   # 148 SMs x 4 SMSPs x 32 flop/clk (DMMA.8x8x4: 512 flop / 16 clk) x 1.965 GHz
# fallback (the first box probed, profiles/r01_box_probe.md); bench.py measures the link of the box it runs on (measure_link)
LINK = dict(h2d_GBps=55.5, d2h_GBps=51.5, duplex_GBps=88.0, source="profiles/r01_box_probe.md")


def meminfo(key):
    with open("/proc/meminfo") as f:
        for line in f:
            if line.startswith(key + ":"):
                return int(line.split()[1]) * 1024
    return 0


def wl_bytes(wl):
    return 8 * (wl["M"] * wl["K"] + wl["K"] * wl["N"] + wl["M"] * wl["N"])


def cfg5_scaled(share=1):
    """BASELINE configs[4] (M = N = 163840, K = 8192, alpha 1, beta 0.5, budget = all free HBM: 236 GB pinned) scaled to
    this host: the largest M = N (a multiple of 2048, at most 163840) whose three matrices leave 14 GiB of the host's
    memory (MemTotal / share, share = ranks on this node) unpinned.  MemTotal, not MemAvailable, so that both arms of a
    run pick the same size."""
    room = meminfo("MemTotal") // share - 14 * GiB
    K, n = 8192, 163840
    while n > 2048 and 8 * (n * n + 2 * n * K) > room:
        n -= 2048
    return dict(M=n, N=n, K=K, alpha=1.0, beta=0.5, budget=0, dist="uniform", seed_idx=5,
                desc=f"{n}x{n}x{K} FP64, alpha=1 beta=0.5, budget = all free HBM (BASELINE configs[4] scaled to this host's memory)")


def pick_workload(name, share=1):
    """`auto`: the largest configuration whose matrices this host can pin (per rank)."""
    if name != "auto":
        return (name, cfg5_scaled(share)) if name == "cfg5s" else (name, WORKLOADS[name])
    room = meminfo("MemTotal") // share - 14 * GiB
    s5 = cfg5_scaled(share)
    if s5["M"] > 65536 and wl_bytes(s5) <= room:
        return "cfg5s", s5
    for cand in ("cfg4", "cfg3", "cfg2"):
        if wl_bytes(WORKLOADS[cand]) <= room:
            return cand, WORKLOADS[cand]
    return "cfg1", WORKLOADS["cfg1"]


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


def ncu_traffic(kernel, launch):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` capture of that kernel at
    that launch shape (profiles/traffic.json, one entry per captured launch), or None when no capture matches."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            for t in json.load(f)["captures"]:
                if t.get("launch") == launch and t.get("kernel") == kernel:
                    return t["dram_bytes"], t.get("source")
    except (OSError, ValueError, KeyError):
        pass
    return None, None


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


def ci95_rel(xs):
    """Half-width of the 95 % confidence interval of the mean over the mean (Student t; PAPER.md:362 asks for 2.5 %)."""
    n = len(xs)
    if n < 2:
        return None
    t95 = {2: 12.71, 3: 4.303, 4: 3.182, 5: 2.776, 6: 2.571, 7: 2.447, 8: 2.365, 9: 2.306, 10: 2.262}.get(n, 2.0 if n > 30 else 2.2)
    return float(t95 * np.std(xs, ddof=1) / np.sqrt(n) / np.mean(xs))


# ---------------------------------------------------------------------------------------------- the oracle legs
def oracle_sample_shape(wl, flops_target, rows=512):
    """A bounded sample of the workload for the oracle: the first `rows` rows (32-row blocks x the OpenMP threads) and as many
    leading columns of C as make about `flops_target` flops, whole K."""
    rows = min(wl["M"], rows)
    cols = int(flops_target / (2.0 * rows * wl["K"])) // 128 * 128
    cols = min(wl["N"], max(128, cols))
    return rows, cols


def time_oracle(wl, rows, cols, seed, steps, warmup, mats=None):
    """oracle.dgemm on C[:rows, :cols] = alpha * A[:rows] * B[:, :cols] + beta * C[:rows, :cols]; `mats` = (A, B, C) numpy views
    of the workload's host matrices when the caller has them, else the sample is generated (same seeds, same elements)."""
    import oracle
    import synthgen
    K = wl["K"]
    if mats is None:
        A = synthgen.fill(np.empty((rows, K)), seed, "A", wl["dist"], logical_cols=K)
        B = synthgen.fill(np.empty((K, cols)), seed, "B", wl["dist"], logical_cols=wl["N"])
        C = synthgen.fill(np.empty((rows, cols)), seed, "C", wl["dist"], logical_cols=wl["N"])
    else:
        A, B, C = mats[0][:rows], mats[1][:, :cols], mats[2][:rows, :cols].copy()
    times = []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        oracle.dgemm(wl["alpha"], A, B, wl["beta"], C)
        dt = time.perf_counter() - t0
        if it >= warmup:
            times.append(dt)
    return 2.0 * rows * cols * K, times


def run_reference(args):
    """Reference arm of this tier: the CPU oracle, as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    share = int(os.environ.get("LOCAL_WORLD_SIZE", os.environ.get("WORLD_SIZE", "1")))
    name, wl = pick_workload(args.workload, share)
    cores = os.cpu_count() or 1
    rows, cols = oracle_sample_shape(wl, args.ref_flops, args.ref_rows)
    steps = args.steps if args.steps else 5
    flops, times = time_oracle(wl, rows, cols, 180805056 + wl["seed_idx"], steps, args.warmup)
    ms = 1e3 * float(np.mean(times))
    val = flops / (ms * 1e-3) / 1e12
    sample = f"first {rows} rows x first {cols} columns of C (K={wl['K']}) per step, oracle.dgemm, OpenMP"
    out = {"impl": "reference", "metric": METRIC, "value": val,
           "unit": "TFLOP/s", "n_gpus": args.gpus, "steps": steps, "warmup": args.warmup, "ms_per_step": ms,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": f"{name}: {wl['desc']}", "sample": sample},
           "cpu_baseline": {"value": val, "unit": "TFLOP/s", "cores": cores, "kind": "oracle", "sample": sample},
           "e2e": {"value": val, "unit": "TFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


# ---------------------------------------------------------------------------------------------- our arm
class Bench:
    def __init__(self, args):
        import torch
        import synthgen
        import paper_1808_05056_b200 as H
        self.torch, self.synthgen, self.H, self.args = torch, synthgen, H, args
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        self.share = int(os.environ.get("LOCAL_WORLD_SIZE", str(self.world)))
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback for the product path")
        torch.cuda.set_device(self.local)
        self.dist = None
        if self.world > 1:
            import torch.distributed as dist
            dist.init_process_group("nccl", device_id=torch.device("cuda", self.local))
            self.dist = dist
        self.ta, self.tb = int(args.trans[0] == "T"), int(args.trans[1] == "T")

    def barrier(self):
        if self.dist:
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def make_ctx(self, budget):
        """PyTorch owns device memory and streams; the library carves its buffers from this workspace.  budget 0 = all free
        HBM (less 2 GiB for the CUDA context and whatever else lives on the device)."""
        torch = self.torch
        if budget == 0:
            torch.cuda.empty_cache()
            free, _ = torch.cuda.mem_get_info()
            budget = int(free) - 2 * GiB
        ws = torch.empty(budget, dtype=torch.uint8, device="cuda")
        streams = [torch.cuda.Stream() for _ in range(10)]
        ctx = self.H.hclooc_ctx_create(self.local, ws, ws.numel(), streams[0], streams[1], streams[2:])
        return ctx, ws, streams, budget

    def host_matrices(self, wl, seed):
        H, sg = self.H, self.synthgen
        M, N, K = wl["M"], wl["N"], wl["K"]
        t0 = time.perf_counter()
        A, B, C = H.HostMatrix(M, K), H.HostMatrix(K, N), H.HostMatrix(M, N)
        t_pin = time.perf_counter() - t0
        sg.fill(A.array, seed, "A", wl["dist"], row0=self.rank * M); sg.fill(B.array, seed, "B", wl["dist"])
        sg.fill(C.array, seed, "C", wl["dist"], row0=self.rank * M)
        return A, B, C, t_pin

    def call(self, ctx, wl, A, B, C, budget):
        H, ta, tb = self.H, self.ta, self.tb
        M, N, K = wl["M"], wl["N"], wl["K"]
        if ta or tb:     # the M*K (K*N) doubles of A (B) read as the stored K x M (N x K) matrix
            return H.hclooc_dgemm_t(ctx, ta, tb, M, N, K, wl["alpha"], A, M if ta else K, B, K if tb else N, wl["beta"], C, N, budget)
        return H.hclooc_dgemm_ex(ctx, M, N, K, wl["alpha"], A, K, B, N, wl["beta"], C, N, budget)

    def timed(self, fn, steps, warmup):
        """W untimed calls, then exactly K calls between barrier + synchronize: device time from CUDA events (max over
        ranks), host wall time of the same region, and the per-call wall times the library reports (t_total_s)."""
        torch = self.torch
        st = None
        for _ in range(warmup):
            st = fn()
        self.barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        per_call = []
        e0.record()
        t0 = time.perf_counter()
        for _ in range(steps):
            st = fn()
            per_call.append(st.t_total_s)
        wall = time.perf_counter() - t0
        e1.record()
        self.barrier()
        ms = e0.elapsed_time(e1)
        if self.dist:
            t = torch.tensor([ms, wall * 1e3], device="cuda", dtype=torch.float64)
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
            ms, wall = float(t[0].item()), float(t[1].item()) * 1e-3
        return {"ms_events": ms / steps, "ms_wall": 1e3 * wall / steps, "stats": st, "ci95_rel": ci95_rel(per_call),
                "call_ms_mean": 1e3 * float(np.mean(per_call)), "call_ms_min": 1e3 * float(np.min(per_call))}

    def e2e_record(self, wl, r):
        st = r["stats"]
        flops = 2.0 * wl["M"] * wl["N"] * wl["K"]
        t_roof, t_flop, t_link = link_roofline_s(flops, st.bytes_h2d, st.bytes_d2h)
        return {"value": self.world * flops / (r["ms_wall"] * 1e-3) / 1e12, "unit": "TFLOP/s", "ms_per_step": r["ms_wall"],
                "h2d_bytes_per_step": int(st.bytes_h2d), "d2h_bytes_per_step": int(st.bytes_d2h),
                "roofline_s": t_roof, "t_flop_s": t_flop, "t_link_s": t_link, "bound": "link" if t_link > t_flop else "fp64",
                "frac_of_roofline": t_roof / (r["ms_wall"] * 1e-3), "ci95_rel": r["ci95_rel"],
                "call_ms_mean": r["call_ms_mean"], "call_ms_min": r["call_ms_min"],
                "timer": "host clock around the K calls (each returns with C complete in host memory)"}

    @staticmethod
    def plan_summary(plan):
        keys = ("mb", "nb", "kb", "h", "w", "kpanels", "n_steps", "n_sets", "n_abuf", "n_bbuf", "ksplit", "direct", "resident", "workspace_bytes")
        return {k: getattr(plan, k) for k in keys}

    def per_config(self, names):
        """BASELINE configs cfg1..cfg4 end to end, one after the other (each pins, runs and frees its own matrices)."""
        out = {}
        steps_of = {"cfg1": 50, "cfg2": 10, "cfg3": 3, "cfg4": 3}
        for name in names:
            wl = WORKLOADS[name]
            if wl_bytes(wl) + 8 * GiB > meminfo("MemAvailable"):
                out[name] = {"skipped": "host memory"}
                continue
            ctx, ws, streams, budget = self.make_ctx(wl["budget"])
            A, B, C, _ = self.host_matrices(wl, self.synthgen.BASE_SEED + wl["seed_idx"])
            try:
                # (config 1 is a 0.2 ms call: 200 untimed calls first, so that clocks and link are in the state a busy process sees)
                r = self.timed(lambda: self.call(ctx, wl, A, B, C, budget), steps_of[name], 200 if name == "cfg1" else 3)
                rec = self.e2e_record(wl, r)
                rec.update({"workload": f"{name}: {wl['desc']}", "steps": steps_of[name], "warmup": 3, "plan": self.plan_summary(r["stats"].plan)})
                for k in ("roofline_s", "call_ms_mean", "call_ms_min", "timer", "unit"):
                    rec.pop(k, None)
                out[name] = rec
            finally:
                self.H.hclooc_ctx_destroy(ctx)
                for X in (A, B, C):
                    X.free()
                del ws, streams
                self.torch.cuda.empty_cache()
        return out

    def kernel_legs(self, wl, plan, steps, warmup):
        """The tile kernel timed alone on device-resident operands of the plan's step shape: one step as the pipeline launches
        it (mb x nb x K, plan.ksplit CTAs per tile) and a GPU-filling launch (up to 16384 rows x nb x K: hclDgemmAsync picks the
        persistent stream-K variant).  Operands: seeded uniform[-1,1) generated on the device (values do not matter here)."""
        torch, H, ta, tb = self.torch, self.H, self.ta, self.tb
        M, N, K = wl["M"], wl["N"], wl["K"]
        if plan.direct:
            mb, nb = M, N
        else:
            mb, nb = min(plan.mb, M), min(plan.nb, N)
        rows = min(M, max(mb, 16384))
        g = torch.Generator(device="cuda"); g.manual_seed(180805056)
        dA = torch.rand((K, rows) if ta else (rows, K), generator=g, dtype=torch.float64, device="cuda") * 2 - 1
        dB = torch.rand((nb, K) if tb else (K, nb), generator=g, dtype=torch.float64, device="cuda") * 2 - 1
        dC = torch.rand((rows, nb), generator=g, dtype=torch.float64, device="cuda") * 2 - 1
        torch.cuda.synchronize()
        cur = torch.cuda.current_stream()
        lda, ldb = (rows if ta else K), (K if tb else nb)

        def time_launch(m, variant, n_iter):
            ts = []
            for it in range(warmup + n_iter):
                k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                k0.record(cur)
                H.hclDgemmAsyncT(ta, tb, m, nb, K, wl["alpha"], dA, lda, dB, ldb, wl["beta"], dC, nb, cur, variant=variant)
                k1.record(cur)
                k1.synchronize()
                if it >= warmup:
                    ts.append(k0.elapsed_time(k1))
            return float(np.mean(ts))

        ks = max(1, plan.ksplit)
        clustered = bool(plan.direct and plan.direct_cm * plan.direct_cn > 1)
        if clustered:      # direct mode: the multicast cluster kernel (here on HBM operands; in the call it reads host memory)
            ks = 100 + 10 * plan.direct_cm + plan.direct_cn
        ms_step = time_launch(mb, ks, max(steps, 10))
        ks = 1 if clustered else ks
        ms_full = time_launch(rows, 0, max(steps, 5))
        step_ctas = min(148, -(-mb // 128) * -(-nb // 128) * ks)
        step_peak = FP64_PEAK_TFLOPS * step_ctas / 148.0
        tiles_full = -(-rows // 128) * -(-nb // 128)
        solo = {"kernel": f"hclooc_dgemm_direct_kernel<{plan.direct_cm},{plan.direct_cn}>" if clustered else f"hclooc_dgemm_tile_kernel<{ks}>", "launch": f"{mb}x{nb}x{K}", "ctas": step_ctas, "ms_per_launch": ms_step,
                "achieved": 2.0 * mb * nb * K / (ms_step * 1e-3) / 1e12, "peak": step_peak,
                "note": "one step's launch timed ALONE; peak = 37.2 TFLOP/s x min(CTAs, 148)/148 (in the pipeline other steps' kernels run beside it and fill its wave tail)"}
        solo["frac"] = solo["achieved"] / step_peak
        # the library's own rule (launch_dgemm_tiles): persistent stream-K unless the tiles fill their waves of 148 to 98.8 % or better
        waves_full = -(-tiles_full // 148)
        full_is_streamk = tiles_full >= 148 and tiles_full < 0.988 * waves_full * 148
        full = {"kernel": "hclooc_dgemm_streamk_kernel" if full_is_streamk else "hclooc_dgemm_tile_kernel<1> (whole waves: one CTA per tile)", "launch": f"{rows}x{nb}x{K}",
                "ms_per_launch": ms_full, "achieved": 2.0 * rows * nb * K / (ms_full * 1e-3) / 1e12, "peak": FP64_PEAK_TFLOPS}
        full["frac"] = full["achieved"] / FP64_PEAK_TFLOPS
        del dA, dB, dC
        return solo, full, 2 * (warmup + max(steps, 10)) - (max(steps, 10) - max(steps, 5))

    def traced_call(self, ctx, fn):
        """One more call with the library's tracing on: every kernel bracketed by timing events on ITS compute stream.  Returns
        (flops of all launches, union of their [start, end] intervals in ms, launches, mean single-launch duration in ms)."""
        H = self.H
        H.hclooc_ctx_set_trace(ctx, True)
        try:
            fn()
            recs = H.hclooc_ctx_get_trace(ctx)
        finally:
            H.hclooc_ctx_set_trace(ctx, False)
        g = recs[recs["kind"] == 3]
        if not len(g):
            return None
        order = np.argsort(g["t_start_ms"])
        s, e = g["t_start_ms"][order], g["t_end_ms"][order]
        union, cur_s, cur_e = 0.0, s[0], e[0]
        for a, b in zip(s[1:], e[1:]):
            if a > cur_e:
                union += cur_e - cur_s
                cur_s, cur_e = a, b
            else:
                cur_e = max(cur_e, b)
        union += cur_e - cur_s
        return float(g["flops"].sum()), float(union), int(len(g)), float(np.mean(e - s))

    def run(self):
        args, H, torch = self.args, self.H, self.torch
        name, wl = pick_workload(args.workload, self.share)
        M, N, K = wl["M"], wl["N"], wl["K"]
        seed = self.synthgen.BASE_SEED + wl["seed_idx"]
        flops = 2.0 * M * N * K
        # N > 1: ONE problem of world*M rows cut into row bands of C (hclooc_shard_rows): rank r owns rows r*M .. of A
        # and C, every rank holds all of B; the bands are independent, so no collective is on
        # the data path and per-GPU work is fixed as N grows (weak scaling).
        row0, rows = H.hclooc_shard_rows(self.world * M, self.world, self.rank, 128)
        assert (row0, rows) == (self.rank * M, M) or M % 128
        heavy = flops / 36e12 > 1.0
        steps = args.steps if args.steps else (3 if heavy else 10)
        warmup = max(args.warmup, 3)

        live = measure_link(H)
        if live:
            LINK.update(live)
        cal = None
        if not args.no_calibrate:      # the planner's cost model takes THIS box's link rates (hclooc_calibrate_link) instead of its defaults
            cal = dict(zip(("h2d_GBps", "d2h_GBps", "duplex_GBps"), H.hclooc_calibrate_link(None)))
        self.calibration = cal
        peak_measured = H.hclooc_probe_fp64(0, 4, 1.0)
        per_config = None
        if self.world == 1 and not args.no_per_config and args.workload == "auto":
            per_config = self.per_config([c for c in ("cfg1", "cfg2", "cfg3", "cfg4") if c != name])

        # ---- the headline workload: pinned host matrices, then the context over (nearly) all that is left of the device
        in_core = None
        if not args.no_in_core:
            in_core = self.in_core_leg(wl, warmup)
        plan0 = H.hclooc_plan_trans(M, N, K, wl["beta"] != 0.0, 0, wl["budget"] or (int(torch.cuda.mem_get_info()[0]) - 4 * GiB), 0, self.ta, self.tb)
        solo, full, n_leg_launches = self.kernel_legs(wl, plan0, steps, warmup)
        torch.cuda.empty_cache()
        A, B, C, t_pin = self.host_matrices(wl, seed)
        ctx, ws, streams, budget = self.make_ctx(wl["budget"])
        fn = lambda: self.call(ctx, wl, A, B, C, budget)
        with ClockSampler(self.local) as clk:
            r = self.timed(fn, steps, warmup)
            clocks = clk.summary()
        st = r["stats"]
        plan = st.plan
        tr = self.traced_call(ctx, fn)
        ks = max(1, plan.ksplit)
        kname = (f"hclooc_dgemm_direct_kernel<{plan.direct_cm},{plan.direct_cn}>" if plan.direct and plan.direct_cm * plan.direct_cn > 1
                 else f"hclooc_dgemm_tile_kernel<{ks}>")
        launch = f"{min(plan.mb, M)}x{min(plan.nb, N)}x{min(plan.kb, K)}"
        traffic, traffic_src = ncu_traffic(kname, launch)
        roof = {"bound": "alu", "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s", "kernel": kname, "launch": launch,
                "peak_source": "derived: 148 SM x 128 FP64 flop/clk (DMMA.8x8x4) x 1.965 GHz; peak_measured = hclooc_probe_fp64 (DMMA register chains) run live",
                "peak_measured": peak_measured, "traffic": traffic, "traffic_source": traffic_src,
                "solo_step": solo, "streamk": full}
        if tr:
            fl, union_ms, n_launch, mean_ms = tr
            roof.update({"achieved": fl / (union_ms * 1e-3) / 1e12, "launches_per_step": n_launch, "ms_kernels_busy": union_ms,
                         "ms_per_launch": union_ms / n_launch, "ms_per_launch_solo_span": mean_ms,
                         "how": "one traced call (timing events around every kernel on its own compute stream): flops of all launches / time during "
                                "which at least one was running; several steps' kernels overlap on up to 8 streams, so the per-launch figure is that time / launches"})
        else:   # direct mode: one launch, the call IS the kernel
            roof.update({"achieved": solo["achieved"], "ms_per_launch": solo["ms_per_launch"], "how": "the call is one launch; see solo_step"})
        roof["frac"] = roof["achieved"] / FP64_PEAK_TFLOPS
        e2e = self.e2e_record(wl, r)
        e2e["link_peaks"] = LINK
        out = {
            "metric": METRIC,
            "value": self.world * flops / (r["ms_events"] * 1e-3) / 1e12, "unit": "TFLOP/s", "n_gpus": self.world, "steps": steps,
            "warmup": warmup, "ms_per_step": r["ms_events"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "ci95_rel": r["ci95_rel"],
            "config": {"workload": f"{name}: {wl['desc']}", "M": M, "N": N, "K": K, "alpha": wl["alpha"], "beta": wl["beta"],
                       "device_budget_bytes": budget, "dist": wl["dist"], "trans": args.trans,
                       "parallelism": (f"{self.world} row bands of C of {M} rows each, one per GPU (hclooc_shard_rows), B on every rank, no collective"
                                       if self.world > 1 else "1 GPU"), "M_global": self.world * M,
                       "matrices_bytes": wl_bytes(wl), "hbm_total_bytes": int(torch.cuda.get_device_properties(self.local).total_memory),
                       "exceeds_hbm": wl_bytes(wl) > int(torch.cuda.get_device_properties(self.local).total_memory),
                       "host_mem_total_bytes": meminfo("MemTotal"), "t_pin_s": t_pin,
                       "cost_model_link": self.calibration or "library defaults (55.5 / 51.5 / 88 GB/s)",
                       "plan": self.plan_summary(plan),
                       "l2": "inputs (A+B+C = %.2f GB) are host-resident and exceed the 126 MB L2; no flush needed" % (wl_bytes(wl) / 1e9),
                       "value_leg": "CUDA events around the K host-resident calls (the pipeline: uploads, kernels, downloads); the in-core kernel rate is under in_core"},
            "e2e": e2e,
            "gpu_launches": int(st.n_kernels * steps),
            "gpu_launches_outside_timed_region": {"traced_call": int(st.n_kernels), "kernel_legs": n_leg_launches},
            "clocks": clocks,
            "roofline": roof,
        }
        if in_core:
            out["in_core"] = in_core
        if per_config is not None:
            out["per_config"] = per_config
        if self.rank == 0 and self.world == 1 and not args.no_cpu_baseline:
            crows, ccols = oracle_sample_shape(wl, args.cpu_flops, 512)
            cflops, times = time_oracle(wl, crows, ccols, seed, 1, 0, mats=(A.view, B.view, C.view))
            out["cpu_baseline"] = {"value": cflops / times[0] / 1e12, "unit": "TFLOP/s", "cores": os.cpu_count(), "kind": "oracle",
                                   "sample": f"first {crows} rows x first {ccols} columns of C (K={K}), {times[0]:.1f} s of oracle.dgemm"}
        H.hclooc_ctx_destroy(ctx)
        for X in (A, B, C):
            X.free()
        if self.dist:
            self.dist.destroy_process_group()
        if self.rank == 0:
            print(json.dumps(out))

    def in_core_leg(self, wl, warmup):
        """The in-core case of the library: all three operands device-resident, one launch, nothing staged
        -- on the workload itself when it fits a quarter of the device, else on its first 16384 rows and columns."""
        torch, H = self.torch, self.H
        free = int(torch.cuda.mem_get_info()[0])
        m, n, k = wl["M"], wl["N"], wl["K"]
        if wl_bytes(wl) > free // 4:
            m, n = min(m, 16384), min(n, 16384)
        g = torch.Generator(device="cuda"); g.manual_seed(180805057)
        ta, tb = self.ta, self.tb
        dA = torch.rand((k, m) if ta else (m, k), generator=g, dtype=torch.float64, device="cuda") * 2 - 1
        dB = torch.rand((n, k) if tb else (k, n), generator=g, dtype=torch.float64, device="cuda") * 2 - 1
        dC = torch.rand((m, n), generator=g, dtype=torch.float64, device="cuda") * 2 - 1
        torch.cuda.synchronize()
        ctx = H.hclooc_ctx_create(self.local)
        sub = dict(wl, M=m, N=n, K=k)
        try:
            r = self.timed(lambda: self.call(ctx, sub, dA, dB, dC, 256 * MiB), 10, warmup)
        finally:
            H.hclooc_ctx_destroy(ctx)
        fl = 2.0 * m * n * k
        val = fl / (r["ms_events"] * 1e-3) / 1e12
        del dA, dB, dC
        torch.cuda.empty_cache()
        return {"value": val, "unit": "TFLOP/s", "ms_per_step": r["ms_events"], "shape": f"{m}x{n}x{k}", "frac_of_fp64_peak": val / FP64_PEAK_TFLOPS,
                "note": "A, B, C resident in HBM: one stream-K launch on the caller's matrices, nothing staged (kernel-only rate; not the metric)"}

    def phases(self):
        """Where the time of a small, latency-bound call goes (BASELINE config 1 in direct mode: ONE kernel launch whose TMA loads
        read A and B from pinned host memory and whose epilogue reads and writes C there): the same call timed with parts of its
        work removed -- a 128 x 128 x 16 call (launch + synchronisation floor), beta = 0 (no C read), alpha = 0 (no A / B stream:
        C read and written only) -- and the plain copies of the same bytes (what a staged path would at least pay)."""
        H, torch = self.H, self.torch
        name, wl = pick_workload(self.args.workload, self.share)
        M, N, K = wl["M"], wl["N"], wl["K"]
        live = measure_link(H)
        if live:
            LINK.update(live)
        ctx, ws, streams, budget = self.make_ctx(wl["budget"])
        A, B, C, _ = self.host_matrices(wl, self.synthgen.BASE_SEED + wl["seed_idx"])
        steps = self.args.steps or 200

        def t_us(fn):
            return 1e3 * self.timed(fn, steps, 200)["ms_wall"]

        out = {"phases": True, "workload": f"{name}: {wl['desc']}", "steps": steps, "unit": "us per call (host clock around the calls)"}
        st = H.hclooc_dgemm_ex(ctx, M, N, K, wl["alpha"], A, K, B, N, wl["beta"], C, N, budget)
        out["plan"] = self.plan_summary(st.plan)
        out["call"] = t_us(lambda: H.hclooc_dgemm_ex(ctx, M, N, K, wl["alpha"], A, K, B, N, wl["beta"], C, N, budget))
        out["call_beta0_no_C_read"] = t_us(lambda: H.hclooc_dgemm_ex(ctx, M, N, K, wl["alpha"], A, K, B, N, 0.0, C, N, budget))
        out["call_alpha0_C_read_and_write_only"] = t_us(lambda: H.hclooc_dgemm_ex(ctx, M, N, K, 0.0, A, K, B, N, wl["beta"], C, N, budget))
        out["call_128x128x16_launch_and_sync_floor"] = t_us(lambda: H.hclooc_dgemm_ex(ctx, 128, 128, 16, wl["alpha"], A, K, B, N, 0.0, C, N, budget))
        nb_in, nb_out = 8 * (M * K + K * N + M * N), 8 * M * N
        d = H.hclMalloc(nb_in)
        s0 = H.hclStreamCreate()

        def copies():
            H.hclMemcpyAsync(d, A, 8 * M * K, H.HCL_H2D, s0); H.hclMemcpyAsync(d + 8 * M * K, B, 8 * K * N, H.HCL_H2D, s0)
            H.hclMemcpyAsync(d + 8 * (M * K + K * N), C, 8 * M * N, H.HCL_H2D, s0); H.hclMemcpyAsync(C, d, nb_out, H.HCL_D2H, s0)
            H.hclStreamSynchronize(s0)
            return st
        out["four_plain_copies_of_the_same_bytes"] = t_us(copies)
        t_roof, t_flop, t_link = link_roofline_s(2.0 * M * N * K, st.bytes_h2d, st.bytes_d2h)
        out["roofline_us"] = 1e6 * t_roof
        out["frac_of_roofline"] = 1e6 * t_roof / out["call"]
        floor = out["call_128x128x16_launch_and_sync_floor"]
        out["cap_on_frac_from_the_floor"] = 1e6 * t_roof / (1e6 * t_roof + floor)
        out["link_peaks"] = LINK
        H.hclFree(d); H.hclStreamDestroy(s0)
        H.hclooc_ctx_destroy(ctx)
        if self.rank == 0:
            print(json.dumps(out))

    def kernel_only(self):
        """Only the kernel legs (for ncu captures of the tile kernel at the workload's step shape)."""
        name, wl = pick_workload(self.args.workload, self.share)
        budget = wl["budget"] or (int(self.torch.cuda.mem_get_info()[0]) - 4 * GiB)
        plan = self.H.hclooc_plan_trans(wl["M"], wl["N"], wl["K"], wl["beta"] != 0.0, 0, budget, 0, self.ta, self.tb)
        with ClockSampler(self.local) as clk:
            solo, full, _ = self.kernel_legs(wl, plan, self.args.steps or 3, max(self.args.warmup, 1))
            clocks = clk.summary()
        if self.rank == 0:
            print(json.dumps({"kernel_only": True, "workload": name, "solo_step": solo, "streamk": full, "clocks": clocks}))


# ---------------------------------------------------------------------------------------------- the other product paths
def run_op(args):
    """`--op dsyrk|dsyr2k|dtrsm|dtrsm_right|dpotrf|dgetrf`: the routines built on the out-of-core DGEMM, timed like the
    DGEMM -- pinned host operands, a context created beforehand, wall time inside the call -- against the roofline of the call
    (the slower of its flops at the FP64 peak and its own bytes at the link rates measured here).  One JSON line."""
    import torch
    import synthgen
    import paper_1808_05056_b200 as H
    torch.cuda.set_device(0)
    live = measure_link(H)
    if live:
        LINK.update(live)
    op, M, N, K, budget = args.op, args.m, args.n, args.k, args.budget
    seed = synthgen.BASE_SEED + 9
    if op in ("dtrsm_dev", "dtrsm_right_dev", "dpotrf_dev", "dgetrf_dev"):
        return run_dev_op(args, H, torch)
    ctx = H.hclooc_ctx_create(0)
    mats = []

    def host(rows, cols, name, dist="uniform"):
        X = H.HostMatrix(rows, cols)
        synthgen.fill(X.array, seed, name, dist)
        mats.append(X)
        return X

    extra = {}
    if op in ("dsyrk", "dsyr2k"):
        A, C = host(N, K, "A"), host(N, N, "C")
        Bm = host(N, K, "B") if op == "dsyr2k" else None
        flops = float(N) * (N + 1) * K * (2 if op == "dsyr2k" else 1)
        if op == "dsyrk":
            call = lambda: H.hclooc_dsyrk(ctx, args.uplo, args.trans, N, K, 1.0, A, A.ld, args.beta, C, N, budget)
        else:
            call = lambda: H.hclooc_dsyr2k(ctx, args.uplo, args.trans, N, K, 1.0, A, A.ld, Bm, Bm.ld, args.beta, C, N, budget)
        shape = {"N": N, "K": K}
    elif op in ("dtrsm", "dtrsm_right"):
        n_tri = M if op == "dtrsm" else N
        A, Bm = host(n_tri, n_tri, "A"), host(M, N, "B")
        synthgen.shape_triangular(A.view, "uniform")
        flops = float(M) * N * n_tri
        B0 = None
        if op == "dtrsm":
            call = lambda: H.hclooc_dtrsm(ctx, args.uplo, args.trans, 0, M, N, 1.0, A, A.ld, Bm, Bm.ld, budget)
        else:
            call = lambda: H.hclooc_dtrsm_side(ctx, H.HCL_SIDE_RIGHT, args.uplo, args.trans, 0, M, N, 1.0, A, A.ld, Bm, Bm.ld, budget)
        shape = {"M": M, "N": N}
    elif op == "dpotrf":
        # symmetric positive definite by construction: uniform[-1,1) entries / N off the diagonal (row sums < 1), diagonal in [1, 2)
        A = host(N, N, "A")
        synthgen.shape_triangular(A.view, "uniform")
        d = np.abs(A.view[np.arange(N), np.arange(N)]).copy()
        A0 = H.HostMatrix(N, N)
        mats.append(A0)
        half = np.tril(A.view, -1)
        A0.view[...] = half
        A0.view[...] += half.T
        A0.view[np.arange(N), np.arange(N)] = d
        del half
        flops = float(N) ** 3 / 3.0
        infos = []

        def call():
            A.view[...] = A0.view                      # the factorization overwrites its input: restore it (outside the timed span:
            info, st = H.hclooc_dpotrf(ctx, args.uplo, N, A, A.ld, budget)      # t_total_s is the wall time inside the call)
            infos.append(info)
            return st
        shape = {"N": N}
        extra["info"] = infos
    elif op == "dgetrf":
        # a general matrix: uniform[-1,1) entries (partial pivoting does the rest); the factorization overwrites its input, which is
        # restored from a copy before every call (outside the timed span: t_total_s is the wall time inside the call)
        A = host(M, N, "A")
        A0 = H.HostMatrix(M, N)
        mats.append(A0)
        A0.view[...] = A.view
        flops = float(M) * N * N - float(N) ** 3 / 3.0 if M >= N else float(N) * M * M - float(M) ** 3 / 3.0
        infos = []

        def call():
            A.view[...] = A0.view
            ipiv, info, st = H.hclooc_dgetrf(ctx, M, N, A, A.ld, budget)
            infos.append(info)
            return st
        shape = {"M": M, "N": N}
        extra["info"] = infos
    else:
        raise SystemExit(f"unknown --op {op}")
    try:
        with ClockSampler(0) as clk:
            ts, st = [], None
            for _ in range(max(2, args.steps or 3)):
                st = call()
                ts.append(st.t_total_s)
            clocks = clk.summary()
    finally:
        H.hclooc_ctx_destroy(ctx)
        for X in mats:
            X.free()
    t = float(np.mean(ts[1:]))
    t_roof, t_flop, t_link = link_roofline_s(flops, st.bytes_h2d, st.bytes_d2h)
    out = {"op": f"hclooc_{op}", **shape, "uplo": args.uplo, "trans": args.trans, "budget_bytes": budget, "t_s": t, "t_all_s": ts,
           "tflops": flops / t / 1e12, "flops": flops, "h2d_GB": st.bytes_h2d / 1e9, "d2h_GB": st.bytes_d2h / 1e9,
           "kernels": int(st.n_kernels), "plan": Bench.plan_summary(st.plan), "t_flop_s": t_flop, "t_link_s": t_link,
           "bound": "fp64" if t_flop >= t_link else "link", "frac_of_roofline": t_roof / t, "link_peaks": LINK, "clocks": clocks, **extra}
    print(json.dumps(out))


def run_cublasxt(args):
    """`--op cublasxt`: SIDE REFERENCE ONLY (north_star: "cuBLAS-XT may be timed as a side reference only"; it is the library the paper
    compares with, PAPER.md:372 / :396).  NVIDIA's out-of-core DGEMM, cublasXtDgemm, on the same pinned host matrices as `bench.py
    --workload ...` / `--m --n --k`, one GPU, block dimension --xt-block (its tile size; the library streams tiles itself), wall time of
    the call, beside hclooc_dgemm_ex on the very same buffers in the same process.  Loaded with ctypes from the CUDA toolkit's libcublas;
    nothing of the product path links or calls it.  Row-major C = A B is the column-major product C^T = B^T A^T, so the operands swap."""
    import ctypes
    import glob
    import torch
    import synthgen
    import paper_1808_05056_b200 as H
    torch.cuda.set_device(0)
    # the copy torch itself loaded its cublasLt from comes first (the toolkit's libcublas wants the toolkit's libcublasLt)
    cands = sorted(glob.glob(os.path.join(os.path.dirname(os.path.dirname(torch.__file__)), "nvidia", "cublas", "lib", "libcublas.so.*"))) + \
        sorted(glob.glob("/usr/local/cuda/lib64/libcublas.so.*")) + ["libcublas.so.12"]
    L, errs = None, []
    for cand in cands:
        try:
            L = ctypes.CDLL(cand)
            cands = [cand]
            break
        except OSError as e:
            errs.append(str(e))
    if L is None:
        print(json.dumps({"op": "cublasXtDgemm", "unavailable": errs}))
        return
    M, N, K, budget = args.m, args.n, args.k, args.budget or 4 * GiB
    live = measure_link(H)
    if live:
        LINK.update(live)
    A, B, C = H.HostMatrix(M, K), H.HostMatrix(K, N), H.HostMatrix(M, N)
    seed = synthgen.BASE_SEED + 9
    for X, nm in ((A, "A"), (B, "B"), (C, "C")):
        synthgen.fill(X.array, seed, nm, "uniform")
    C0 = C.view[:64].copy()
    handle = ctypes.c_void_p()
    vp, i32, sz, dbl = ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t, ctypes.c_double
    L.cublasXtCreate.argtypes = [ctypes.POINTER(vp)]
    L.cublasXtDestroy.argtypes = [vp]
    L.cublasXtDeviceSelect.argtypes = [vp, i32, ctypes.POINTER(i32)]
    L.cublasXtSetBlockDim.argtypes = [vp, i32]
    L.cublasXtSetPinningMemMode.argtypes = [vp, i32]
    L.cublasXtDgemm.argtypes = [vp, i32, i32, sz, sz, sz, ctypes.POINTER(dbl), vp, sz, vp, sz, ctypes.POINTER(dbl), vp, sz]

    def chk(rc, what):
        if rc != 0:
            raise SystemExit(f"{what}: cublasStatus {rc}")
    chk(L.cublasXtCreate(ctypes.byref(handle)), "cublasXtCreate")
    dev = (i32 * 1)(0)
    chk(L.cublasXtDeviceSelect(handle, 1, dev), "cublasXtDeviceSelect")
    chk(L.cublasXtSetBlockDim(handle, args.xt_block), "cublasXtSetBlockDim")
    alpha, beta = dbl(1.0), dbl(args.beta)
    flops = 2.0 * M * N * K
    rec = {"op": "cublasXtDgemm (side reference, not the product path)", "M": M, "N": N, "K": K, "beta": args.beta, "xt_block_dim": args.xt_block, "lib": cands[0]}
    try:
        ts = []
        for _ in range(max(2, args.steps or 3)):
            t0 = time.perf_counter()
            # column-major: C^T (N x M, ld N) = B^T (N x K, ld N) * A^T (K x M, ld K);  CUBLAS_OP_N = 0
            chk(L.cublasXtDgemm(handle, 0, 0, N, M, K, ctypes.byref(alpha), B.ptr, N, A.ptr, K, ctypes.byref(beta), C.ptr, N), "cublasXtDgemm")
            torch.cuda.synchronize()
            ts.append(time.perf_counter() - t0)
        t = float(np.mean(ts[1:]))
        t_roof, t_flop, t_link = link_roofline_s(flops, 8 * (M * K + K * N + (M * N if args.beta else 0)), 8 * M * N)
        rec["cublasxt"] = {"t_s": t, "t_all_s": ts, "tflops": flops / t / 1e12, "frac_of_roofline_on_compulsory_bytes": t_roof / t}
        # the product path on the very same buffers
        ctx = H.hclooc_ctx_create(0)
        try:
            ts2, st = [], None
            for _ in range(max(2, args.steps or 3)):
                st = H.hclooc_dgemm_ex(ctx, M, N, K, 1.0, A, K, B, N, args.beta, C, N, budget)
                ts2.append(st.t_total_s)
        finally:
            H.hclooc_ctx_destroy(ctx)
        t2 = float(np.mean(ts2[1:]))
        t_roof2, _, _ = link_roofline_s(flops, st.bytes_h2d, st.bytes_d2h)
        rec["hclooc_dgemm"] = {"t_s": t2, "tflops": flops / t2 / 1e12, "budget_bytes": budget, "frac_of_roofline": t_roof2 / t2, "plan": Bench.plan_summary(st.plan)}
        rec["hclooc_over_cublasxt"] = t / t2
        rec["link_peaks"] = LINK
    finally:
        L.cublasXtDestroy(handle)
        for X in (A, B, C):
            X.free()
    print(json.dumps(rec))


def run_dev_op(args, H, torch):
    """`--op dtrsm_dev|dtrsm_right_dev|dpotrf_dev|dgetrf_dev`: the DEVICE phases alone (hclDtrsmAsync / hclDpotrfAsync / hclDgetrf on device-resident operands:
    recursive halving down to the 128 x 128 block kernels), CUDA events on the launching stream, median of --steps launches.  With
    --m 128 (dtrsm_dev) / --n 128 (the others) the call is ONE launch of the block kernel."""
    op, M, N = args.op, args.m, args.n
    cur = torch.cuda.current_stream()
    g = torch.Generator(device="cuda"); g.manual_seed(180805056)
    n = M if op == "dtrsm_dev" else N
    T = None if op == "dgetrf_dev" else torch.rand((n, n), generator=g, dtype=torch.float64, device="cuda") / n + torch.eye(n, dtype=torch.float64, device="cuda") * 1.5
    if op == "dpotrf_dev":
        S = (T + T.T) / 2 + torch.eye(n, dtype=torch.float64, device="cuda")
        W = S.clone()
        info = torch.zeros(1, dtype=torch.int64, device="cuda")
        fn = lambda: H.hclDpotrfAsync(args.uplo, n, W, n, info, cur)
        pre = lambda: W.copy_(S)
        flops, shape = n ** 3 / 3.0, {"N": n}
    elif op == "dgetrf_dev":
        S = torch.rand((M, N), generator=g, dtype=torch.float64, device="cuda") * 2 - 1
        W = S.clone()
        fn = lambda: H.hclDgetrf(M, N, W, N, cur)           # synchronous: the host folds the interchanges (include/hclooc.h)
        pre = lambda: W.copy_(S)
        flops = float(M) * N * N - float(N) ** 3 / 3.0 if M >= N else float(N) * M * M - float(M) ** 3 / 3.0
        shape = {"M": M, "N": N}
    else:
        Bm = torch.rand((M, N), generator=g, dtype=torch.float64, device="cuda")
        side = 0 if op == "dtrsm_dev" else 1
        fn = lambda: H.hclDtrsmAsync(side, args.uplo, args.trans, 0, M, N, 1.0, T, n, Bm, N, cur)
        pre = lambda: None
        flops, shape = float(M) * N * n, {"M": M, "N": N}
    torch.cuda.synchronize()
    ts = []
    for it in range(3 + max(5, args.steps or 20)):
        pre()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(cur); fn(); e1.record(cur); e1.synchronize()
        if it >= 3:
            ts.append(e0.elapsed_time(e1))
    ms = float(np.median(ts))
    print(json.dumps({"op": "hcl" + {"dtrsm_dev": "DtrsmAsync (Left)", "dtrsm_right_dev": "DtrsmAsync (Right)", "dpotrf_dev": "DpotrfAsync", "dgetrf_dev": "Dgetrf"}[op], **shape,
                      "uplo": args.uplo, "trans": args.trans, "ms": ms, "tflops": flops / ms / 1e9, "frac_of_fp64_peak": flops / ms / 1e9 / FP64_PEAK_TFLOPS}))


TRANSITION_SIZES = [4096, 8192, 12288, 16384, 20480, 22528, 23552, 24576, 28672, 32768, 36864, 40960, 46080]


def run_transition_sweep(args):
    """`--sweep transition`: the paper's own experiment shape: square FP64 DGEMM, N
    swept across the point where A, B and C stop fitting the device budget (default 12.2e9 bytes: the paper's 12 GB cards
    switched to out-of-core above N = 22528), end to end, for the tuned scheduler (hclooc_dgemm_ex) and the paper's Figure-2
    pipeline (hclooc_dgemm_fig2), each with its fraction of max(T_flop, T_link).  One JSON line per size, then a Markdown table."""
    import ctypes
    import torch
    import synthgen
    import paper_1808_05056_b200 as H
    torch.cuda.set_device(0)
    live = measure_link(H)
    if live:
        LINK.update(live)
    budget = args.budget if args.budget else 12_200_000_000
    if not args.no_calibrate:          # the choice between the resident schedule and the slice pipeline rests on the link rates
        print(json.dumps({"cost_model_link": dict(zip(("h2d_GBps", "d2h_GBps", "duplex_GBps"), H.hclooc_calibrate_link(None)))}), flush=True)
    sizes = sorted(int(x) for x in args.sizes.split(",")) if args.sizes else TRANSITION_SIZES
    nmax = sizes[-1]
    bufs = [H.HostMatrix(nmax, nmax) for _ in range(3)]        # one pinned allocation per matrix, reused as a dense N x N matrix
    ctx = H.hclooc_ctx_create(0)
    rows = []
    try:
        for n in sizes:
            A, B, C = (np.frombuffer((ctypes.c_double * (n * n)).from_address(X.ptr), dtype=np.float64).reshape(n, n) for X in bufs)
            for arr, nm in ((A, "A"), (B, "B"), (C, "C")):
                synthgen.fill(arr, synthgen.BASE_SEED + 9, nm, "uniform")
            rec = {"N": n, "fits_budget": 24 * n * n <= budget, "budget_bytes": budget, "flops": 2.0 * n ** 3}
            for label, call in (("tuned", lambda: H.hclooc_dgemm_ex(ctx, n, n, n, 1.0, A, n, B, n, args.beta, C, n, budget)),
                                ("fig2", lambda: H.hclooc_dgemm_fig2(n, n, n, 1.0, A, n, B, n, args.beta, C, n, budget))):
                ts, st = [], None
                for _ in range(max(2, args.steps or 3)):
                    st = call()
                    ts.append(st.t_total_s)
                t = float(np.mean(ts[1:]))
                t_roof, t_flop, t_link = link_roofline_s(2.0 * n ** 3, st.bytes_h2d, st.bytes_d2h)
                rec[label] = {"t_s": t, "tflops": 2.0 * n ** 3 / t / 1e12, "h": st.plan.h, "w": st.plan.w, "kpanels": st.plan.kpanels, "steps": st.plan.n_steps,
                              "h2d_GB": st.bytes_h2d / 1e9, "d2h_GB": st.bytes_d2h / 1e9, "frac_of_roofline": t_roof / t,
                              "bound": "fp64" if t_flop >= t_link else "link", "t_model_s": st.plan.t_model_s}
                if label == "tuned":
                    st_tuned = st
            rec["tuned"]["resident"] = st_tuned.plan.resident
            if st_tuned.plan.resident:
                # the resident schedule was picked (the matrices fit the budget): the slice pipeline on the same call, for comparison
                prev = os.environ.get("HCLOOC_RESIDENT")
                os.environ["HCLOOC_RESIDENT"] = "0"
                try:
                    ts = []
                    for _ in range(max(2, args.steps or 3)):
                        st = H.hclooc_dgemm_ex(ctx, n, n, n, 1.0, A, n, B, n, args.beta, C, n, budget)
                        ts.append(st.t_total_s)
                finally:
                    if prev is None:
                        del os.environ["HCLOOC_RESIDENT"]
                    else:
                        os.environ["HCLOOC_RESIDENT"] = prev
                t = float(np.mean(ts[1:]))
                t_roof, t_flop, t_link = link_roofline_s(2.0 * n ** 3, st.bytes_h2d, st.bytes_d2h)
                rec["slices"] = {"t_s": t, "tflops": 2.0 * n ** 3 / t / 1e12, "h": st.plan.h, "w": st.plan.w, "kpanels": st.plan.kpanels,
                                 "frac_of_roofline": t_roof / t, "t_model_s": st.plan.t_model_s}
            rec["fig2_over_tuned"] = rec["fig2"]["tflops"] / rec["tuned"]["tflops"]
            rows.append(rec)
            print(json.dumps(rec), flush=True)
    finally:
        H.hclooc_ctx_destroy(ctx)
        for X in bufs:
            X.free()
    print("| N | fits budget | tuned TFLOP/s (h x w x kpanels) | schedule | tuned / roofline | slice pipeline on the same call / roofline | Figure-2 TFLOP/s (h x w) | Figure-2 / roofline | Figure-2 / tuned |")
    print("|---|---|---|---|---|---|---|---|---|")
    for r in rows:
        sl = f"{r['slices']['frac_of_roofline']:.3f} ({r['slices']['h']} x {r['slices']['w']} x {r['slices']['kpanels']})" if "slices" in r else "-"
        sched = f"resident, switch at panel {r['tuned']['resident'] - 1}" if r["tuned"]["resident"] else "slices"
        print(f"| {r['N']} | {'yes' if r['fits_budget'] else 'no'} | {r['tuned']['tflops']:.2f} ({r['tuned']['h']} x {r['tuned']['w']} x {r['tuned']['kpanels']}) | {sched} | "
              f"{r['tuned']['frac_of_roofline']:.3f} ({r['tuned']['bound']}) | {sl} | {r['fig2']['tflops']:.2f} ({r['fig2']['h']} x {r['fig2']['w']}) | "
              f"{r['fig2']['frac_of_roofline']:.3f} | {r['fig2_over_tuned']:.3f} |")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=0, help="timed calls (0 = 3 for workloads of more than a second per call, else 10)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="auto", choices=["auto", "cfg5s"] + sorted(WORKLOADS))
    ap.add_argument("--ref-rows", type=int, default=512, help="rows of C per oracle step (reference arm)")
    ap.add_argument("--ref-flops", type=float, default=1.5e11, help="flops per oracle step (reference arm): about 2 s on 16 cores")
    ap.add_argument("--cpu-flops", type=float, default=1.0e12, help="flops of the cpu_baseline sample: 10-30 s of the oracle")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the cfg1-cfg4 block of the default (auto) run")
    ap.add_argument("--no-in-core", action="store_true")
    ap.add_argument("--no-calibrate", action="store_true", help="leave the planner's cost model on its default link rates")
    ap.add_argument("--phases", action="store_true", help="--workload cfg1: where the time of the call goes (launch + synchronisation floor, "
                                                          "C read, C write, operand stream), one JSON line")
    ap.add_argument("--trans", default="NN", choices=["NN", "TN", "NT", "TT"],
                    help="e2e leg through hclooc_dgemm_t with op(A), op(B) transposed (the same buffers read as the stored K x M / N x K matrices)")
    ap.add_argument("--kernel-only", action="store_true", help="only the kernel legs (for ncu captures of the tile kernel)")
    ap.add_argument("--op", default="dgemm", choices=["dgemm", "dsyrk", "dsyr2k", "dtrsm", "dtrsm_right", "dpotrf", "dgetrf", "dtrsm_dev", "dtrsm_right_dev", "dpotrf_dev", "dgetrf_dev", "cublasxt"],
                    help="time another routine of the library instead (sizes from --m/--n/--k/--budget; --steps calls, the first discarded)")
    ap.add_argument("--xt-block", type=int, default=8192, help="--op cublasxt: cublasXtSetBlockDim (the side reference's tile size)")
    ap.add_argument("--sweep", default="", choices=["", "transition"], help="transition: the paper's N sweep across the in-core / out-of-core point")
    ap.add_argument("--m", type=int, default=32768)
    ap.add_argument("--n", type=int, default=32768)
    ap.add_argument("--k", type=int, default=8192)
    ap.add_argument("--budget", type=int, default=0, help="--op / --sweep: device budget in bytes (0: 4 GiB for --op, 12.2e9 for the sweep)")
    ap.add_argument("--uplo", type=int, default=0)
    ap.add_argument("--beta", type=float, default=1.0)
    ap.add_argument("--sizes", default="", help="--sweep transition: comma-separated N")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    if args.sweep == "transition":
        return run_transition_sweep(args)
    if args.op != "dgemm":
        args.trans = int(args.trans[0] == "T") if isinstance(args.trans, str) else args.trans
        args.budget = args.budget or (4 << 30)
        return run_cublasxt(args) if args.op == "cublasxt" else run_op(args)
    if args.impl == "reference":
        return run_reference(args)
    b = Bench(args)
    if args.phases:
        return b.phases()
    if args.kernel_only:
        return b.kernel_only()
    b.run()


if __name__ == "__main__":
    main()
