"""Host logic without a GPU: the C ABI exports, the planner (S1) and the schedule (S2-S7).

The schedule is the exact operation list the executor issues, so coverage, byte counts and the
hazard rule of PAPER.md:311 ("data stored in device buffers is not overwritten until kernel
executions that operate on the data have completed") are checked here by simulating stream/event
semantics on the list itself.
"""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_1808_05056_b200 as H

MiB = 1 << 20
GiB = 1 << 30
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
K_H2D_A, K_H2D_B, K_H2D_C, K_GEMM, K_D2H_C, K_WAIT, K_RECORD = range(7)


# ------------------------------------------------------------------ the boundary
def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "hclooc.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(hcl\w+|hclooc_\w+)\s*\(", hdr))
    declared -= {"hclooc_ctx"}
    assert declared == set(H.EXPORTS), declared ^ set(H.EXPORTS)
    L = ctypes.CDLL(H.lib()._name)
    for name in declared:
        assert hasattr(L, name), name
    assert "sm_100a" in H.hclooc_version()
    assert "pageable" in H.hclooc_strerror(2) and H.hclooc_strerror(0) == "success"


def test_binding_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_1808_05056_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cpp", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "liboracle" not in src, f


# ------------------------------------------------------------------ the paper's partitioner rule
def test_paper_example_partition():
    # PAPER.md:301 / Figure 3 (:281): A 4x8, B 8x4, C 4x4, 44 elements -> 4 slices of A, 2 of B, 8 blocks
    assert H.hclMatrixPartitioner(4, 4, 8, 44) == (4, 2)
    assert H.hclMatrixPartitioner(4, 4, 8, 1000) == (1, 1)
    with pytest.raises(H.HclError) as e:
        H.hclMatrixPartitioner(4, 4, 8, 19)
    assert e.value.status == 1


def test_partitioner_agrees_with_brute_force_enumeration():
    rng = np.random.default_rng(0)
    for _ in range(200):
        M, N, K = (int(x) for x in rng.integers(1, 25, 3))
        S = int(rng.integers(1, 3 * (M * K + K * N + M * N)))
        best = None
        for h in range(1, M + 1):
            if M % h:
                continue
            for w in range(1, N + 1):
                if N % w:
                    continue
                mb, nb = M // h, N // w
                if K * nb + 2 * mb * K + 2 * mb * nb > S:
                    continue
                key = (w * M * K + K * N + M * N, h * w, h)
                if best is None or key < best[0]:
                    best = (key, (h, w))
        if best is None:
            with pytest.raises(H.HclError):
                H.hclMatrixPartitioner(M, N, K, S)
        else:
            assert H.hclMatrixPartitioner(M, N, K, S) == best[1], (M, N, K, S)


# ------------------------------------------------------------------ hclooc_plan invariants
CONFIGS = {  # BASELINE.json configs: (M, N, K, beta != 0, budget)
    "cfg1": (512, 512, 512, 1, 1 * MiB),
    "cfg2": (8192, 8192, 8192, 1, 256 * MiB),
    "cfg3": (32768, 32768, 32768, 0, 4 * GiB),
    "cfg4": (65536, 65536, 16384, 1, 16 * GiB),
    "cfg5": (163840, 163840, 8192, 1, 178 * GiB),
}


def plan_checks(p, M, N, K, bnz, budget):
    assert p.workspace_bytes <= budget
    assert p.workspace_bytes == p.n_bbuf * p.bytes_b_buf + p.n_abuf * p.bytes_a_buf + p.n_sets * p.bytes_c_buf + p.n_scratch * p.bytes_scratch
    assert p.h == -(-M // p.mb) and p.w == -(-N // p.nb)
    assert p.n_steps == p.h * p.w * p.kpanels and p.n_sets >= 2
    assert p.ldc_dev >= p.nb and p.ldc_dev % 2 == 0 and p.bytes_c_buf >= p.mb * p.ldc_dev * 8
    if not p.scale_only:
        assert p.kpanels == -(-K // p.kb)
        assert p.lda_dev >= p.kb and p.lda_dev % 2 == 0 and p.ldb_dev >= p.nb and p.ldb_dev % 2 == 0
        assert p.bytes_a_buf >= p.mb * p.lda_dev * 8 and p.bytes_b_buf >= p.kb * p.ldb_dev * 8
        assert p.n_abuf >= p.n_sets
        # A slices: once per column of blocks, minus the min(n_abuf, h) slices the serpentine order finds
        # still resident at each of the (w - 1) column switches of every K panel (restated here)
        a_el = 0
        reuse = min(p.n_abuf, p.h)
        for sl in range(p.w * p.kpanels):
            kk = min(p.kb, K - (sl // p.w) * p.kb)
            if sl % p.w == 0:
                a_el += M * kk
            else:
                kept = min(M, reuse * p.mb) if (sl - 1) % 2 else M - (p.h - reuse) * p.mb
                a_el += (M - kept) * kk
        assert M * K <= a_el <= p.w * M * K
        want_h2d = 8 * (a_el + K * N + (M * N if bnz else 0) + (p.kpanels - 1) * M * N)
    else:
        want_h2d = 8 * (M * N if bnz else 0)
    assert p.bytes_h2d == want_h2d
    assert p.bytes_d2h == 8 * p.kpanels * M * N


@pytest.mark.parametrize("name", list(CONFIGS))
def test_plans_for_the_baseline_configs(name):
    M, N, K, bnz, budget = CONFIGS[name]
    p = H.hclooc_plan(M, N, K, bnz, 0, budget)
    plan_checks(p, M, N, K, bnz, budget)
    assert p.kpanels == 1                       # none of the configs needs a K split
    if name in ("cfg1", "cfg2"):                # link-bound: least traffic the budget allows
        assert p.t_link_s > p.t_flop_s
    else:                                       # FP64-bound
        assert p.t_flop_s > p.t_link_s
    assert p.n_scratch == 0 and p.ksplit >= 1
    if name in ("cfg3", "cfg4"):
        simulate(p, H.hclooc_schedule(p, 8))
    if name == "cfg2":
        assert p.w == 3 and p.bytes_h2d < 8 * 5 * 8192 * 8192     # 5 matrix volumes minus the reused A slices


def test_plans_for_random_shapes_and_budgets():
    rng = np.random.default_rng(1)
    n_ok = 0
    for _ in range(300):
        M, N, K = (int(x) for x in rng.integers(1, 3000, 3))
        budget = int(rng.integers(64 * 1024, 64 * MiB))
        bnz, az = int(rng.integers(0, 2)), int(rng.integers(0, 8) == 0)
        try:
            p = H.hclooc_plan(M, N, K, bnz, az, budget)
        except H.HclError as e:
            assert e.status == 1
            continue
        n_ok += 1
        plan_checks(p, M, N, K, bnz, budget)
    assert n_ok > 250
    with pytest.raises(H.HclError):
        H.hclooc_plan(100, 100, 100, 1, 0, 1024)
    assert H.hclooc_plan(0, 5, 5, 1, 0, MiB).n_steps == 0
    assert H.hclooc_plan(64, 64, 100000, 1, 0, 600 * 1024).kpanels > 1     # K split only when forced


def test_plan_with_c_on_the_device_counts_only_a_and_b_as_link_traffic():
    M, N, K = 2000, 1500, 700
    host = H.hclooc_plan_ex(M, N, K, 1, 0, 6 * MiB, 0)
    cdev = H.hclooc_plan_ex(M, N, K, 1, 0, 6 * MiB, 2)
    assert host.c_on_device == 0 and cdev.c_on_device == 1
    assert cdev.bytes_d2h == 0 and host.bytes_d2h == 8 * M * N
    assert cdev.bytes_h2d <= host.bytes_h2d - 8 * M * N + 8 * (host.w * M * K)      # A and B only
    assert 8 * (M * K + K * N) <= cdev.bytes_h2d <= 8 * (cdev.w * M * K + K * N)
    ops = H.hclooc_schedule(cdev, 4)
    assert int((ops["kind"] == K_H2D_C).sum()) == cdev.h * cdev.w == int((ops["kind"] == K_D2H_C).sum())   # still staged


def test_in_core_plan_for_device_resident_operands():
    p = H.hclooc_plan_ex(8192, 8192, 8192, 1, 0, 256 * MiB, 1)
    assert (p.h, p.w, p.kpanels, p.n_steps) == (1, 1, 1, 1) and (p.mb, p.nb, p.kb) == (8192, 8192, 8192)
    assert p.workspace_bytes == 0 and p.bytes_h2d == 0 and p.bytes_d2h == 0 and p.flops == 2.0 * 8192 ** 3
    q = H.hclooc_plan_ex(8192, 8192, 8192, 1, 0, 256 * MiB, 0)
    assert q.asdict() == H.hclooc_plan(8192, 8192, 8192, 1, 0, 256 * MiB).asdict()


# ------------------------------------------------------------------ schedule: coverage, bytes, hazards
def simulate(plan, ops, alpha_zero=False):
    """Vector-clock simulation of CUDA stream/event semantics over the op list.
    Returns nothing; asserts coverage, byte counts and that conflicting buffer accesses are ordered."""
    n_streams = int(ops["stream"].max()) + 1
    clock = [np.zeros(n_streams, dtype=np.int64) for _ in range(n_streams)]   # per-stream vector clocks
    event_clock = {}
    accesses = {}          # buffer -> list of (vector clock at completion, stream, is_write, row range, tag)
    covered = np.zeros((plan.kpanels, plan.M, plan.N), dtype=np.int8) if plan.M * plan.N * plan.kpanels <= 4e6 else None
    h2d = d2h = n_h2d = n_d2h = 0
    content = {}           # buffer -> what it currently holds (for data-flow checks)

    def access(buf, s, write, lo, hi, tag):
        vc = clock[s].copy()
        for (ovc, os_, ow, olo, ohi, otag) in accesses.setdefault(buf, []):
            if not (write or ow):
                continue
            if hi <= olo or ohi <= lo:
                continue
            # the earlier access must happen-before this one: its clock entry on its own stream <= ours
            assert ovc[os_] <= vc[os_], f"hazard on buffer {buf}: {otag} vs {tag}"
        accesses[buf].append((vc, s, write, lo, hi, tag))
        if len(accesses[buf]) > 64:
            del accesses[buf][:32]

    for idx, o in enumerate(ops):
        s, kind = int(o["stream"]), int(o["kind"])
        clock[s][s] += 1
        if kind == K_RECORD:
            event_clock[int(o["event"])] = clock[s].copy()
        elif kind == K_WAIT:
            assert int(o["event"]) in event_clock, "wait on an event never recorded"
            clock[s] = np.maximum(clock[s], event_clock[int(o["event"])])
        elif kind in (K_H2D_A, K_H2D_B, K_H2D_C):
            assert s == 0
            lo = int(o["dev_r0"]); hi = lo + int(o["nr"])
            access(int(o["buf"]), s, True, lo, hi, (idx, "h2d", kind))
            h2d += int(o["nr"]) * int(o["nc"]) * 8; n_h2d += 1
            key = (kind, int(o["r0"]), int(o["nr"]), int(o["c0"]), int(o["nc"]))
            if kind == K_H2D_C:      # reads the HOST block: ordered after the download that wrote it (K panels p > 0)
                access(("host C", int(o["r0"]), int(o["c0"])), s, False, 0, int(o["nr"]), (idx, "h2d reads host C"))
            if kind == K_H2D_B:
                held = content.setdefault(int(o["buf"]), {})
                for old in [r for r in held if not (r[1] <= lo or hi <= r[0])]:
                    del held[old]                      # overwritten rows
                held[(lo, hi)] = key
            else:
                content[int(o["buf"])] = key
        elif kind == K_GEMM:
            assert s >= 2
            i0, mi, j0, nj, k0, kk = (int(o[f]) for f in ("r0", "nr", "c0", "nc", "k0", "kk"))
            p = k0 // plan.kb if plan.kb else 0
            if not plan.scale_only:
                access(int(o["buf"]), s, False, 0, mi, (idx, "gemm-A"))
                access(int(o["buf2"]), s, False, 0, kk, (idx, "gemm-B"))
                assert content[int(o["buf"])] == (K_H2D_A, i0, mi, k0, kk)          # the right A slice is resident
                rows = sorted(content[int(o["buf2"])].items())
                got = [v for (lo, hi), v in rows if lo < kk]
                assert sum(v[2] for v in got) == kk and all(v[3] == j0 and v[4] == nj for v in got)
                assert min(v[1] for v in got) == k0 and max(v[1] + v[2] for v in got) == k0 + kk
            cload = plan.beta_nonzero or p > 0
            if cload:
                assert content[int(o["buf3"])] == (K_H2D_C, i0, mi, j0, nj)
            access(int(o["buf3"]), s, True, 0, mi, (idx, "gemm-C"))
            content[int(o["buf3"])] = ("result", i0, mi, j0, nj, p)
            assert (o["beta"] == 1.0) == (p > 0)
            if covered is not None:
                covered[p, i0:i0 + mi, j0:j0 + nj] += 1
        elif kind == K_D2H_C:
            assert s == 1
            access(int(o["buf"]), s, False, 0, int(o["nr"]), (idx, "d2h"))
            c = content[int(o["buf"])]
            assert c[0] == "result" and c[1:5] == (int(o["r0"]), int(o["nr"]), int(o["c0"]), int(o["nc"]))
            access(("host C", int(o["r0"]), int(o["c0"])), s, True, 0, int(o["nr"]), (idx, "d2h writes host C"))
            d2h += int(o["nr"]) * int(o["nc"]) * 8; n_d2h += 1
    assert h2d == plan.bytes_h2d and d2h == plan.bytes_d2h
    assert n_h2d == plan.n_copies_h2d and n_d2h == plan.n_copies_d2h
    assert int((ops["kind"] == K_GEMM).sum()) == plan.n_steps
    if covered is not None:
        assert (covered == 1).all()            # every C element computed exactly once per K panel


@pytest.mark.parametrize("shape", [
    (512, 512, 512, 1, 0, 1 * MiB), (515, 389, 301, 1, 0, 1 * MiB), (515, 389, 301, 0, 0, 4 * MiB),
    (96, 112, 20000, 1, 0, 600 * 1024), (300, 200, 150, 1, 1, 1 * MiB), (300, 200, 150, 0, 1, 1 * MiB),
    (2000, 1500, 700, 1, 0, 6 * MiB), (2000, 1500, 700, 0, 0, 64 * MiB), (1, 1, 1, 1, 0, 1 * MiB),
])
@pytest.mark.parametrize("n_compute", [1, 3, 8])
def test_schedule_is_complete_and_hazard_free(shape, n_compute):
    M, N, K, bnz, az, budget = shape
    p = H.hclooc_plan(M, N, K, bnz, az, budget)
    ops = H.hclooc_schedule(p, n_compute)
    simulate(p, ops)


def test_schedule_with_two_b_buffers_prefetches_in_chunks(monkeypatch):
    monkeypatch.setenv("HCLOOC_FORCE_BBUF", "2")     # experiment knob of the planner: two B buffers
    p = H.hclooc_plan(4096, 4096, 2048, 0, 0, 40 * MiB)
    assert p.n_bbuf == 2 and p.w > 1
    ops = H.hclooc_schedule(p, 4)
    simulate(p, ops)
    b_loads = ops[ops["kind"] == K_H2D_B]
    assert len(b_loads) > p.w                   # later slices arrive in several chunks


def test_simulator_catches_a_missing_wait():
    """The checker is not vacuous: dropping the Wait(eA) before the A uploads (buffer free) or
    the waits before a B reload is reported."""
    p = H.hclooc_plan(515, 389, 301, 1, 0, 1 * MiB)
    ops = H.hclooc_schedule(p, 4)
    a_free0 = 3 * p.n_sets + 2 * p.n_bbuf              # event ids: a_free(a) = 3*n_sets + 2*n_bbuf + a
    idx = [i for i, o in enumerate(ops) if o["kind"] == K_WAIT and o["stream"] == 0 and o["event"] >= a_free0]
    assert idx
    with pytest.raises(AssertionError, match="hazard"):
        simulate(p, np.delete(ops, idx))
    if p.n_bbuf == 1 and p.w > 1:
        idx = [i for i, o in enumerate(ops) if o["kind"] == K_WAIT and o["stream"] == 0
               and p.n_sets <= o["event"] < 2 * p.n_sets]      # kernel_done waits before S(b_j)
        assert idx
        with pytest.raises(AssertionError, match="hazard"):
            simulate(p, np.delete(ops, idx))


@pytest.mark.parametrize("shape", [(256, 16, 200000, 1 * MiB), (8, 16, 1000000, 1 * MiB), (4096, 16, 2000000, 64 * MiB),
                                   (96, 112, 20000, 600 * 1024), (64, 1500, 9000, 1 * MiB)])
def test_k_panels_reread_host_c_only_after_its_download(shape):
    """K split (kpanels > 1): S(c_ij) of panel p reads the host block R(c_ij) of panel p-1 wrote, possibly through another
    C buffer (h*w < n_sets, e.g. w == 1 with few rows).  The simulator tracks the host blocks (D2H = write, H2D_C = read);
    the schedule must order the two, and the check is not vacuous: without the extra waits the first three plans race."""
    M, N, K, budget = shape
    p = H.hclooc_plan(M, N, K, 1, 0, budget)
    assert p.kpanels > 1
    for ncs in (1, 3, 8):
        ops = H.hclooc_schedule(p, ncs)
        simulate(p, ops)
    if p.h * p.w < p.n_sets or (p.h * p.w) % p.n_sets:
        ops = H.hclooc_schedule(p, 8)
        c_stored = range(2 * p.n_sets, 3 * p.n_sets)
        # the waits of the H2D stream on c_stored that directly precede an H2D_C of a panel p > 0 and are not its own buffer's
        drop = []
        for i, o in enumerate(ops):
            if o["kind"] == K_H2D_C and o["step"] >= p.h * p.w:
                own = 2 * p.n_sets + (int(o["buf"]) - p.n_abuf)
                k = i - 1
                while k >= 0 and ops[k]["kind"] == K_WAIT and ops[k]["stream"] == 0:
                    if int(ops[k]["event"]) in c_stored and int(ops[k]["event"]) != own:
                        drop.append(k)
                    k -= 1
        if shape[:2] in ((256, 16), (8, 16), (4096, 16)):
            assert drop
        if drop:
            with pytest.raises(AssertionError, match="hazard on buffer \\('host C'"):
                simulate(p, np.delete(ops, drop))


def test_serpentine_order_reuses_resident_a_slices():
    """Rows run down the even columns of blocks and up the odd ones; the A slices still in the cache when a
    column ends are not uploaded again (hits need no S(a_i)), and every kernel still finds the right slice."""
    p = H.hclooc_plan(2000, 1500, 700, 1, 0, 6 * MiB)
    assert p.w >= 3 and p.h > p.n_abuf
    ops = H.hclooc_schedule(p, 4)
    simulate(p, ops)
    gemms = ops[ops["kind"] == K_GEMM]
    rows = (gemms["r0"] // p.mb).reshape(p.w, p.h)
    assert (rows[0] == np.arange(p.h)).all() and (rows[1] == np.arange(p.h)[::-1]).all() and (rows[2] == rows[0]).all()
    n_a = int((ops["kind"] == K_H2D_A).sum())
    assert n_a == p.h * p.w - (p.w - 1) * p.n_abuf
    # with everything cached (h <= n_abuf) A is uploaded exactly once
    q = H.hclooc_plan(256, 4096, 64, 0, 0, 3 * MiB)
    if q.w > 1 and q.h <= q.n_abuf and q.kpanels == 1:
        assert int((H.hclooc_schedule(q, 2)["kind"] == K_H2D_A).sum()) == q.h


@pytest.mark.parametrize("bbuf", [0, 1, 2])
def test_random_plans_simulate_clean(monkeypatch, bbuf):
    """Fuzz: random shapes, budgets, stream counts and buffer counts; every schedule must cover C exactly
    once per K panel, move exactly the plan's bytes and order every conflicting buffer access."""
    if bbuf:
        monkeypatch.setenv("HCLOOC_FORCE_BBUF", str(bbuf))
    rng = np.random.default_rng(100 + bbuf)
    done = 0
    for _ in range(120):
        M, N, K = (int(x) for x in rng.integers(1, 1200, 3))
        budget = int(rng.integers(128 * 1024, 6 * MiB))
        bnz, az = int(rng.integers(0, 2)), int(rng.integers(0, 10) == 0)
        sets = int(rng.choice([0, 2, 3, 5]))
        if sets:
            monkeypatch.setenv("HCLOOC_FORCE_SETS", str(sets))
        else:
            monkeypatch.delenv("HCLOOC_FORCE_SETS", raising=False)
        try:
            p = H.hclooc_plan(M, N, K, bnz, az, budget)
        except H.HclError:
            continue
        if p.n_steps > 600:
            continue
        simulate(p, H.hclooc_schedule(p, int(rng.integers(1, 9))))
        done += 1
    assert done > 40


def test_cached_slices_read_by_many_columns_then_overwritten(monkeypatch):
    """All A slices of a K panel stay cached and are read by every column of blocks (3+ readers per buffer,
    recorded alternately into two events); the next K panel then overwrites them.  The upload must wait for
    every reader, not just the last one."""
    monkeypatch.setenv("HCLOOC_FORCE_MB", "32")          # experiment knob: two row slices, both cached
    found = 0
    for budget in (1 * MiB, 1536 * 1024, 2 * MiB, 3 * MiB):
        p = H.hclooc_plan(64, 1500, 9000, 1, 0, budget)
        assert p.kpanels > 1 and p.w >= 3 and p.h <= p.n_abuf
        for ncs in (1, 4, 8):
            ops = H.hclooc_schedule(p, ncs)
            simulate(p, ops)
            assert int((ops["kind"] == K_H2D_A).sum()) == p.h * p.kpanels      # one upload per slice and panel
        found += 1
    assert found == 4


def test_streamk_steps_use_one_scratch_buffer_per_compute_stream():
    """Experiment knob HCLOOC_STREAMK_STEPS (read once per process, so in a subprocess): compute-bound plans run
    each step as one persistent stream-K launch; the schedule then uses as many compute streams as the plan has
    scratch buffers, and the scratch is part of the workspace."""
    import subprocess, sys
    code = ("import paper_1808_05056_b200 as H, numpy as np\n"
            "p = H.hclooc_plan(65536, 65536, 16384, 1, 0, 16 << 30)\n"
            "ops = H.hclooc_schedule(p, 8)\n"
            "print(p.ksplit, p.n_scratch, int(p.bytes_scratch > 0), sorted(set(int(x) for x in ops['stream'][ops['kind'] == 3])),"
            " int(p.workspace_bytes == p.n_bbuf * p.bytes_b_buf + p.n_abuf * p.bytes_a_buf + p.n_sets * p.bytes_c_buf + p.n_scratch * p.bytes_scratch))")
    out = subprocess.run([sys.executable, "-c", code], cwd=ROOT, env=dict(os.environ, HCLOOC_STREAMK_STEPS="1"),
                         capture_output=True, text=True, check=True).stdout.strip()
    assert out == "-1 2 1 [2, 3] 1", out


def test_direct_mode_is_chosen_only_where_copy_latency_dominates():
    """plan.direct (operands_on_device = 3: host matrices the device can address): the cost model takes it for
    BASELINE config 1 (512^3 under 1 MiB: hundreds of <= 64 KiB copies) and leaves configs 2-4 staged; the plan
    uses no device memory and counts every tile's own reads as host-link traffic."""
    MiB = 1 << 20
    p = H.hclooc_plan_ex(512, 512, 512, 1, 0, 1 * MiB, 3)
    assert p.direct == 1 and p.workspace_bytes == 0 and p.n_steps == 1 and p.h == p.w == p.kpanels == 1
    assert (p.direct_cm, p.direct_cn) == (4, 4)              # 4 x 4 tiles in one 16-CTA cluster: A and B cross the link once
    assert p.bytes_h2d == 8 * 3 * 512 * 512 and p.bytes_d2h == 8 * 512 * 512
    assert p.n_copies_h2d == 0 and p.n_copies_d2h == 0
    staged = H.hclooc_plan_ex(512, 512, 512, 1, 0, 1 * MiB, 0)
    assert staged.direct == 0 and p.t_model_s < staged.t_model_s
    for (M, N, K, budget) in ((8192, 8192, 8192, 256 * MiB), (32768, 32768, 32768, 4096 * MiB), (65536, 65536, 16384, 16384 * MiB)):
        q = H.hclooc_plan_ex(M, N, K, 1, 0, budget, 3)
        assert q.direct == 0 and q.workspace_bytes > 0
    forced = H.hclooc_plan_ex(8192, 8192, 8192, 0, 0, 256 * MiB, 4)
    assert forced.direct == 1 and forced.bytes_h2d == 8 * 2 * 16 * 8192 * 8192      # 64 x 64 tiles in 4 x 4 clusters
    # a budget too small for any staged plan is no obstacle: direct mode needs none
    tiny = H.hclooc_plan_ex(300, 300, 300, 1, 0, 4096, 3)
    assert tiny.direct == 1


def test_plans_for_transposed_operands_keep_the_stored_layout():
    """hclooc_plan_trans: an A slice of a transposed A is kb x mb (lda_dev >= mb), a B slice of a transposed B is nb x kb
    (ldb_dev >= kb); everything still fits the budget and the traffic is that of the untransposed plan."""
    MiB = 1 << 20
    for (M, N, K, budget) in ((512, 512, 512, 1 * MiB), (8192, 8192, 8192, 256 * MiB), (3000, 5000, 7000, 64 * MiB), (96, 112, 20000, 900 * 1024)):
        base = H.hclooc_plan_trans(M, N, K, 1, 0, budget, 0, 0, 0)
        same = H.hclooc_plan_ex(M, N, K, 1, 0, budget, 0)
        assert bytes(base) == bytes(same)
        for ta, tb in ((1, 0), (0, 1), (1, 1)):
            p = H.hclooc_plan_trans(M, N, K, 1, 0, budget, 0, ta, tb)
            assert p.trans == ta + 2 * tb and p.workspace_bytes <= budget
            assert p.workspace_bytes == p.n_bbuf * p.bytes_b_buf + p.n_abuf * p.bytes_a_buf + p.n_sets * p.bytes_c_buf
            if ta:
                assert p.lda_dev >= p.mb and p.lda_dev % 16 == 0 and p.bytes_a_buf >= 8 * p.kb * p.lda_dev
            else:
                assert p.lda_dev >= p.kb and p.bytes_a_buf >= 8 * p.mb * p.lda_dev
            if tb:
                assert p.ldb_dev >= p.kb and p.ldb_dev % 16 == 0 and p.bytes_b_buf >= 8 * p.nb * p.ldb_dev
            else:
                assert p.ldb_dev >= p.nb and p.bytes_b_buf >= 8 * p.kb * p.ldb_dev
            assert p.bytes_d2h == 8 * M * N * p.kpanels and p.n_steps == p.h * p.w * p.kpanels
    with pytest.raises(H.HclError) as e:
        H.hclooc_plan_trans(8, 8, 8, 1, 0, 1 * MiB, 0, 2, 0)
    assert e.value.status == -8


@pytest.mark.parametrize("tri", [1, 2])
def test_triangle_schedule_has_steps_only_for_blocks_that_touch_the_triangle(tri):
    """plan.tri (hclooc_dsyrk): a block of C wholly in the triangle that is not referenced is not a step -- no upload, no
    kernel, no download; every other block is computed exactly once per K panel, in the usual buffers and event order."""
    MiB = 1 << 20
    for (N, K, budget) in ((3000, 700, 8 * MiB), (4096, 4096, 64 * MiB), (1000, 30000, 2 * MiB)):
        p = H.hclooc_plan_ex(N, N, K, 1, 0, budget, 0)
        full = H.hclooc_schedule(p, 8)
        p.tri = tri
        ops = H.hclooc_schedule(p, 8)
        gemm = ops[ops["kind"] == 3]
        seen = {}
        for o in gemm:
            i, j, pnl = int(o["r0"]) // p.mb, int(o["c0"]) // p.nb, int(o["k0"]) // p.kb
            seen[(i, j, pnl)] = seen.get((i, j, pnl), 0) + 1
        for i in range(p.h):
            for j in range(p.w):
                r0, r1 = i * p.mb, min(N, (i + 1) * p.mb)
                c0, c1 = j * p.nb, min(N, (j + 1) * p.nb)
                touches = (c0 <= r1 - 1) if tri == 1 else (c1 - 1 >= r0)
                for pnl in range(p.kpanels):
                    assert seen.get((i, j, pnl), 0) == (1 if touches else 0), (tri, i, j, pnl)
        up_c, down_c = ops[ops["kind"] == 2], ops[ops["kind"] == 4]
        assert len(down_c) == len(gemm) and len(up_c) == len(gemm)          # beta != 0: one upload and one download per live block
        assert len(gemm) < len(full[full["kind"] == 3]) or p.h * p.w == 1
        # every B slice is still loaded whole, once per K panel
        b = ops[ops["kind"] == 1]
        assert int((b["nr"] * b["nc"]).sum()) == K * N


def test_dtrsm_plan_respects_the_budget_and_its_own_rules():
    """hclooc_dtrsm_plan (host arithmetic of hclooc_dtrsm): block-row height, chunk width, resident block rows and the device
    bytes of the diagonal phase over a grid of shapes and budgets."""
    import paper_1808_05056_b200 as H
    MiB = 1 << 20
    seen = set()
    for M in (1, 31, 77, 128, 300, 1000, 4096, 6000, 32768, 163840):
        for N in (1, 64, 333, 4500, 32768):
            for budget in (64 * 1024, 512 * 1024, 1 * MiB, 3 * MiB, 48 * MiB, 256 * MiB, 1024 * MiB, 4096 * MiB, 170 * 1024 * MiB):
                for own in (True, False):
                    NB, chunk, res, dev = H.hclooc_dtrsm_plan(M, N, budget, own)
                    assert 1 <= NB <= min(M, 8192 if own else 4096) and NB * NB * 8 <= max(budget // 2, 32 * 32 * 8)
                    assert NB == M or NB % 128 == 0 or (NB < 128 and NB % 32 == 0)
                    assert chunk % 64 == 0 and 64 <= chunk <= (N + 63) // 64 * 64
                    assert res in (0, 1, 2) and (own or res == 0)
                    nblk = -(-M // NB)
                    assert res < 2 or nblk > 1
                    if res:
                        assert dev + budget // 4 <= budget                       # the DGEMM pipeline keeps a quarter
                        assert dev >= res * NB * N * 8 + NB * NB * 8
                    else:
                        assert dev <= budget and dev >= NB * NB * 8 + 2 * NB * chunk * 8
                    seen.add(res)
    assert seen == {0, 1, 2}
    # the cases the GPU tests and the profile rely on
    assert H.hclooc_dtrsm_plan(32768, 32768, 4096 * MiB)[:3] == (4096, 16384, 2)
    assert H.hclooc_dtrsm_plan(16384, 16384, 256 * MiB)[::2] == (4096, 0)
    assert H.hclooc_dtrsm_plan(6000, 4500, 1024 * MiB)[::2] == (6000, 1)          # 8192-row block rows allowed: one block row
    assert H.hclooc_dtrsm_plan(10000, 2000, 2048 * MiB)[::2] == (8192, 2)
    assert H.hclooc_dtrsm_plan(32768, 32768, 16384 * MiB)[::2] == (8192, 2)
    assert H.hclooc_dtrsm_plan(32768, 32768, 16384 * MiB, False)[::2] == (4096, 0)
    assert H.hclooc_dtrsm_plan(3000, 300, 48 * MiB, False)[2] == 0
    for args, code in (((0, 5, MiB), -1), ((5, 0, MiB), -2), ((200, 100, 16 * 1024), 1)):
        with pytest.raises(H.HclError) as e:
            H.hclooc_dtrsm_plan(*args)
        assert e.value.status == code
