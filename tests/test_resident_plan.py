"""The resident schedule's host logic (resident.cu, hclooc_plan_resident; DESIGN.md section 7 "Resident schedule"): no GPU needed.
What the executor relies on: the K panels tile [0, K) exactly and are graded, the device copies + scratch + staging ring stay within
the budget, phase 2 owns at least the last panel, and the schedule is offered only where it can pay."""
import numpy as np
import pytest

import paper_1808_05056_b200 as H

GB = 10 ** 9


@pytest.fixture(autouse=True)
def no_env(monkeypatch):
    monkeypatch.delenv("HCLOOC_RESIDENT", raising=False)
    monkeypatch.delenv("HCLOOC_RESIDENT_KB", raising=False)


def shape_ok(M, N, K, beta_nonzero, budget, p):
    k0 = np.array(p.panel_k0[:p.npanels]); kk = np.array(p.panel_kk[:p.npanels])
    assert p.npanels >= 2 and k0[0] == 0 and (k0[1:] == k0[:-1] + kk[:-1]).all() and k0[-1] + kk[-1] == K      # the panels tile K
    assert (kk[:-1] % 32 == 0).all() and (kk > 0).all()                       # whole k blocks of the kernel, except a ragged last panel
    assert kk[0] in (256, 512) and kk[:-1].max() <= p.kb <= 2048
    assert (np.diff(kk[:-1]) >= 0).all() and (kk[:-1][1:] <= 2 * kk[:-1][:-1]).all()   # graded: never shrinking, at most doubling
    assert 1 <= p.p_switch <= p.npanels - 1                                      # phase 2 owns at least the last panel
    assert p.h == -(-M // p.mb) and p.h <= 16 and (p.mb % 128 == 0 or p.mb == M)
    assert p.lda_dev >= K and p.ldb_dev >= N and p.ldc_dev >= N and p.lda_dev % 16 == p.ldb_dev % 16 == p.ldc_dev % 16 == 0
    need = 8 * (M * p.lda_dev + K * p.ldb_dev + M * p.ldc_dev) + p.ring * 8 * p.mb * p.ldc_dev
    assert need <= p.workspace_bytes <= budget                                   # + the stream-K scratch and slack
    assert p.ring == (0 if not beta_nonzero else min(p.h, p.ring)) and (not beta_nonzero or p.ring >= min(2, p.h))
    assert p.t_model_s >= max(p.t_flop_s, 0.0) and p.t_flop_s == pytest.approx(2.0 * M * N * K / 37.17e12, rel=0.2)


@pytest.mark.parametrize("M,N,K,beta", [(8192, 8192, 8192, 1), (4096, 4096, 4096, 1), (12288, 12288, 12288, 0), (16384, 16384, 16384, 1),
                                        (5000, 3000, 7001, 1), (1024, 20000, 2048, 1), (20480, 20480, 20480, 1)])
def test_shape_of_the_resident_schedule(M, N, K, beta):
    budget = int(12.2 * GB)
    p = H.hclooc_plan_resident(M, N, K, beta, budget, 0.0)       # no slice model to compare with: applies where it fits and is not small
    assert p.applies == 1
    shape_ok(M, N, K, beta, budget, p)


def test_it_is_offered_only_where_it_fits_and_can_pay(monkeypatch):
    n = 8192
    fits = H.hclooc_plan_resident(n, n, n, 1, 2 * GB, 0.0)
    assert fits.applies == 1 and fits.workspace_bytes <= 2 * GB
    tight = H.hclooc_plan_resident(n, n, n, 1, 3 * 8 * n * n + 10 * 2 ** 20, 0.0)     # the three matrices fit, the scratch and the ring do not
    assert tight.applies == 0 and tight.npanels == 0
    assert H.hclooc_plan_resident(n, n, n, 0, 3 * 8 * n * n + 64 * 2 ** 20, 0.0).applies == 1   # beta == 0 needs no ring
    # against the slice plan's estimate: taken only below 0.985 of it
    t = fits.t_model_s
    assert H.hclooc_plan_resident(n, n, n, 1, 2 * GB, t / 0.98).applies == 1
    assert H.hclooc_plan_resident(n, n, n, 1, 2 * GB, t / 0.99).applies == 0
    # small calls are latency bound: never by itself, the shape is still described; the environment forces the answer
    small = H.hclooc_plan_resident(1000, 1000, 1000, 1, 2 * GB, 0.0)
    assert small.applies == 0 and small.npanels >= 2
    monkeypatch.setenv("HCLOOC_RESIDENT", "1")
    forced = H.hclooc_plan_resident(1000, 1000, 1000, 1, 2 * GB, 1e-9)
    assert forced.applies == 1
    shape_ok(1000, 1000, 1000, 1, 2 * GB, forced)
    monkeypatch.setenv("HCLOOC_RESIDENT", "0")
    assert H.hclooc_plan_resident(n, n, n, 1, 2 * GB, 0.0).applies == 0
    monkeypatch.delenv("HCLOOC_RESIDENT")
    assert H.hclooc_plan_resident(300, 200, 400, 1, 2 * GB, 0.0).npanels == 0          # below the hard minimum: not described at all
    for args, code in (((0, n, n, 1, GB, 0.0), -1), ((n, 0, n, 1, GB, 0.0), -2), ((n, n, 0, 1, GB, 0.0), -3)):
        with pytest.raises(H.HclError) as e:
            H.hclooc_plan_resident(*args)
        assert e.value.status == code


def test_compute_bound_calls_start_with_short_panels_and_switch_late():
    """N = 8192 under PCIe-class links is balanced: the kernels lag the uploads, so phase 1 runs past the middle of K; a
    link-bound call (N = 4096) starts with 512-column panels (2 KiB rows cost link rate) and switches at the last panel."""
    p8 = H.hclooc_plan_resident(8192, 8192, 8192, 1, int(12.2 * GB), 0.0)
    assert p8.panel_kk[0] == 256 and p8.kb == 1024 and 0.4 * 8192 <= p8.panel_k0[p8.p_switch] < 8192
    p4 = H.hclooc_plan_resident(4096, 4096, 4096, 1, int(12.2 * GB), 0.0)
    assert p4.panel_kk[0] == 512 and p4.p_switch == p4.npanels - 1
    assert p4.t_model_s > p4.t_flop_s * 1.5                                       # the link is the bound there


# ------------------------------------------------------------------------------------------------ the schedule under a hazard check
# hclooc_resident_schedule is the exact op list dgemm_resident issues (resident.cu builds it and walks it).  Below: a vector-clock
# simulation of CUDA stream semantics over that list -- program order inside a stream, record -> wait edges between streams -- that
# requires every pair of conflicting accesses to a device buffer region or to a host row block of C to be ORDERED
# ("data stored in device buffers is not overwritten until kernel executions that operate on the data have
# completed"), every element of the product to be computed exactly once, and C to come down only after beta * C0 went in.
H2D_A, H2D_B, H2D_C, GEMM, D2H_C, WAIT, RECORD, AXPY = range(8)


def accesses(o, M, N, K):
    """[(buffer, (r0, r1), (c0, c1), is_write)] of one operation.  Buffers: 'A', 'B', 'C' (device copies), ('S', slot), 'hostC'."""
    r = (int(o["r0"]), int(o["r0"] + o["nr"])); k = (int(o["k0"]), int(o["k0"] + o["kk"]))
    kind = int(o["kind"])
    if kind == H2D_A:
        return [("A", (0, M), k, True)]
    if kind == H2D_B:
        return [("B", k, (0, N), True)]
    if kind == GEMM:
        return [("A", r, k, False), ("B", k, (0, N), False), ("C", r, (0, N), True)] + ([("C", r, (0, N), False)] if o["beta"] != 0 else [])
    if kind == H2D_C:
        return [("hostC", r, (0, N), False), (("S", int(o["buf"]) - 3), (0, 1), (0, 1), True)]
    if kind == AXPY:
        return [(("S", int(o["buf"]) - 3), (0, 1), (0, 1), False), ("C", r, (0, N), True), ("C", r, (0, N), False)]
    if kind == D2H_C:
        return [("C", r, (0, N), False), ("hostC", r, (0, N), True)]
    return []


def simulate_resident(ops, M, N, K, beta_nonzero, drop=None):
    """Returns the list of violations (empty = the schedule is sound).  drop: index of a WAIT to ignore (mutation tests)."""
    streams = sorted({int(o["stream"]) for o in ops})
    sid = {s: i for i, s in enumerate(streams)}
    clock = {s: [0] * len(streams) for s in streams}
    ev_clock, done, bad = {}, [], []
    leq = lambda a, b: all(x <= y for x, y in zip(a, b))
    for idx, o in enumerate(ops):
        s, kind = int(o["stream"]), int(o["kind"])
        if kind == WAIT:
            if idx == drop:
                continue
            if int(o["event"]) not in ev_clock:
                bad.append(f"op {idx}: wait for event {int(o['event'])} that has not been recorded yet (a no-op in CUDA)")
                continue
            clock[s] = [max(a, b) for a, b in zip(clock[s], ev_clock[int(o["event"])])]
            continue
        if kind == RECORD:
            ev_clock[int(o["event"])] = list(clock[s])
            continue
        clock[s][sid[s]] += 1
        mine = accesses(o, M, N, K)
        for (jdx, cj, acc_j) in done:
            if leq(cj, clock[s]):
                continue                                                      # ordered before this op
            for (b1, r1, c1, w1) in mine:
                for (b2, r2, c2, w2) in acc_j:
                    if b1 == b2 and (w1 or w2) and r1[0] < r2[1] and r2[0] < r1[1] and c1[0] < c2[1] and c2[0] < c1[1]:
                        bad.append(f"ops {jdx} and {idx} touch {b1} rows {r1}/{r2} cols {c1}/{c2} unordered")
        done.append((idx, list(clock[s]), mine))
    # coverage: every (row, k) once, first touch of a row with beta 0, AXPY once per row block after its last GEMM, download last
    cover = np.zeros((M, K), dtype=np.int32)
    started = np.zeros(M, dtype=bool); joined = np.zeros(M, dtype=np.int32); down = np.zeros(M, dtype=np.int32)
    for idx, o in enumerate(ops):
        kind = int(o["kind"]); r0, r1 = int(o["r0"]), int(o["r0"] + o["nr"])
        if kind == GEMM:
            k0, k1 = int(o["k0"]), int(o["k0"] + o["kk"])
            cover[r0:r1, k0:k1] += 1
            if o["beta"] == 0 and started[r0:r1].any():
                bad.append(f"op {idx}: beta = 0 over rows that already hold partial sums")
            if o["beta"] != 0 and not started[r0:r1].all():
                bad.append(f"op {idx}: accumulates into rows that were never initialised")
            if joined[r0:r1].any() or down[r0:r1].any():
                bad.append(f"op {idx}: GEMM after the rows were joined with C0 / downloaded")
            started[r0:r1] = True
        elif kind == AXPY:
            if (cover[r0:r1] != 1).any():
                bad.append(f"op {idx}: beta * C0 added before the products of the rows are complete")
            joined[r0:r1] += 1
        elif kind == D2H_C:
            if (cover[r0:r1] != 1).any() or (beta_nonzero and (joined[r0:r1] != 1).any()):
                bad.append(f"op {idx}: rows downloaded before they are final")
            down[r0:r1] += 1
    if (cover != 1).any():
        bad.append("some (row, k) not covered exactly once")
    if (down != 1).any() or (joined != (1 if beta_nonzero else 0)).any():
        bad.append("row blocks not joined / downloaded exactly once")
    return bad


@pytest.mark.parametrize("M,N,K,beta,budget,n_compute", [
    (8192, 8192, 8192, 1, int(12.2 * GB), 8),
    (4096, 4096, 4096, 1, int(12.2 * GB), 8),         # link bound: phase 2 is the last panel only
    (5000, 3000, 7001, 1, 2 * GB, 8),                 # ragged rows and a ragged last panel
    (12288, 12288, 12288, 0, int(12.2 * GB), 8),      # beta == 0: no staging, no AXPY
    (8192, 8192, 8192, 1, int(12.2 * GB), 1),         # a context with one compute stream
    (4096, 1024, 1536, 1, 160 * 2 ** 20, 8),          # the staging ring is shorter than the row blocks: slots are reused
])
def test_resident_schedule_has_no_unordered_conflict_and_covers_the_product(monkeypatch, M, N, K, beta, budget, n_compute):
    monkeypatch.setenv("HCLOOC_RESIDENT", "1")
    p = H.hclooc_plan_resident(M, N, K, beta, budget, 0.0)
    assert p.applies == 1
    ops = H.hclooc_resident_schedule(p, M, N, K, beta, n_compute)
    assert simulate_resident(ops, M, N, K, bool(beta)) == []
    kinds = ops["kind"]
    assert (kinds == H2D_A).sum() == p.npanels == (kinds == H2D_B).sum() and (kinds == D2H_C).sum() == p.h
    assert (kinds == GEMM).sum() == p.p_switch + p.h and (kinds == AXPY).sum() == (p.h if beta else 0) == (kinds == H2D_C).sum()
    assert set(ops["stream"][kinds == GEMM]) <= ({2, 3} if n_compute >= 2 else {2})
    if beta and p.ring < p.h:
        assert (ops["buf"][kinds == H2D_C] - 3).max() == p.ring - 1             # the slots are reused round robin


def test_the_hazard_check_is_not_vacuous(monkeypatch):
    """Dropping any single wait of the schedule must be noticed -- as an unordered conflict or as work done on incomplete data --
    except the few waits that another edge already implies (at most one in twenty)."""
    monkeypatch.setenv("HCLOOC_RESIDENT", "1")
    M, N, K = 4096, 1024, 1536
    p = H.hclooc_plan_resident(M, N, K, 1, 160 * 2 ** 20, 0.0)
    ops = H.hclooc_resident_schedule(p, M, N, K, 1, 8)
    assert p.ring < p.h and simulate_resident(ops, M, N, K, True) == []
    waits = [i for i, o in enumerate(ops) if int(o["kind"]) == WAIT]
    unnoticed = [i for i in waits if simulate_resident(ops, M, N, K, True, drop=i) == []]
    assert len(waits) >= 40 and len(unnoticed) <= len(waits) // 20, (len(waits), unnoticed)
    by_event = lambda lo, hi: [i for i in waits if lo <= int(ops[i]["event"]) < hi]
    np_, h = p.npanels, p.h
    for name, idxs in (("panel uploaded", by_event(0, np_)), ("C0 block uploaded", by_event(np_, np_ + h)),
                       ("staging slot free", by_event(np_ + h, np_ + 2 * h)), ("row block finished", by_event(np_ + 2 * h, np_ + 3 * h))):
        assert idxs and all(i not in unnoticed for i in idxs[1:]), name
