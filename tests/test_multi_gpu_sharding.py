"""N > 1: one process per GPU, each owning a band of rows of A and C and all of B (PAPER.md:289,
:293: the row blocks of C are independent, so the path shards with no exchange step and no collective).

CPU part (gloo, world_size 2): the band arithmetic of hclooc_shard_rows, the rank-offset generation of the
bands (what bench.py's ranks do) and the gather of the results -- each rank computes ITS band with the oracle
standing in for the device call, the bands are gathered over gloo and must equal the oracle on the whole
problem bit for bit (same per-element operation order, whatever the banding).
"""
import os
import socket

import numpy as np
import pytest

import paper_1808_05056_b200 as H


def test_shard_rows_covers_every_row_once():
    rng = np.random.default_rng(5)
    for _ in range(300):
        M = int(rng.integers(0, 5000)); world = int(rng.integers(1, 9)); align = int(rng.choice([1, 16, 128]))
        bands = [H.hclooc_shard_rows(M, world, r, align) for r in range(world)]
        pos = 0
        for r0, n in bands:
            assert r0 == pos and n >= 0
            pos += n
        assert pos == M
        sizes = [n for _, n in bands]
        nonempty = [n for n in sizes if n]
        assert all(n % align == 0 for n in nonempty[:-1])                    # only the last band may be ragged
        if nonempty:
            assert max(sizes) - min(nonempty[:-1] or nonempty) <= align or len(nonempty) == 1   # balanced to one unit
    with pytest.raises(H.HclError):
        H.hclooc_shard_rows(10, 2, 2)
    with pytest.raises(H.HclError):
        H.hclooc_shard_rows(10, 0, 0)
    assert H.hclooc_shard_rows(65536, 8, 3) == (3 * 8192, 8192)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, M, N, K, alpha, beta, seed, out_q):
    import torch
    import torch.distributed as dist
    import oracle
    import synthgen
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        row0, rows = H.hclooc_shard_rows(M, world, rank, 16)
        # the band of A and C this rank owns, generated at its row offset; B whole (every rank needs all of it)
        A = synthgen.fill(np.empty((rows, K)), seed, "A", "uniform", row0=row0, logical_cols=K)
        B = synthgen.fill(np.empty((K, N)), seed, "B", "uniform")
        C = synthgen.fill(np.empty((rows, N)), seed, "C", "uniform", row0=row0, logical_cols=N)
        if rows:
            oracle.dgemm(alpha, A, B, beta, C)                                # stands in for hclooc_dgemm on this rank's GPU
        # gather the bands on every rank (padded to the largest band)
        sizes = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
        dist.all_gather(sizes, torch.tensor([rows], dtype=torch.int64))
        top = max(int(s.item()) for s in sizes)
        pad = torch.zeros(top, N, dtype=torch.float64)
        pad[:rows] = torch.from_numpy(C)
        parts = [torch.zeros(top, N, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(parts, pad)
        full = np.vstack([p[: int(s.item())].numpy() for p, s in zip(parts, sizes)])
        if rank == 0:
            Af = synthgen.fill(np.empty((M, K)), seed, "A", "uniform")
            Cf = synthgen.fill(np.empty((M, N)), seed, "C", "uniform")
            oracle.dgemm(alpha, Af, B, beta, Cf)
            out_q.put(("ok", bool(np.array_equal(full, Cf)), full.shape, [int(s.item()) for s in sizes]))
    except Exception as e:                                                   # pragma: no cover
        if rank == 0:
            out_q.put(("error", repr(e)))
        raise
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(180)
def test_two_ranks_over_gloo_reproduce_the_whole_problem():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    M, N, K = 301, 70, 50
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, M, N, K, 1.5, -0.5, 4242, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = q.get(timeout=150)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0] == "ok", res
    assert res[1] is True and res[2] == (M, N) and sum(res[3]) == M and res[3] == [160, 141]


@pytest.mark.gpu
@pytest.mark.parametrize("M,world,dist", [(1000, 3, "uniform"), (1000, 3, "int"), (777, 2, "uniform"), (130, 4, "int")])
def test_bands_through_the_cuda_path_equal_the_single_call_bitwise(M, world, dist):
    """What bench.py's ranks do, on one GPU: the M rows (ragged, align 128) are cut into `world` bands with hclooc_shard_rows and
    hclooc_dgemm runs on each band's POINTERS into the same host matrices (rows row0.. of A and C, all of B).  The stacked
    bands must equal the single call bit for bit (K is not split, so every element sums in the same order whatever the banding)
    and the oracle within the gate (exactly on integers).  Trailing ranks with no rows do nothing."""
    import oracle
    import synthgen
    N, K, alpha, beta, budget = 390, 300, 1.5, -0.5, 2 << 20
    A, B, C = H.HostMatrix(M, K, K + 2), H.HostMatrix(K, N, N + 4), H.HostMatrix(M, N, N + 6)
    for X in (A, B, C):
        X.array[...] = np.nan
    synthgen.fill(A.array, 51, "A", dist, cols=K); synthgen.fill(B.array, 51, "B", dist, cols=N); synthgen.fill(C.array, 51, "C", dist, cols=N)
    C0 = C.view.copy()
    ref = C0.copy()
    D = oracle.dgemm(alpha, A.view, B.view, beta, ref, want_denominator=True)
    st = H.hclooc_dgemm_ex(None, M, N, K, alpha, A, A.ld, B, B.ld, beta, C, C.ld, budget)
    assert st.plan.kpanels == 1
    whole = C.view.copy()
    C.view[...] = C0
    covered = 0
    for rank in range(world):
        row0, rows = H.hclooc_shard_rows(M, world, rank, 128)
        assert row0 == covered
        covered += rows
        st = H.hclooc_dgemm_ex(None, rows, N, K, alpha, A.ptr + 8 * row0 * A.ld, A.ld, B, B.ld, beta, C.ptr + 8 * row0 * C.ld, C.ld, budget)
        assert st.bytes_d2h == rows * N * 8
    assert covered == M
    assert np.array_equal(C.view.view(np.uint64), whole.view(np.uint64))
    assert np.isnan(C.array[:, N:]).all()
    if dist == "int":
        assert np.array_equal(C.view, ref)
    else:
        ok, worst = oracle.within_gate(C.view, ref, D, 1e-13)
        assert ok, worst
