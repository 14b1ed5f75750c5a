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
