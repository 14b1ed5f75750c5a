"""Host logic of hclooc_dgetrf (no GPU): hclooc_dgetrf_plan -- the panel width and the device bytes the routine keeps for itself."""
import pytest

import paper_1808_05056_b200 as H

MiB = 1 << 20


@pytest.mark.parametrize("M,N", [(1, 1), (5, 3), (300, 300), (1000, 1000), (1100, 1500), (8192, 8192), (32768, 32768), (65536, 16384), (147456, 147456)])
def test_dgetrf_plan_respects_the_budget_and_grows_with_it(M, N):
    last_nb = 0
    for budget in (1 * MiB, 3 * MiB, 24 * MiB, 256 * MiB, 1 << 30, 4 << 30, 16 << 30, 150 << 30):
        try:
            NB, reserved = H.hclooc_dgetrf_plan(M, N, budget)
        except H.HclError as e:
            assert e.status == 1                                     # HCLOOC_ERR_BUDGET: not even two 32-column panels
            assert 2 * M * 32 * 8 > budget * 5 // 8 - (1 << 18) or last_nb == 0
            continue
        assert 1 <= NB <= min(N, 4096) and (NB == N or NB % 32 == 0)
        assert NB >= last_nb                                         # a larger budget never narrows the panel
        last_nb = NB
        npanels = -(-N // NB)
        assert reserved <= budget * 7 // 8
        assert reserved >= min(npanels, 2) * M * NB * 8              # at least two panels (one if one covers the matrix)
        if npanels >= 3 and reserved >= 3 * M * NB * 8:              # three resident panels: only inside 7/8 of the budget
            assert 3 * M * NB * 8 <= budget * 7 // 8
        if npanels >= 2 and reserved < 3 * M * NB * 8:               # two: inside 5/8
            assert reserved <= budget * 5 // 8


def test_dgetrf_plan_knob_and_errors(monkeypatch):
    nb3, r3 = H.hclooc_dgetrf_plan(32768, 32768, 4 << 30)
    monkeypatch.setenv("HCLOOC_GETRF_PANELS", "2")
    nb2, r2 = H.hclooc_dgetrf_plan(32768, 32768, 4 << 30)
    assert nb3 == nb2 == 4096 and r3 - r2 == 32768 * 4096 * 8         # the third panel
    monkeypatch.delenv("HCLOOC_GETRF_PANELS")
    for args, code in (((0, 5, MiB), -1), ((5, 0, MiB), -2)):
        with pytest.raises(H.HclError) as e:
            H.hclooc_dgetrf_plan(*args)
        assert e.value.status == code
    with pytest.raises(H.HclError) as e:
        H.hclooc_dgetrf_plan(100000, 64, MiB)
    assert e.value.status == 1
