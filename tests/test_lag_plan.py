"""Host logic of step S5 (one accumulator per requested lag, every pair counted once):
invariants of the lag plan nfs_create builds — checked without a GPU through nfs_plan_lags.

A plan cuts the sorted lag list into tasks (one consumer warp each) and tasks into groups (one CTA per
group and pixel tile).  Whatever the list: every lag belongs to exactly one task, every task is placed on
exactly one consumer warp of its group, exactly one task accumulates the I sums, and the group's window
fits the shared memory the plan reports.
"""
import numpy as np
import pytest

from paper_1209_3362_b200 import binding, synth

KG = 13          # lags per register-window task (nfs_common.cuh: kG)
KS = 6           # lags per lag-list task (kSparseMax)
MAX_TASKS = 8    # consumer warps per CTA (kMaxTasks)
SMEM_SM = 233472   # B200: shared memory per SM
SMEM_OPTIN = 232448  # B200: opt-in maximum per CTA


def check_plan(lags, plan):
    lags = list(lags)
    groups, tasks = plan["groups"], plan["tasks"]
    covered = np.zeros(len(lags), dtype=int)
    n_I = 0
    seen_tasks = set()
    assert sum(g["flags"] & 1 for g in groups) == 1, "exactly one group accumulates the I sums"
    for g in groups:
        assert 1 <= g["ntasks"] <= MAX_TASKS
        placed = [w for w in g["warp_task"] if w >= 0]
        assert sorted(placed) == list(range(g["ntasks"])), "every task of a group runs on exactly one warp"
        assert all(w < 0 for w in g["warp_task"][MAX_TASKS:])
        lo, hi = 1 << 30, 0
        has_I = 0
        for k in range(g["ntasks"]):
            ti = g["task0"] + k
            assert ti not in seen_tasks
            seen_tasks.add(ti)
            t = tasks[ti]
            assert 0 <= t["cnt"] <= (KG if (t["kind"] & 1) == 0 else KS)
            has_I += (t["kind"] >> 1) & 1
            if t["cnt"] == 0:
                assert t["kind"] == 3, "a task without lags only accumulates I"
                continue
            own = lags[t["l0"]:t["l0"] + t["cnt"]]
            assert len(own) == t["cnt"] and own[0] == t["tau0"]
            if (t["kind"] & 1) == 0:
                assert own == list(range(t["tau0"], t["tau0"] + t["cnt"])), "a dense task is a run of consecutive lags"
            covered[t["l0"]:t["l0"] + t["cnt"]] += 1
            lo, hi = min(lo, own[0]), max(hi, own[-1])
        assert has_I == (g["flags"] & 1)
        n_I += has_I
        assert (g["tau_min"], g["tau_max"]) == (lo, hi)
    assert n_I == 1
    # persistent CTAs: contiguous shares, at least one per group, all resident slots handed out
    at = 0
    for g in groups:
        assert g["cta0"] == at and g["nctas"] >= 1
        at += g["nctas"]
    assert at == max(2 * 148, len(groups))
    assert len(seen_tasks) == len(tasks)
    assert np.all(covered == 1), "every lag is accumulated by exactly one task"
    assert 2 <= plan["stages"] <= 8
    assert 0 < plan["smem"] <= SMEM_OPTIN


@pytest.mark.parametrize("ci", [0, 1, 2, 3, 4])
def test_plan_of_baseline_configs(ci):
    cfg = synth.config(ci)
    plan = binding.nfs_plan_lags(cfg.lags, SMEM_SM, SMEM_OPTIN)
    check_plan(cfg.lags, plan)
    if ci in (1, 2):  # 100 consecutive lags: 8 register-window tasks in one group, two CTAs per SM
        assert len(plan["groups"]) == 1 and len(plan["tasks"]) == 8
        assert plan["smem"] <= SMEM_SM // 2 - 1024


@pytest.mark.parametrize("seed", range(12))
def test_plan_of_random_lag_lists(seed):
    rng = np.random.default_rng(seed)
    n = int(rng.integers(1, 120))
    top = int(rng.choice([n, 2 * n, 10 * n, 2000]))
    lags = np.sort(rng.choice(np.arange(1, max(top, n) + 1), size=n, replace=False))
    plan = binding.nfs_plan_lags(lags, SMEM_SM, SMEM_OPTIN)
    check_plan(lags, plan)


def test_plan_edge_cases():
    for lags in ([1], [7], [1, 2], list(range(1, 14)), list(range(1, 15)), [1, 1000], list(range(5, 12)) + [400, 401]):
        check_plan(lags, binding.nfs_plan_lags(lags, SMEM_SM, SMEM_OPTIN))
    with pytest.raises(binding.NFSError):
        binding.nfs_plan_lags([3, 2], SMEM_SM, SMEM_OPTIN)
    with pytest.raises(binding.NFSError):
        binding.nfs_plan_lags([0, 1], SMEM_SM, SMEM_OPTIN)
