"""Host logic of step S5 (one accumulator per requested lag, every pair counted once):
invariants of the lag plan nfs_create builds — checked without a GPU through nfs_plan_lags.

A plan cuts the sorted lag list into tasks (one consumer warp each per 32-pixel sub-tile) and tasks into groups (one
CTA per group and pixel tile).  Whatever the list: every lag belongs to exactly one task, every task is placed on
exactly one task slot of its group, exactly one task accumulates the I sums, and the group's window
fits the shared memory the plan reports.
"""
import numpy as np
import pytest

import synth
from paper_1209_3362_b200 import binding

KG = 13          # lags per register-window task (nfs_common.cuh: kG)
KS = 6           # lags per lag-list task (kSparseMax)
N_SM = 148
P_1024 = 1024 * 513   # Fourier pixels of a 1024 x 1024 frame
SMEM_SM = 233472   # B200: shared memory per SM
SMEM_OPTIN = 232448  # B200: opt-in maximum per CTA


def plan_of(lags, n_px=P_1024):
    return binding.nfs_plan_lags(lags, n_px, SMEM_SM, SMEM_OPTIN, N_SM)


def check_plan(lags, plan, n_px=P_1024):
    lags = list(lags)
    groups, tasks = plan["groups"], plan["tasks"]
    covered = np.zeros(len(lags), dtype=int)
    n_I2 = n_I1 = 0
    seen_tasks = set()
    assert sum(g["flags"] & 1 for g in groups) == 1, "exactly one group accumulates the I sums"
    MAX_TASKS = plan["slots"]   # task slots per group: 8, or 16 for one 32-pixel CTA of 16 consumer warps per SM
    assert MAX_TASKS in (8, 16) and (MAX_TASKS == 8 or (plan["tile_px"], plan["ctas_per_sm"]) == (32, 1))
    for g in groups:
        assert 1 <= g["ntasks"] <= MAX_TASKS
        placed = [w for w in g["warp_task"] if w >= 0]
        assert sorted(placed) == list(range(g["ntasks"])), "every task of a group runs on exactly one warp"
        assert all(w < 0 for w in g["warp_task"][MAX_TASKS:])
        lo, hi = 1 << 30, 0
        has_I2 = has_I1 = 0
        for k in range(g["ntasks"]):
            ti = g["task0"] + k
            assert ti not in seen_tasks
            seen_tasks.add(ti)
            t = tasks[ti]
            assert 0 <= t["cnt"] <= (KG if (t["kind"] & 1) == 0 else KS)
            if (t["kind"] & 1) == 0:
                assert t["cnt"] >= 2, "a register-window task has a direct lag and at least one neighbour"
            has_I2 += (t["kind"] >> 1) & 1
            has_I1 += (t["kind"] >> 2) & 1
            if t["cnt"] == 0:
                assert t["kind"] == 7, "a task without lags only accumulates I"
                continue
            own = lags[t["l0"]:t["l0"] + t["cnt"]]
            assert len(own) == t["cnt"] and own[0] == t["tau0"]
            if (t["kind"] & 1) == 0:
                assert own == list(range(t["tau0"], t["tau0"] + t["cnt"])), "a dense task is a run of consecutive lags"
            covered[t["l0"]:t["l0"] + t["cnt"]] += 1
            lo, hi = min(lo, own[0]), max(hi, own[-1])
        assert has_I2 == has_I1 == (g["flags"] & 1), "sum |F'|^2 and sum F' each ride on exactly one task"
        n_I2 += has_I2
        n_I1 += has_I1
        assert (g["tau_min"], g["tau_max"]) == (lo, hi)
    assert n_I2 == 1 and n_I1 == 1
    # persistent CTAs: contiguous shares, at least one per group, all resident slots handed out
    at = 0
    for g in groups:
        assert g["cta0"] == at and g["nctas"] >= 1
        at += g["nctas"]
    assert plan["tile_px"] in (32, 64) and plan["ctas_per_sm"] in (1, 2)
    assert plan["tile_px"] == 32 or plan["ctas_per_sm"] == 1, "64-pixel tiles: 17 warps, one CTA per SM"
    slots = max(plan["ctas_per_sm"] * N_SM, len(groups))
    ntiles = -(-n_px // plan["tile_px"])
    assert all(g["nctas"] <= max(1, ntiles) for g in groups), "no more persistent CTAs than pixel tiles"
    assert at == slots or (at < slots and all(g["nctas"] == ntiles for g in groups))
    if plan["ctas_per_sm"] == 2:
        assert plan["smem"] <= SMEM_SM // 2 - 1024
    assert len(seen_tasks) == len(tasks)
    assert np.all(covered == 1), "every lag is accumulated by exactly one task"
    assert 2 <= plan["stages"] <= 8
    assert 0 < plan["smem"] <= SMEM_OPTIN


@pytest.mark.parametrize("ci", [0, 1, 2, 3, 4])
def test_plan_of_baseline_configs(ci):
    cfg = synth.config(ci)
    plan = plan_of(cfg.lags, cfg.H * (cfg.W // 2 + 1))
    check_plan(cfg.lags, plan, cfg.H * (cfg.W // 2 + 1))
    if ci in (1, 2):  # 100 consecutive lags: 8 register-window tasks in one single-stream group, 64-pixel tiles
        assert len(plan["groups"]) == 1 and len(plan["tasks"]) == 8
        assert plan["groups"][0]["flags"] == 3 and plan["tile_px"] == 64
    if ci == 3:       # 40 log-spaced lags <= 500: one pass over the tile (one group, the whole window in shared memory)
        assert len(plan["groups"]) == 1 and plan["groups"][0]["flags"] == 3 and plan["tile_px"] == 32
        assert plan["slots"] == 16 and len(plan["tasks"]) > 8
    if ci == 4:       # lags 1..1000: ten groups of ~104 lags, only the first streams the batch as the head of its window
        assert len(plan["groups"]) == 10
        assert [g["flags"] & 2 for g in plan["groups"]] == [2] + [0] * 9


@pytest.mark.parametrize("seed", range(12))
def test_plan_of_random_lag_lists(seed):
    rng = np.random.default_rng(seed)
    n = int(rng.integers(1, 120))
    top = int(rng.choice([n, 2 * n, 10 * n, 2000]))
    lags = np.sort(rng.choice(np.arange(1, max(top, n) + 1), size=n, replace=False))
    check_plan(lags, plan_of(lags))
    check_plan(lags, plan_of(lags, 32 * 17), 32 * 17)   # the smallest frame: 32-pixel tiles only


def test_plan_edge_cases():
    for lags in ([1], [7], [1, 2], list(range(1, 14)), list(range(1, 15)), [1, 1000], list(range(5, 12)) + [400, 401]):
        check_plan(lags, plan_of(lags))
    with pytest.raises(binding.NFSError):
        plan_of([3, 2])
    with pytest.raises(binding.NFSError):
        plan_of([0, 1])
