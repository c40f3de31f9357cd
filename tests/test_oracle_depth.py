"""Pins of the NEXT-1 oracle (oracle/tangram_oracle_depth.cpp: depth-aware activation memory under 1F1B,
PAPER.md:246-250, :258(i)): literal enumeration on tiny instances, reduction to the core oracle when the
activation footprint is zero, monotonicity, and an independent re-scorer of the returned plan."""
import numpy as np
import pytest

import oracle
import tg_inputs as gen

INVALID = 0x7FFFFFFF
STYLES = ["mixed", "ties", "tightmem", "asym", "sparse"]


def rescore_depth(inst, stages):
    """(sum, T, iter, mask) of a plan straight from the RAW tables under the depth rule: stage i of n is
    feasible iff mem + (n - i) * actmem <= cap."""
    L, m, n = inst.L, inst.m, len(stages)
    total, T, mask = 0, 0, 0
    for i, (a, k, p) in enumerate(stages):
        b = stages[i + 1][0] if i + 1 < n else L
        s = gen.slice_index(L, a, b)
        t = int(inst.time_us[s, k, p])
        assert t != INVALID
        assert int(inst.mem_mb[s, k, p]) + (n - i) * int(inst.actmem_mb[s, k, p]) <= int(inst.island_cap_mb[k])
        assert not (mask >> k) & 1
        mask |= 1 << k
        total += t
        T = max(T, t)
        if i + 1 < n:
            total += -((-inst.act_mb * 1000) // int(inst.bw_gbps[k, stages[i + 1][1]]))
    return total, T, total + (m - 1) * T, mask


@pytest.mark.parametrize("style", STYLES)
def test_depth_dp_equals_bruteforce(style):
    n_feasible = n_depth_matters = 0
    for seed in range(900):
        base = gen.random_small(seed + 60_000, Lmax=6, Kmax=4, Pmax=3, style=style)
        inst = gen.with_actmem(base, seed)
        bf = oracle.bruteforce_depth(inst)
        dp = oracle.solve_depth(inst)
        assert bf.feasible == dp.feasible, inst.name
        if not dp.feasible:
            continue
        n_feasible += 1
        assert bf.plan_key() == dp.plan_key(), inst.name
        assert rescore_depth(inst, dp.stages) == (dp.sum_us, dp.bottleneck_us, dp.iter_time_us, dp.island_mask)
        core = oracle.solve(base)
        assert core.feasible and core.iter_time_us <= dp.iter_time_us     # the footprint can only hurt
        n_depth_matters += core.plan_key() != dp.plan_key()
    assert n_feasible > 150 and n_depth_matters > 20


@pytest.mark.parametrize("seed", range(60))
def test_zero_footprint_is_the_core_problem(seed):
    base = gen.random_small(seed + 61_000, Lmax=7, Kmax=4, Pmax=3, style=STYLES[seed % 5])
    inst = gen.with_actmem(base, seed, 0, 0)
    assert oracle.solve_depth(inst).plan_key() == oracle.solve(base).plan_key()


@pytest.mark.parametrize("seed", range(40))
def test_larger_footprint_never_improves(seed):
    base = gen.random_small(seed + 62_000, Lmax=6, Kmax=4, Pmax=3, style=STYLES[seed % 5])
    prev = None
    for hi in (0, 20, 60, 200):
        r = oracle.solve_depth(gen.with_actmem(base, seed, hi // 2, hi))
        v = r.iter_time_us                      # INT64_MAX when infeasible
        assert prev is None or v >= prev
        prev = v


def test_hand_worked_depth():
    """L=2, K=2, P=2, m=1, no transfers.  Island 0: cap 100.  Its plan 0 is fast (10 us, mem 50, act 30):
    feasible only at depth 1 (50+30 <= 100 < 50+60); plan 1 is slow (40 us, mem 10, act 10).  Island 1: every
    slice 25 us, no memory.  Plans: [0,1) on 0 then [1,2) on 1: island 0 is FIRST of two stages -> depth 2 ->
    must use the slow plan: 40+25 = 65.  [0,1) on 1 then [1,2) on 0: island 0 is last -> depth 1 -> 25+10 = 35.
    Single stage [0,2) on island 0 at depth 1 (fast plan 10 us per layer -> 20): best = 20."""
    L, K, P = 2, 2, 2
    t = np.array([[[10, 40], [25, 25]], [[20, 80], [50, 50]], [[10, 40], [25, 25]]], np.int32)
    mm = np.array([[[50, 10], [0, 0]]] * 3, np.int32)
    am = np.array([[[30, 10], [0, 0]]] * 3, np.int32)
    inst = gen.Instance("hand", L, K, P, 1, t, mm, np.ones(K, np.int32), np.array([100, 100], np.int32),
                        np.full((K, K), 100, np.int32), 0, {}, am)
    r = oracle.solve_depth(inst)
    assert (r.iter_time_us, r.stages) == (20, [(0, 0, 0)])
    inst.time_us[1, 0, :] = INVALID             # forbid the whole model on island 0
    r = oracle.solve_depth(inst)
    assert (r.iter_time_us, r.stages) == (35, [(0, 1, 0), (1, 0, 0)])
    inst.time_us[2, 0, :] = INVALID             # ... and island 0 as the last stage
    r = oracle.solve_depth(inst)
    assert (r.iter_time_us, r.stages) == (50, [(0, 1, 0)])          # whole model on island 1 beats 40 + 25
    inst.time_us[1, 1, :] = INVALID
    r = oracle.solve_depth(inst)
    assert (r.iter_time_us, r.stages) == (65, [(0, 0, 1), (1, 1, 0)])    # island 0 first: depth 2: slow plan
