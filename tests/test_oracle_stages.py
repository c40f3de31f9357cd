"""Pins of the NEXT-2 oracle (oracle/tangram_oracle_stages.cpp: multi-stage partial plans, SURVEY.md §8(f) NEXT-2;
PAPER.md:163, :248, :250 (1) "ranks the slowest stages in all model-slice/island plans"): literal enumeration over cut
sets, island orders AND plan choices on tiny instances; slow == time reduces to the core oracle; a hand-worked case;
monotonicity in the slowest-stage values; the reported T* is the slowest stage of the returned plan; an independent
re-scorer from the raw tables."""
import numpy as np
import pytest

import oracle
import tg_inputs as gen

INVALID = 0x7FFFFFFF
STYLES = ["mixed", "ties", "tightmem", "asym", "sparse"]


def rescore_stages(inst, stages):
    """(sum, T, iter, mask, total q) of a plan straight from the RAW tables: sum of the partial plans' times and the
    transfers, T = the slowest internal stage of any partial plan."""
    L, m, n = inst.L, inst.m, len(stages)
    total, T, mask, tq = 0, 0, 0, 0
    for i, (a, k, p) in enumerate(stages):
        b = stages[i + 1][0] if i + 1 < n else L
        s = gen.slice_index(L, a, b)
        t = int(inst.time_us[s, k, p])
        assert t != INVALID and int(inst.mem_mb[s, k, p]) <= int(inst.island_cap_mb[k])
        assert not (mask >> k) & 1
        mask |= 1 << k
        total += t
        T = max(T, int(inst.slow_us[s, k, p]))
        tq += 1 if inst.q_stages is None else int(inst.q_stages[s, k, p])
        if i + 1 < n:
            total += -((-inst.act_mb * 1000) // int(inst.bw_gbps[k, stages[i + 1][1]]))
    return total, T, total + (m - 1) * T, mask, tq


@pytest.mark.parametrize("style", STYLES)
def test_dp_equals_literal_enumeration(style):
    for s in range(120):
        base = gen.random_small(6000 + s, Lmax=6, Kmax=4, Pmax=3, style=style)
        inst = gen.with_stages(base, s, qmax=1 + s % 4)
        dp, tq = oracle.solve_stages(inst)
        bf, tq2, n = oracle.bruteforce_stages(inst)
        assert dp.plan_key() == bf.plan_key() and tq == tq2, inst.name
        if dp.feasible:
            sm, T, it, mask, q = rescore_stages(inst, dp.stages)
            assert (sm, T, it, mask, q) == (dp.sum_us, dp.bottleneck_us, dp.iter_time_us, dp.island_mask, tq)


@pytest.mark.parametrize("style", STYLES)
def test_single_stage_plans_reduce_to_the_core_oracle(style):
    """slow == time, q == 1: the definition of the core path, bit for bit (value and plan)."""
    for s in range(60):
        base = gen.random_small(6500 + s, Lmax=8, Kmax=5, Pmax=3, style=style)
        inst = base.copy()
        inst.slow_us = np.where(base.time_us == INVALID, 0, base.time_us).astype(np.int32)
        st, tq = oracle.solve_stages(inst)
        core = oracle.solve(base)
        assert st.plan_key() == core.plan_key()
        assert tq == core.n_stages


def test_hand_worked_slowest_stage_decides():
    """One layer, one island, two plans.  Plan 0: one stage of 100 us.  Plan 1: three internal stages 50 + 40 + 40 = 130 us,
    slowest 50.  m = 1: iter = sum, plan 0 wins (100 < 130).  m = 4: plan 0 costs 100 + 3*100 = 400, plan 1 costs
    130 + 3*50 = 280 -> plan 1, T* = 50, 3 pipeline stages.  Break-even m: 100 m = 130 + 50 (m-1) -> m = 1.6."""
    t = np.array([[[100, 130]]], dtype=np.int32)
    inst = gen.Instance("hand", 1, 1, 2, 1, t, np.zeros_like(t), np.array([1], np.int32), np.array([10], np.int32),
                        np.array([[1]], np.int32), 64)
    inst.slow_us = np.array([[[100, 50]]], dtype=np.int32)
    inst.q_stages = np.array([[[1, 3]]], dtype=np.int32)
    r, tq = oracle.solve_stages(inst)
    assert (r.iter_time_us, r.bottleneck_us, r.stages, tq) == (100, 100, [(0, 0, 0)], 1)
    inst.m = 2
    r, tq = oracle.solve_stages(inst)
    assert (r.iter_time_us, r.bottleneck_us, r.stages, tq) == (180, 50, [(0, 0, 1)], 3)
    inst.m = 4
    r, tq = oracle.solve_stages(inst)
    assert (r.iter_time_us, r.sum_us, r.bottleneck_us, r.stages, tq) == (280, 130, 50, [(0, 0, 1)], 3)


def test_hand_worked_two_layers_two_islands():
    """Two layers, two islands, one plan each, free transfers (act_mb = 0), m = 3.
    Whole model on island 0: time 90, slowest 30 (three internal stages)          -> 90 + 2*30 = 150
    Whole model on island 1: time 80, slowest 80                                   -> 80 + 2*80 = 240
    Layer 0 on island 0 (40, slowest 40), layer 1 on island 1 (45, slowest 45)     -> 85 + 2*45 = 175
    Layer 0 on island 1 (50, slowest 25), layer 1 on island 0 (35, slowest 35)     -> 85 + 2*35 = 155
    Optimum: the whole model on island 0, T* = 30."""
    L, K = 2, 2
    t = np.zeros((3, K, 1), dtype=np.int32)
    sl = np.zeros_like(t)
    q = np.ones_like(t)
    s01, s02, s12 = gen.slice_index(L, 0, 1), gen.slice_index(L, 0, 2), gen.slice_index(L, 1, 2)
    t[s02, 0, 0], sl[s02, 0, 0], q[s02, 0, 0] = 90, 30, 3
    t[s02, 1, 0], sl[s02, 1, 0] = 80, 80
    t[s01, 0, 0], sl[s01, 0, 0] = 40, 40
    t[s12, 1, 0], sl[s12, 1, 0] = 45, 45
    t[s01, 1, 0], sl[s01, 1, 0], q[s01, 1, 0] = 50, 25, 2
    t[s12, 0, 0], sl[s12, 0, 0] = 35, 35
    inst = gen.Instance("hand2", L, K, 1, 3, t, np.zeros_like(t), np.ones(K, np.int32), np.full(K, 10, np.int32),
                        np.full((K, K), 100, np.int32), 0)
    inst.slow_us, inst.q_stages = sl, q
    r, tq = oracle.solve_stages(inst)
    assert (r.iter_time_us, r.sum_us, r.bottleneck_us, r.island_mask, r.stages, tq) == (150, 90, 30, 1, [(0, 0, 0)], 3)
    sl[s02, 0, 0] = 40                       # a slower internal stage: 90 + 2*40 = 170 > 155 -> the split 1 -> 0 wins
    r, tq = oracle.solve_stages(inst)
    assert (r.iter_time_us, r.bottleneck_us, r.island_mask, r.stages, tq) == (155, 35, 3, [(0, 1, 0), (1, 0, 0)], 3)


def test_lower_slowest_stages_never_worsen():
    for s in range(80):
        base = gen.random_small(7000 + s, Lmax=7, Kmax=4, Pmax=3, style=STYLES[s % 5])
        hi = gen.with_stages(base, s, qmax=1)                      # slow == time
        lo = gen.with_stages(base, s, qmax=4)                      # slow <= time entry by entry
        assert (lo.slow_us <= hi.slow_us).all()
        a, _ = oracle.solve_stages(lo)
        b, _ = oracle.solve_stages(hi)
        assert a.feasible == b.feasible
        if a.feasible:
            assert a.iter_time_us <= b.iter_time_us


def test_bottleneck_is_a_slowest_stage_of_the_plan_and_m1_is_the_shortest_path():
    for s in range(60):
        inst = gen.with_stages(gen.random_small(7200 + s, Lmax=7, Kmax=4, Pmax=3, style=STYLES[s % 5]), s)
        r, _ = oracle.solve_stages(inst)
        if not r.feasible:
            continue
        _, T, _, _, _ = rescore_stages(inst, r.stages)
        assert T == r.bottleneck_us
        one = inst.copy()
        one.m = 1                                                   # iter = sum: the slowest stages do not matter
        r1, _ = oracle.solve_stages(one)
        core = inst.copy()
        core.slow_us = None
        assert r1.iter_time_us == oracle.solve(gen.Instance(**{**core.__dict__, "m": 1})).iter_time_us
