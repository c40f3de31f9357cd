"""Pins for oracle.prune (tg_prune rules R1-R4; PAPER.md:234-236 policies, :43/:360
incompatible plans; pin P-prune PAPER.md:360, :364 "pruning leaves the composed plan the same") and for
oracle.reduce (steps 1-3) against a hand-computed fixture."""
import json
import os

import numpy as np
import pytest

import oracle
import tg_inputs as gen

INVALID = 0x7FFFFFFF
STYLES = ["mixed", "ties", "tightmem", "asym", "sparse"]
HERE = os.path.dirname(os.path.abspath(__file__))


def same_up_to_equal_time_plans(inst, r0, r1):
    """R2 may kill the lowest-p plan of a cell in favour of an equal-time, lower-memory plan with a
    higher index (reading R-prune-ties): everything but stage_plan is identical, and the
    chosen plans have the same time."""
    assert r0.feasible == r1.feasible
    if not r0.feasible:
        return
    assert r0.plan_key()[:4] == r1.plan_key()[:4]
    assert [(a, k) for a, k, _ in r0.stages] == [(a, k) for a, k, _ in r1.stages]
    L = inst.L
    for i, ((a, k, p0), (_, _, p1)) in enumerate(zip(r0.stages, r1.stages)):
        b = r0.stages[i + 1][0] if i + 1 < len(r0.stages) else L
        s = gen.slice_index(L, a, b)
        assert inst.time_us[s, k, p0] == inst.time_us[s, k, p1] and inst.mem_mb[s, k, p1] <= inst.mem_mb[s, k, p0]


def py_prune_exact(inst):
    """R1 + R2 straight from their definitions, O(P^2) per cell, independent of the oracle's loops."""
    t = inst.time_us.astype(np.int64).copy()
    mm = inst.mem_mb.astype(np.int64)
    NS, K, P = t.shape
    c1 = c2 = 0
    for s in range(NS):
        for k in range(K):
            for p in range(P):
                if t[s, k, p] != INVALID and mm[s, k, p] > inst.island_cap_mb[k]:
                    t[s, k, p] = INVALID; c1 += 1
            live = [p for p in range(P) if t[s, k, p] != INVALID]
            dead = []
            for p in live:
                for q in live:
                    if q == p:
                        continue
                    tq, tp, mq, mp = t[s, k, q], t[s, k, p], mm[s, k, q], mm[s, k, p]
                    if (tq < tp and mq <= mp) or (tq <= tp and mq < mp) or (tq == tp and mq == mp and q < p):
                        dead.append(p); break
            for p in dead:
                t[s, k, p] = INVALID; c2 += 1
    return t.astype(np.int32), c1, c2


@pytest.mark.parametrize("seed", range(60))
def test_exact_rules_match_definition_and_keep_the_result(seed):
    inst = gen.random_small(seed + 5000, Lmax=7, Kmax=4, Pmax=5, style=STYLES[seed % 5])
    pr, counts = oracle.prune(inst, 0)
    t, c1, c2 = py_prune_exact(inst)
    assert np.array_equal(pr.time_us.reshape(t.shape), t)
    assert counts.tolist() == [c1, c2, 0, 0]
    same_up_to_equal_time_plans(inst, oracle.solve(inst), oracle.solve(pr))          # P-prune
    pr2, counts2 = oracle.prune(pr, 0)                                             # idempotent
    assert counts2.tolist() == [0, 0, 0, 0] and np.array_equal(pr2.time_us, pr.time_us)
    # survivors form a strict Pareto front: sorted by time ascending, memory strictly descending
    tt = pr.time_us.reshape(t.shape)
    for s in range(t.shape[0]):
        for k in range(t.shape[1]):
            live = sorted((int(tt[s, k, p]), int(inst.mem_mb[s, k, p])) for p in range(t.shape[2]) if tt[s, k, p] != INVALID)
            assert all(a[0] < b[0] and a[1] > b[1] for a, b in zip(live, live[1:]))


@pytest.mark.parametrize("seed", range(40))
def test_bottleneck_cap_exact_above_T_star(seed):
    inst = gen.random_small(seed + 6000, Lmax=7, Kmax=4, Pmax=3, style=STYLES[seed % 5])
    r = oracle.solve(inst)
    if not r.feasible:
        return
    pr, counts = oracle.prune(inst, 2, r.bottleneck_us)                             # R4, cap = T*
    same_up_to_equal_time_plans(inst, r, oracle.solve(pr))
    live = pr.time_us[pr.time_us != INVALID]
    assert live.size == 0 or live.max() <= r.bottleneck_us
    pr0, _ = oracle.prune(inst, 2, 0)                                               # cap 0 kills all positive times
    assert (pr0.time_us[pr0.time_us != INVALID] == 0).all()


@pytest.mark.parametrize("seed", range(40))
def test_imbalance_monotone_and_never_improves(seed):
    inst = gen.random_small(seed + 7000, Lmax=8, Kmax=4, Pmax=2, style=STYLES[seed % 3])
    r = oracle.solve(inst)
    prev_kill = None
    for theta in (16384, 8000, 4000, 2000, 1500, 1000):
        pr, counts = oracle.prune(inst, 1, theta)
        killed = int(counts[2])
        assert prev_kill is None or killed >= prev_kill                             # monotone in theta
        prev_kill = killed
        q = oracle.solve(pr)
        if q.feasible:
            assert r.feasible and q.iter_time_us >= r.iter_time_us                  # lossy, never better
        dead_before = inst.time_us == INVALID
        assert (pr.time_us.reshape(inst.time_us.shape)[dead_before] == INVALID).all()   # never revives


def test_imbalance_hand_worked():
    """L=4, K=2, P=1.  Atom times: island0 10 us/layer, island1 30 us/layer -> tau = 40, 120;
    C_k = floor(2^32/tau) -> shares 3/4 and 1/4 (up to flooring).  theta = 2000 permille:
    island0 keeps len/L in [0.375, 1.5] -> len 2,3,4 ; island1 keeps [0.125, 0.5] -> len 1,2."""
    L, K = 4, 2
    a, b = gen.slice_bounds(L)
    ln = (b - a)
    t = np.stack([ln * 10, ln * 30], axis=1)[:, :, None].astype(np.int32)
    inst = gen.Instance("hand", L, K, 1, 4, t, np.zeros_like(t), np.ones(K, np.int32), np.full(K, 10, np.int32),
                        np.full((K, K), 100, np.int32), 0)
    pr, counts = oracle.prune(inst, 1, 2000)
    alive = pr.time_us.reshape(t.shape)[:, :, 0] != INVALID
    assert sorted(set(ln[alive[:, 0]].tolist())) == [2, 3, 4]
    assert sorted(set(ln[alive[:, 1]].tolist())) == [1, 2]
    assert counts.tolist() == [0, 0, 4 + 3, 0]      # island0 loses 4 len-1 slices; island1 2 len-3 + 1 len-4


def test_reduce_golden_fixture():
    """tests/golden/reduce_small.json: raw tables and the reduced c/argp/x/candidates worked by hand
    (citations inside the file)."""
    with open(os.path.join(HERE, "golden", "reduce_small.json")) as f:
        g = json.load(f)
    L, K, P = g["L"], g["K"], g["P"]
    inst = gen.Instance("golden", L, K, P, 2, np.array(g["time_us"], np.int32).reshape(-1, K, P),
                        np.array(g["mem_mb"], np.int32).reshape(-1, K, P), np.ones(K, np.int32),
                        np.array(g["cap_mb"], np.int32), np.array(g["bw_gbps"], np.int32), g["act_mb"])
    c, argp, x, cand = oracle.reduce(inst)
    assert c.tolist() == g["c"] and argp.tolist() == g["argp"] and x.tolist() == g["x"] and cand.tolist() == g["candidates"]
    r = oracle.solve(inst)
    assert [r.iter_time_us, r.bottleneck_us, r.island_mask, [list(s) for s in r.stages]] == g["result"]
