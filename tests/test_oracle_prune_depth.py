"""Pins for oracle.prune_depth (tg_prune on instances with a footprint table; SURVEY.md §8(f) NEXT-1 "R2 dominance
becomes 3-way", reading N1-prune; PAPER.md:43/:360 incompatible plans, :246 deeper stages hold more
activations, :364 "pruning leaves the composed plan the same")."""
import numpy as np
import pytest

import oracle
import tg_inputs as gen

INVALID = 0x7FFFFFFF
STYLES = ["mixed", "ties", "tightmem", "asym", "sparse"]


def py_prune3(inst):
    """R1 + 3-way R2 restated on sets of (time, mem, actmem, index) tuples, no shared loops with the oracle."""
    t = inst.time_us.astype(np.int64).copy()
    NS, K, P = t.shape
    c1 = c2 = 0
    for s in range(NS):
        for k in range(K):
            cell = []
            for p in range(P):
                if t[s, k, p] == INVALID:
                    continue
                if int(inst.mem_mb[s, k, p]) + int(inst.actmem_mb[s, k, p]) > int(inst.island_cap_mb[k]):
                    t[s, k, p] = INVALID; c1 += 1
                else:
                    cell.append((int(t[s, k, p]), int(inst.mem_mb[s, k, p]), int(inst.actmem_mb[s, k, p]), p))
            for v in cell:
                better = [w for w in cell if w is not v and all(x <= y for x, y in zip(w[:3], v[:3]))
                          and (w[:3] != v[:3] or w[3] < v[3])]
                if better:
                    t[s, k, v[3]] = INVALID; c2 += 1
    return t.astype(np.int32), c1, c2


def same_up_to_equal_plans(inst, r0, r1):
    """R2 may replace the lowest-p plan of a cell by an equal-time plan with a higher index that needs no more
    memory on either axis; everything but stage_plan is identical."""
    assert r0.feasible == r1.feasible
    if not r0.feasible:
        return
    assert r0.plan_key()[:4] == r1.plan_key()[:4]
    assert [(a, k) for a, k, _ in r0.stages] == [(a, k) for a, k, _ in r1.stages]
    for i, ((a, k, p0), (_, _, p1)) in enumerate(zip(r0.stages, r1.stages)):
        b = r0.stages[i + 1][0] if i + 1 < len(r0.stages) else inst.L
        s = gen.slice_index(inst.L, a, b)
        assert inst.time_us[s, k, p0] == inst.time_us[s, k, p1]
        assert inst.mem_mb[s, k, p1] <= inst.mem_mb[s, k, p0] and inst.actmem_mb[s, k, p1] <= inst.actmem_mb[s, k, p0]


@pytest.mark.parametrize("seed", range(100))
def test_exact_rules_match_definition_and_keep_the_enumerated_optimum(seed):
    base = gen.random_small(seed + 90_000, Lmax=6, Kmax=4, Pmax=5, style=STYLES[seed % 5])
    inst = gen.with_actmem(base, seed)
    pr, counts = oracle.prune_depth(inst, 0)
    t, c1, c2 = py_prune3(inst)
    assert np.array_equal(pr.time_us.reshape(t.shape), t)
    assert counts.tolist() == [c1, c2, 0, 0]
    # the literal enumeration of every plan (not the DP) sees the same optimum on the pruned tables
    same_up_to_equal_plans(inst, oracle.bruteforce_depth(inst), oracle.bruteforce_depth(pr))
    same_up_to_equal_plans(inst, oracle.solve_depth(inst), oracle.solve_depth(pr))
    pr2, counts2 = oracle.prune_depth(pr, 0)
    assert counts2.tolist() == [0, 0, 0, 0] and np.array_equal(pr2.time_us, pr.time_us)
    # survivors of a cell form an antichain on (time, mem, actmem) with no duplicates
    tt = pr.time_us.reshape(t.shape)
    for s in range(t.shape[0]):
        for k in range(t.shape[1]):
            live = [(int(tt[s, k, p]), int(inst.mem_mb[s, k, p]), int(inst.actmem_mb[s, k, p]))
                    for p in range(t.shape[2]) if tt[s, k, p] != INVALID]
            for i, v in enumerate(live):
                for j, w in enumerate(live):
                    assert i == j or not all(x <= y for x, y in zip(w, v))


def test_the_third_axis_kills_and_spares():
    n_spared = n_killed = 0
    for seed in range(60):
        base = gen.random_small(seed + 91_000, Lmax=6, Kmax=4, Pmax=5, style=STYLES[seed % 5])
        inst = gen.with_actmem(base, seed)
        d3 = oracle.prune_depth(inst, 0)[0].time_us.reshape(inst.time_us.shape) == INVALID
        flat = inst.copy(); flat.actmem_mb = np.zeros_like(inst.actmem_mb)
        d2 = oracle.prune_depth(flat, 0)[0].time_us.reshape(inst.time_us.shape) == INVALID
        n_spared += int((d2 & ~d3).sum())        # 2-way dominated, saved by a smaller footprint
        n_killed += int((d3 & ~d2).sum())        # alive on two axes, dead because mem + actmem > cap
    assert n_spared > 20 and n_killed > 20


@pytest.mark.parametrize("seed", range(40))
@pytest.mark.parametrize("mode,thr", [(0, 0), (1, 2000), (2, 900)])
def test_zero_footprint_is_the_core_prune(seed, mode, thr):
    base = gen.random_small(seed + 92_000, Lmax=7, Kmax=4, Pmax=5, style=STYLES[seed % 5])
    inst = gen.with_actmem(base, seed, 0, 0)
    a, ca = oracle.prune_depth(inst, mode, thr)
    b, cb = oracle.prune(base, mode, thr)
    assert ca.tolist() == cb.tolist() and np.array_equal(a.time_us, b.time_us)


def test_hand_worked_cell():
    """L=1, K=1, cap 100.  Plans (time, mem, actmem):
       p0 (10, 50, 30)  kept;          p1 (10, 50, 30)  duplicate of p0, higher index -> R2;
       p2 ( 9, 60, 10)  kept (faster); p3 (12, 50, 30)  slower than p0, nothing smaller -> R2;
       p4 (11, 40, 40)  kept: less mem than p0 but a larger footprint (2-way on (time, mem+actmem) would differ);
       p5 ( 8, 90, 11)  R1: 90 + 11 > 100;     p6 (20, 10, 5) kept (smallest on both memory axes);
       p7 invalid."""
    t = np.array([10, 10, 9, 12, 11, 8, 20, INVALID], np.int32).reshape(1, 1, 8)
    mm = np.array([50, 50, 60, 50, 40, 90, 10, 0], np.int32).reshape(1, 1, 8)
    am = np.array([30, 30, 10, 30, 40, 11, 5, 0], np.int32).reshape(1, 1, 8)
    inst = gen.Instance("hand3", 1, 1, 8, 4, t, mm, np.ones(1, np.int32), np.full(1, 100, np.int32),
                        np.full((1, 1), 100, np.int32), 0)
    inst.actmem_mb = am
    pr, counts = oracle.prune_depth(inst, 0)
    assert (pr.time_us.reshape(-1) != INVALID).tolist() == [True, False, True, False, True, False, True, False]
    assert counts.tolist() == [1, 2, 0, 0]


@pytest.mark.parametrize("seed", range(30))
def test_lossy_modes_with_footprint(seed):
    base = gen.random_small(seed + 93_000, Lmax=7, Kmax=4, Pmax=3, style=STYLES[seed % 5])
    inst = gen.with_actmem(base, seed)
    r = oracle.solve_depth(inst)
    if r.feasible:                                                  # R4 at T* keeps the optimum
        pr, _ = oracle.prune_depth(inst, 2, r.bottleneck_us)
        same_up_to_equal_plans(inst, r, oracle.solve_depth(pr))
        live = pr.time_us[pr.time_us != INVALID]
        assert live.size == 0 or live.max() <= r.bottleneck_us
    prev = None
    for theta in (16384, 4000, 2000, 1000):                         # R3 monotone in theta, never better, never revives
        pr, counts = oracle.prune_depth(inst, 1, theta)
        assert prev is None or int(counts[2]) >= prev
        prev = int(counts[2])
        q = oracle.solve_depth(pr)
        if q.feasible:
            assert r.feasible and q.iter_time_us >= r.iter_time_us
        assert (pr.time_us.reshape(inst.time_us.shape)[inst.time_us == INVALID] == INVALID).all()
