"""Pins of the NEXT-3(b) variant oracle (oracle/tangram_oracle_depth.cpp, orc_variant_*: transfers count toward
the bottleneck): literal enumeration on tiny instances (alone and
combined with the depth-aware memory of NEXT-1), reduction to the core oracle when the flag is off or no transfer can
bind, monotonicity, an independent re-scorer, and a hand-worked case."""
import numpy as np
import pytest

import oracle
import tg_inputs as gen

INVALID = 0x7FFFFFFF
STYLES = ["mixed", "ties", "tightmem", "asym", "sparse"]


def rescore_xbound(inst, stages):
    """(sum, T, iter, mask) straight from the RAW tables: T is the largest stage time or boundary transfer;
    with a footprint, stage i of n must fit mem + (n - i) * actmem."""
    L, m, n = inst.L, inst.m, len(stages)
    total, T, mask = 0, 0, 0
    for i, (a, k, p) in enumerate(stages):
        b = stages[i + 1][0] if i + 1 < n else L
        s = gen.slice_index(L, a, b)
        t = int(inst.time_us[s, k, p])
        assert t != INVALID
        act = 0 if inst.actmem_mb is None else int(inst.actmem_mb[s, k, p])
        assert int(inst.mem_mb[s, k, p]) + (n - i) * act <= int(inst.island_cap_mb[k])
        assert not (mask >> k) & 1
        mask |= 1 << k
        total += t
        T = max(T, t)
        if i + 1 < n:
            x = -((-inst.act_mb * 1000) // int(inst.bw_gbps[k, stages[i + 1][1]]))
            total += x
            if inst.transfer_bound:
                T = max(T, x)
    return total, T, total + (m - 1) * T, mask


@pytest.mark.parametrize("style", STYLES)
def test_xbound_dp_equals_bruteforce(style):
    n_feasible = n_matters = 0
    for seed in range(700):
        base = gen.random_small(seed + 80_000, Lmax=6, Kmax=4, Pmax=3, style=style)
        inst = gen.with_transfer_bound(base)
        bf = oracle.bruteforce_variant(inst)
        dp = oracle.solve_variant(inst)
        assert bf.feasible == dp.feasible, inst.name
        core = oracle.solve(base)
        assert core.feasible == dp.feasible            # feasibility does not depend on the bound (T can grow)
        if not dp.feasible:
            continue
        n_feasible += 1
        assert bf.plan_key() == dp.plan_key(), inst.name
        assert rescore_xbound(inst, dp.stages) == (dp.sum_us, dp.bottleneck_us, dp.iter_time_us, dp.island_mask)
        assert core.iter_time_us <= dp.iter_time_us    # a larger bottleneck can only hurt
        n_matters += core.plan_key() != dp.plan_key()
    assert n_feasible > 150 and n_matters >= 3, (n_feasible, n_matters)


@pytest.mark.parametrize("style", STYLES)
def test_xbound_with_depth_equals_bruteforce(style):
    n_feasible = 0
    for seed in range(300):
        base = gen.random_small(seed + 81_000, Lmax=6, Kmax=4, Pmax=3, style=style)
        inst = gen.with_transfer_bound(gen.with_actmem(base, seed))
        bf = oracle.bruteforce_variant(inst)
        dp = oracle.solve_variant(inst)
        assert bf.feasible == dp.feasible, inst.name
        if not dp.feasible:
            continue
        n_feasible += 1
        assert bf.plan_key() == dp.plan_key(), inst.name
        assert rescore_xbound(inst, dp.stages) == (dp.sum_us, dp.bottleneck_us, dp.iter_time_us, dp.island_mask)
        assert oracle.solve_depth(inst).iter_time_us <= dp.iter_time_us
    assert n_feasible > 50


@pytest.mark.parametrize("seed", range(60))
def test_flag_off_and_free_transfers_are_the_core_problem(seed):
    base = gen.random_small(seed + 82_000, Lmax=7, Kmax=4, Pmax=3, style=STYLES[seed % 5])
    assert oracle.solve_variant(base).plan_key() == oracle.solve(base).plan_key()          # neither variant switched on
    free = base.copy()
    free.act_mb = 0                                                                         # x = 0 everywhere: never binds
    assert oracle.solve_variant(gen.with_transfer_bound(free)).plan_key() == oracle.solve(free).plan_key()


@pytest.mark.parametrize("seed", range(40))
def test_slower_links_never_improve(seed):
    base = gen.random_small(seed + 83_000, Lmax=6, Kmax=4, Pmax=3, style=STYLES[seed % 5])
    prev = None
    for act in (0, 16, 64, 256, 1024):
        inst = gen.with_transfer_bound(base)
        inst.act_mb = act
        v = oracle.solve_variant(inst).iter_time_us
        assert prev is None or v >= prev
        prev = v


def _two_layer(act_mb):
    """L=2, K=2, P=1, m=10, no memory limits.  One layer costs 10 us on either island, both layers 30 us
    (a single stage is slower than the two halves); bandwidth 1000 GB/s both ways, so x = act_mb us."""
    t = np.array([[[10], [10]], [[30], [30]], [[10], [10]]], np.int32)      # slices [0,1), [0,2), [1,2)
    z = np.zeros_like(t)
    return gen.Instance("hand_xb", 2, 2, 1, 10, t, z, np.array([1, 1], np.int32), np.array([100, 100], np.int32),
                        np.array([[1000, 1000], [1000, 1000]], np.int32), act_mb)


def test_hand_worked_transfer_bound():
    """x = 25: two stages cost 10 + 25 + 10 = 45.  Core: T = 10 -> 45 + 9*10 = 135.  Bounded: T = max(10, 25) = 25 ->
    45 + 9*25 = 270, still better than the single stage 30 + 9*30 = 300.
    x = 35: two stages cost 55.  Core: 55 + 90 = 145.  Bounded: T = 35 -> 55 + 315 = 370 > 300: the single stage wins,
    on island 0 (lowest mask among the two equal single-stage plans)."""
    a = _two_layer(25)
    core, xb = oracle.solve(a), oracle.solve_variant(gen.with_transfer_bound(a))
    assert (core.iter_time_us, core.bottleneck_us, core.sum_us) == (135, 10, 45)
    assert (xb.iter_time_us, xb.bottleneck_us, xb.sum_us, xb.stages) == (270, 25, 45, [(0, 0, 0), (1, 1, 0)])
    b = _two_layer(35)
    core, xb = oracle.solve(b), oracle.solve_variant(gen.with_transfer_bound(b))
    assert (core.iter_time_us, core.bottleneck_us, core.sum_us) == (145, 10, 55)
    assert (xb.iter_time_us, xb.bottleneck_us, xb.sum_us, xb.island_mask, xb.stages) == (300, 30, 30, 1, [(0, 0, 0)])


@pytest.mark.parametrize("style", ["mixed", "ties", "tightmem", "asym", "sparse"])
def test_threaded_variant_solve_equals_sequential_and_bruteforce(style):
    """orc_variant_solve_mt (bisection + blocks of threads, used for the K = 16 goldens) against the plain ascending
    sweep and against the literal enumeration: value, plan and candidate count, with and without either variant."""
    for s in range(60):
        inst = gen.random_small(4000 + s, Lmax=7, Kmax=5, Pmax=3, style=style)
        if s % 2:
            inst = gen.with_actmem(inst, s, 0, 40)
        if s % 3 == 0:
            inst = gen.with_transfer_bound(inst)
        seq = oracle.solve_variant(inst)
        for nt in (1, 3):
            mt = oracle.solve_variant(inst, nt)
            assert mt.plan_key() == seq.plan_key() and mt.n_candidates == seq.n_candidates, inst.name
        if inst.actmem_mb is None:
            inst.actmem_mb = np.zeros_like(inst.time_us)
        bf = oracle.bruteforce_variant(inst)
        assert bf.plan_key() == seq.plan_key(), inst.name
