"""Pins of the per-boundary activation sizes (oracle/tangram_oracle_depth.cpp: orc_variant_solve_b / _bruteforce_b; SURVEY.md
§8(f) NEXT-3(b) second half, PAPER.md:240 (1) "only transferring stage inputs and outputs", :350): literal enumeration
alone and combined with the transfer bound and the footprint; a constant size is the scalar act_mb; a hand-worked case
where the cut moves to the boundary with the small activation; monotonicity; re-scoring from the raw tables."""
import numpy as np
import pytest

import oracle
import tg_inputs as gen

INVALID = 0x7FFFFFFF
STYLES = ["mixed", "ties", "tightmem", "asym", "sparse"]


def rescore_b(inst, stages):
    L, m, n = inst.L, inst.m, len(stages)
    total, T, mask = 0, 0, 0
    for i, (a, k, p) in enumerate(stages):
        b = stages[i + 1][0] if i + 1 < n else L
        s = gen.slice_index(L, a, b)
        t = int(inst.time_us[s, k, p])
        act = 0 if inst.actmem_mb is None else int(inst.actmem_mb[s, k, p])
        assert t != INVALID and int(inst.mem_mb[s, k, p]) + (n - i) * act <= int(inst.island_cap_mb[k])
        assert not (mask >> k) & 1
        mask |= 1 << k
        total += t
        T = max(T, t)
        if i + 1 < n:
            amb = inst.act_mb if inst.act_mb_b is None else int(inst.act_mb_b[b])
            x = -((-amb * 1000) // int(inst.bw_gbps[k, stages[i + 1][1]]))
            total += x
            if inst.transfer_bound:
                T = max(T, x)
    return total, T, total + (m - 1) * T, mask


@pytest.mark.parametrize("style", STYLES)
def test_dp_equals_literal_enumeration(style):
    for s in range(100):
        inst = gen.with_boundary_act(gen.random_small(9000 + s, Lmax=7, Kmax=4, Pmax=3, style=style), s,
                                     sizes=[(4, 64, 900), (16, 64, 256), (0, 64)][s % 3])
        if s % 2:
            inst = gen.with_transfer_bound(inst)
        if s % 3 == 0:
            inst = gen.with_actmem(inst, s, 0, 40)
        dp = oracle.solve_variant_b(inst)
        if inst.actmem_mb is None:
            inst.actmem_mb = np.zeros_like(inst.time_us)
        bf = oracle.bruteforce_variant_b(inst)
        assert dp.plan_key() == bf.plan_key(), inst.name
        if dp.feasible:
            assert rescore_b(inst, dp.stages) == (dp.sum_us, dp.bottleneck_us, dp.iter_time_us, dp.island_mask)


def test_constant_size_is_the_scalar_definition():
    for s in range(60):
        base = gen.random_small(9300 + s, Lmax=8, Kmax=5, Pmax=3, style=STYLES[s % 5])
        if s % 2:
            base = gen.with_transfer_bound(base)
        inst = base.copy()
        inst.act_mb_b = np.full(base.L + 1, base.act_mb, dtype=np.int32)
        a, b = oracle.solve_variant_b(inst), oracle.solve_variant(base)
        assert a.plan_key() == b.plan_key()
        if base.L >= 2:                        # (a one-layer model has no boundary: the per-boundary list holds no transfer times)
            assert a.n_candidates == b.n_candidates
        assert oracle.solve_variant_b(base).plan_key() == b.plan_key()           # act_mb_b = None


def test_hand_worked_cut_moves_to_the_cheap_boundary():
    """Three layers, two islands, one plan, m = 1 (iter = sum).  On either island a slice of 1 / 2 / 3 layers takes
    10 / 20 / 9000 us, so the model is split in two.  bw = 1 GB/s: x = act * 1000 us.  Boundary 1 carries 5 MB (5000 us),
    boundary 2 carries 1 MB (1000 us).
    Cut at 1: 10 + 5000 + 20 = 5030.   Cut at 2: 20 + 1000 + 10 = 1030  <- optimum (one stage: 9000); first stage on island 0
    (lowest k_0).  With the sizes swapped the cut moves to boundary 1: 10 + 1000 + 20 = 1030."""
    L, K = 3, 2
    t = np.zeros((6, K, 1), dtype=np.int32)
    for a in range(L):
        for b in range(a + 1, L + 1):
            t[gen.slice_index(L, a, b), :, 0] = {1: 10, 2: 20, 3: 9000}[b - a]
    inst = gen.Instance("handb", L, K, 1, 1, t, np.zeros_like(t), np.ones(K, np.int32), np.full(K, 10, np.int32),
                        np.ones((K, K), np.int32), 3)
    inst.act_mb_b = np.array([0, 5, 1, 0], dtype=np.int32)
    r = oracle.solve_variant_b(inst)
    assert (r.iter_time_us, r.stages) == (1030, [(0, 0, 0), (2, 1, 0)])
    inst.act_mb_b = np.array([0, 1, 5, 0], dtype=np.int32)
    r = oracle.solve_variant_b(inst)
    assert (r.iter_time_us, r.stages) == (1030, [(0, 0, 0), (1, 1, 0)])
    inst.act_mb_b = None                                                        # scalar 3 MB everywhere: 10 + 3000 + 20, cut at 1 (lowest b)
    r = oracle.solve_variant_b(inst)
    assert (r.iter_time_us, r.stages) == (3030, [(0, 0, 0), (1, 1, 0)])


def test_smaller_activations_never_worsen():
    for s in range(60):
        base = gen.random_small(9500 + s, Lmax=7, Kmax=4, Pmax=3, style=STYLES[s % 5])
        big = gen.with_boundary_act(base, s, sizes=(64, 256, 900))
        small = big.copy()
        small.act_mb_b = (big.act_mb_b // 2).astype(np.int32)
        a, b = oracle.solve_variant_b(small), oracle.solve_variant_b(big)
        assert a.feasible == b.feasible or a.feasible
        if b.feasible:
            assert a.iter_time_us <= b.iter_time_us
