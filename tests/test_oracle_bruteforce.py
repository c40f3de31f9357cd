"""Pins for oracle.solve: literal enumeration of the plain definition on
thousands of tiny random instances, value AND plan; windowed sweep == full sweep (A7)."""
import pytest

import oracle
import tg_inputs as gen
from conftest import rescore

STYLES = ["mixed", "ties", "tightmem", "asym", "sparse"]


def _same(a, b):
    assert a.feasible == b.feasible
    if not a.feasible:
        return
    assert (a.iter_time_us, a.sum_us, a.bottleneck_us, a.island_mask) == \
           (b.iter_time_us, b.sum_us, b.bottleneck_us, b.island_mask)
    assert a.stages == b.stages


@pytest.mark.parametrize("style", STYLES)
def test_dp_equals_bruteforce_random(style):
    n_feasible = 0
    for seed in range(2200):
        inst = gen.random_small(seed, Lmax=7, Kmax=4, Pmax=3, style=style)
        bf, _ = oracle.bruteforce(inst)
        dp = oracle.solve(inst)
        _same(bf, dp)
        if seed % 8 == 0:
            _same(bf, oracle.solve(inst, full_sweep=True))
            _same(bf, oracle.solve(inst, n_threads=3))
        if dp.feasible:
            n_feasible += 1
            s, T, it, mask = rescore(inst, dp.stages)
            assert (s, T, it, mask) == (dp.sum_us, dp.bottleneck_us, dp.iter_time_us, dp.island_mask)
    assert n_feasible > 500


def test_bruteforce_counts_compositions():
    # number of compositions for (L,K) = (8,3) is 171 when nothing is infeasible
    inst = gen.config1()
    _, n = oracle.bruteforce(inst)
    assert n == 171


@pytest.mark.parametrize("cap_div", [1, 10, 20])
def test_config1_and_tiny_mem_twins(cap_div):
    inst = gen.config1(0, cap_div)
    bf, _ = oracle.bruteforce(inst)
    _same(bf, oracle.solve(inst))
    _same(bf, oracle.solve(inst, full_sweep=True))


def test_larger_k5():
    for seed in range(60):
        inst = gen.random_small(seed + 10_000, Lmax=8, Kmax=5, Pmax=2, style="asym")
        bf, _ = oracle.bruteforce(inst)
        _same(bf, oracle.solve(inst))
