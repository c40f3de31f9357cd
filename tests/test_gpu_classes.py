"""GPU parity of SURVEY.md §8(f) NEXT-3(a) (tables per signature class, tg_instance_create_classes):
by definition the instance is the expanded one, so the oracle is the core oracle on the expanded tables."""
import numpy as np
import pytest

import oracle
import tg_inputs as gen
from test_gpu_parity import same, STYLES

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_16907_b200 as tg
    tg.lib()
    return tg


def create(tg, inst, class_of, ct, cm):
    return tg.tg_instance_create_classes(inst.L, inst.K, inst.P, inst.m, class_of, ct, cm, inst.island_gpus,
                                         inst.island_cap_mb, inst.bw_gbps, inst.act_mb)


def test_length_classes_equal_the_expanded_instance(tg):
    bases = [gen.random_small(s + 97_000, Lmax=8, Kmax=5, Pmax=3, style=STYLES[s % 5]) for s in range(120)] + \
            [gen.config2(), gen.config3(0, L=22, K=7), gen.config4(0, L=18, K=8), gen.config5_one(1, L=20, K=6)]
    hs, exp = [], []
    for b in bases:
        class_of, ct, cm, e = gen.length_classes(b)
        assert ct.shape == (b.L, b.K, b.P)
        hs.append(create(tg, b, class_of, ct, cm))
        exp.append(e)
    for h, e in zip(hs[-4:], exp[-4:]):
        assert np.array_equal(tg.tg_instance_read_time(h), e.time_us)       # the device expansion is the definition
    res = tg.tg_solve_batch(hs)
    res_exp = tg.tg_solve_batch([tg.instance_from_inputs(e) for e in exp])
    n_feasible = 0
    for e, g, g2 in zip(exp, res, res_exp):
        o = oracle.solve(e)
        same(o, g, e.name)
        same(o, g2, e.name + " (expanded on the host)")
        n_feasible += o.feasible
    assert n_feasible > 60
    for h in hs:
        h.destroy()


def test_class_instances_in_a_batch_that_fills_the_gpu(tg):
    """320 class instances of one P: the batch takes the row-group loader, which reads a cell's row through the class map
    (the mixed batch above takes the cell-order loader)."""
    bases = [gen.config5_one(s + 40, L=11 + s % 6, K=5 + s % 3) for s in range(320)]
    hs, exp = [], []
    for b in bases:
        class_of, ct, cm, e = gen.length_classes(b)
        hs.append(create(tg, b, class_of, ct, cm))
        exp.append(e)
    for e, g in zip(exp, tg.tg_solve_batch(hs)):
        same(oracle.solve(e), g, e.name)
    for h in hs:
        h.destroy()


def test_arbitrary_classes(tg):
    """Classes need not be slice lengths: random class maps with as few as one class and as many as NS."""
    for seed in range(40):
        b = gen.random_small(seed + 98_000, Lmax=7, Kmax=4, Pmax=3, style=STYLES[seed % 5])
        NS = b.L * (b.L + 1) // 2
        nc = [1, 2, NS, max(1, NS // 2)][seed % 4]
        class_of = gen.urand(seed, 777, np.arange(NS), 0, nc - 1).astype(np.int32)
        ct, cm = b.time_us[:nc].copy(), b.mem_mb[:nc].copy()
        e = b.copy()
        e.time_us, e.mem_mb = ct[class_of], cm[class_of]
        h = create(tg, b, class_of, ct, cm)
        same(oracle.solve(e), tg.tg_solve_batch([h])[0], f"seed {seed}")
        h.destroy()


def test_class_errors(tg):
    b = gen.config2()
    class_of, ct, cm, _ = gen.length_classes(b)
    bad = class_of.copy()
    bad[3] = b.L                                   # one past the last class
    with pytest.raises(tg.TangramError) as e:
        create(tg, b, bad, ct, cm)
    assert e.value.status == 3 and "32" in str(e.value)
    bad[3] = -1
    with pytest.raises(tg.TangramError) as e:
        create(tg, b, bad, ct, cm)
    assert e.value.status == 3
    neg = ct.copy()
    neg[0, 0, 0] = -5
    with pytest.raises(tg.TangramError) as e:
        create(tg, b, class_of, neg, cm)
    assert e.value.status == 3
    with pytest.raises(tg.TangramError) as e:        # more classes than slices
        NS = b.L * (b.L + 1) // 2
        big = np.zeros((NS + 1, b.K, b.P), np.int32)
        create(tg, b, class_of, big, big)
    assert e.value.status == 2


def test_class_instances_after_prune_and_variant_tables(tg):
    """The loader of a class instance reads the class tables; pruning or attaching footprint / stage tables makes the
    expanded tables the instance (the class tables would be stale): results must follow the expanded definition."""
    for seed in range(12):
        b = gen.random_small(seed + 99_000, Lmax=8, Kmax=5, Pmax=3, style=STYLES[seed % 5])
        class_of, ct, cm, e = gen.length_classes(b)
        h = create(tg, b, class_of, ct, cm)
        same(oracle.solve(e), tg.tg_solve_batch([h])[0], "class tables")
        tg.tg_prune(h, tg.TG_PRUNE_BOTTLENECK, int(np.median(e.time_us[e.time_us != 0x7FFFFFFF])))
        pr, _ = oracle.prune(e, 2, int(np.median(e.time_us[e.time_us != 0x7FFFFFFF])))
        g = tg.tg_solve_batch([h])[0]
        o = oracle.solve(pr)
        assert o.feasible == (int(g["iter_time_us"]) != (1 << 63) - 1)
        if o.feasible:
            assert (o.iter_time_us, o.bottleneck_us, o.island_mask) == (int(g["iter_time_us"]), int(g["bottleneck_us"]), int(g["island_mask"]))
        h.destroy()
        h = create(tg, b, class_of, ct, cm)
        ea = gen.with_actmem(e, seed, 0, 40)
        tg.tg_instance_set_actmem(h, ea.actmem_mb)
        od = oracle.solve_depth(ea)
        g = tg.tg_solve_batch([h])[0]
        assert od.feasible == (int(g["iter_time_us"]) != (1 << 63) - 1)
        if od.feasible:
            assert (od.iter_time_us, od.bottleneck_us, od.island_mask) == (int(g["iter_time_us"]), int(g["bottleneck_us"]), int(g["island_mask"]))
        h.destroy()
