"""Seeded random sweep over what the other GPU tests fix by hand: batch sizes on both sides of every scheduling mode (1-4
instances: every probe of the last round back-tracks; <= 8: a warp lays out an instance's probes; < 64: rounds on CTA 0;
64-1024: queue mode; team vs solo by the item count), random shapes (L, K, P) and table styles, the core path and the four
variants of SURVEY.md §8(f) -- every instance against its oracle, value and plan, bit-exact through the C ABI.
(The same loop ran for seven minutes on the final kernels of round 2: 4 608 batches, 478 886 instances, no difference.)
The second test does the same with mid-size instances of the paper's workload shapes (K = 10-13 islands): team mode with
wide levels (two masks per warp, the split team barrier), the strided rank tables beyond K = 9, a K >= 10 batch on the
round scheduler.  (Its loop with random shapes ran for 13 minutes on the same kernels: 77 batches, 1 198 instances.)"""
import random

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


ORACLE = {"core": oracle.solve, "act": oracle.solve_depth, "xb": oracle.solve_variant, "bact": oracle.solve_variant_b,
          "st": lambda inst: oracle.solve_stages(inst)[0]}


def variant(kind, inst, s):
    if kind == "act":
        return gen.with_actmem(inst, s)
    if kind == "xb":
        return gen.with_transfer_bound(inst)
    if kind == "st":
        return gen.with_stages(inst, s, qmax=1 + s % 4)
    if kind == "bact":
        return gen.with_boundary_act(inst, s)
    return inst


@pytest.mark.parametrize("seed", [11, 12, 13])
def test_random_batches_shapes_and_variants(tg, seed):
    rng = random.Random(seed)
    n_inst = 0
    for _ in range(40):
        n = rng.choice([1, 2, 3, 4, 7, 8, 9, 20, 63, 64, 80, 150, 296, 300, 600])
        kind = rng.choice(["core", "core", "core", "act", "xb", "st", "bact"])
        Lmax, Kmax, Pmax = rng.choice([6, 9, 12, 16]), rng.choice([3, 5, 7, 9]), rng.choice([2, 3, 4, 7, 8])
        if n > 100:
            Lmax, Kmax = min(Lmax, 10), min(Kmax, 6)
        seed0 = rng.randrange(1 << 30)
        insts = [variant(kind, gen.random_small(seed0 + s, Lmax=Lmax, Kmax=Kmax, Pmax=Pmax, style=STYLES[(seed0 + s) % 5]), s)
                 for s in range(n)]
        hs = [tg.instance_from_inputs(i) for i in insts]
        res = tg.tg_solve_batch(hs)
        for inst, g in zip(insts, res):
            same(ORACLE[kind](inst), g, f"{kind} n={n} {inst.name} Lmax={Lmax} Kmax={Kmax} Pmax={Pmax} seed0={seed0}")
        for h in hs:
            h.destroy()
        n_inst += n
    assert n_inst > 1000


# (instances, shape, L, K, kind): about 25 s of oracle time in all
MID = [(1, "config3", 12, 13, "core"), (2, "config4", 16, 12, "core"), (3, "config3", 20, 12, "core"),
       (4, "config4", 16, 13, "core"), (9, "config3", 12, 11, "core"), (2, "config5_one", 24, 10, "core"),
       (1, "config5_one", 12, 10, "act"), (3, "config3", 12, 12, "xb"), (20, "config5_one", 12, 10, "core"),
       (5, "config3", 20, 10, "act")]


def test_mid_size_paper_shapes(tg):
    rng = random.Random(21)
    for n, shape, L, K, kind in MID:
        seed0 = rng.randrange(1 << 20)
        insts = [variant(kind, getattr(gen, shape)(seed0 + s, L=L, K=K), s) for s in range(n)]
        hs = [tg.instance_from_inputs(i) for i in insts]
        res = tg.tg_solve_batch(hs)
        for inst, g in zip(insts, res):
            same(ORACLE[kind](inst), g, f"{kind} n={n} {shape} L={L} K={K} seed0={seed0} {inst.name}")
        for h in hs:
            h.destroy()
