"""GPU parity of the per-boundary activation sizes (tg_instance_set_boundary_act, SURVEY.md §8(f) NEXT-3(b) second half)
against the variant oracle (orc_variant_solve_b), bit-exact on value and plan, through the C ABI."""
import numpy as np
import pytest

import oracle
import tg_inputs as gen
from test_oracle_boundary_act import rescore_b

pytestmark = pytest.mark.gpu
STYLES = ["mixed", "ties", "tightmem", "asym", "sparse"]
I64MAX = (1 << 63) - 1


@pytest.fixture(scope="module")
def tg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_16907_b200 as tg
    tg.lib()
    return tg


def stages_of(g):
    return [(int(g["stage_begin"][i]), int(g["stage_island"][i]), int(g["stage_plan"][i])) for i in range(int(g["n_stages"]))]


def same(inst, g, what=""):
    o = oracle.solve_variant_b(inst)
    feas = int(g["iter_time_us"]) != I64MAX
    assert o.feasible == feas, what
    if not feas:
        return
    assert (o.iter_time_us, o.sum_us, o.bottleneck_us, o.island_mask) == \
           (int(g["iter_time_us"]), int(g["sum_us"]), int(g["bottleneck_us"]), int(g["island_mask"])), what
    assert o.stages == stages_of(g), what
    assert rescore_b(inst, stages_of(g)) == (o.sum_us, o.bottleneck_us, o.iter_time_us, o.island_mask)


@pytest.mark.parametrize("style", STYLES)
def test_random_small_with_boundary_sizes(tg, style):
    insts = []
    for s in range(300):
        inst = gen.with_boundary_act(gen.random_small(9700 + s, Lmax=9, Kmax=6, Pmax=3, style=style), s,
                                     sizes=[(4, 64, 900), (16, 64, 256), (0, 64), (1, 2, 3, 5, 8, 13, 21, 34)][s % 4])
        if s % 2:
            inst = gen.with_transfer_bound(inst)
        if s % 5 == 0:
            inst = gen.with_actmem(inst, s, 0, 40)
        insts.append(inst)
    hs = [tg.instance_from_inputs(i) for i in insts]
    res = tg.tg_solve_batch(hs)
    for inst, g in zip(insts, res):
        same(inst, g, inst.name)
    for h in hs:
        h.destroy()


def test_mid_size_and_constant_size(tg):
    """Every config family at mid size, alone (team mode) and batched; a constant array equals the scalar instance."""
    insts = [gen.with_boundary_act(gen.config2(0), 1), gen.with_boundary_act(gen.config3(0, L=22, K=6), 2),
             gen.with_transfer_bound(gen.with_boundary_act(gen.config4(0, L=18, K=7), 3)),
             gen.with_boundary_act(gen.config5_one(3, L=21, K=6), 4, sizes=(8, 512))]
    hs = [tg.instance_from_inputs(i) for i in insts]
    for inst, h in zip(insts, hs):
        same(inst, tg.tg_solve_batch([h])[0], inst.name + " alone")
    for inst, g in zip(insts, tg.tg_solve_batch(hs)):
        same(inst, g, inst.name + " batched")
    for h in hs:
        h.destroy()
    for seed in range(20):
        base = gen.random_small(9900 + seed, Lmax=10, Kmax=6, Pmax=3, style=STYLES[seed % 5])
        h = tg.instance_from_inputs(base)
        core = tg.tg_solve_batch([h])[0]
        tg.tg_instance_set_boundary_act(h, np.full(base.L + 1, base.act_mb, dtype=np.int32))
        a = tg.tg_solve_batch([h])[0]
        assert a.tobytes()[:24] == core.tobytes()[:24] and stages_of(a) == stages_of(core)
        var = gen.with_boundary_act(base, seed)
        tg.tg_instance_set_boundary_act(h, var.act_mb_b)
        same(var, tg.tg_solve_batch([h])[0], "switched on a live instance")
        tg.tg_instance_set_boundary_act(h, None)
        b = tg.tg_solve_batch([h])[0]
        assert b.tobytes()[:24] == core.tobytes()[:24] and stages_of(b) == stages_of(core)
        h.destroy()


def test_boundary_act_errors(tg):
    base = next(b for b in (gen.random_small(s, Lmax=12, Kmax=4, Pmax=3, style="mixed") for s in range(9990, 10400)) if b.L >= 11)
    h = tg.instance_from_inputs(base)
    with pytest.raises(tg.TangramError) as e:                      # nine distinct sizes
        tg.tg_instance_set_boundary_act(h, np.arange(base.L + 1, dtype=np.int32))
    assert e.value.status == 2
    bad = np.full(base.L + 1, 5, dtype=np.int32)
    bad[1] = -1
    with pytest.raises(tg.TangramError) as e:
        tg.tg_instance_set_boundary_act(h, bad)
    assert e.value.status == 3
    tg.tg_instance_set_boundary_act(h, np.full(base.L + 1, 5, dtype=np.int32))
    st = gen.with_stages(base, 1)
    with pytest.raises(tg.TangramError) as e:
        tg.tg_instance_set_stages(h, st.slow_us)
    assert e.value.status == 2
    h.destroy()
