"""GPU parity of SURVEY.md §8(f) NEXT-2 (multi-stage partial plans, tg_instance_set_stages) against the stages oracle
(oracle/tangram_oracle_stages.cpp), bit-exact on value, plan and pipeline-stage count, through the C ABI."""
import numpy as np
import pytest

import oracle
import tg_inputs as gen
from test_oracle_stages import rescore_stages

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


def same(tg, inst, h, g, what=""):
    o, tq = oracle.solve_stages(inst)
    feas = int(g["iter_time_us"]) != I64MAX
    assert o.feasible == feas, what
    if not feas:
        assert int(g["n_stages"]) == 0
        return
    assert (o.iter_time_us, o.sum_us, o.bottleneck_us, o.island_mask) == \
           (int(g["iter_time_us"]), int(g["sum_us"]), int(g["bottleneck_us"]), int(g["island_mask"])), what
    assert o.stages == stages_of(g), what
    assert tg.tg_plan_pipeline_stages(h, g) == tq, what
    assert rescore_stages(inst, stages_of(g))[:4] == (o.sum_us, o.bottleneck_us, o.iter_time_us, o.island_mask)


@pytest.mark.parametrize("style", STYLES)
def test_random_small_with_stages(tg, style):
    insts = [gen.with_stages(gen.random_small(8000 + s, Lmax=9, Kmax=6, Pmax=4, style=style), s, qmax=1 + s % 4) for s in range(300)]
    hs = [tg.instance_from_inputs(i) for i in insts]
    res = tg.tg_solve_batch(hs)
    for inst, h, g in zip(insts, hs, res):
        same(tg, inst, h, g, inst.name)
    full = tg.tg_solve_batch(hs[:60], flags=tg.TG_SOLVE_FULL_SWEEP)        # every candidate threshold: same answer
    for inst, h, g in zip(insts[:60], hs[:60], full):
        same(tg, inst, h, g, inst.name + " full sweep")
    for h in hs:
        h.destroy()


def test_mid_size_with_stages(tg):
    """Every config family at a size the oracle finishes in seconds (several tiles, ragged tails), alone (team mode, the
    L2 fallback at wide thresholds) and in one batch, plus the transfer bound on top."""
    insts = [gen.with_stages(gen.config2(0), 1), gen.with_stages(gen.config3(0, L=22, K=6), 2),
             gen.with_stages(gen.config4(0, L=18, K=7), 3), gen.with_stages(gen.config5_one(3, L=21, K=6), 4),
             gen.with_transfer_bound(gen.with_stages(gen.config3(1, L=19, K=5), 5))]
    hs = [tg.instance_from_inputs(i) for i in insts]
    for inst, h in zip(insts, hs):
        if inst.transfer_bound:
            continue                                    # (the stages oracle has no transfer bound: batch-vs-alone below)
        same(tg, inst, h, tg.tg_solve_batch([h])[0], inst.name + " alone")
    res = tg.tg_solve_batch(hs)
    for inst, h, g in zip(insts, hs, res):
        if not inst.transfer_bound:
            same(tg, inst, h, g, inst.name + " batched")
    alone = tg.tg_solve_batch([hs[4]])[0]
    assert alone.tobytes()[:24] == res[4].tobytes()[:24] and stages_of(alone) == stages_of(res[4])
    for h in hs:
        h.destroy()


def test_single_stage_tables_are_the_core_path(tg):
    """slow_us == time_us: results identical to the instance without the tables; removing the tables restores it."""
    for seed in range(20):
        base = gen.random_small(8600 + seed, Lmax=10, Kmax=6, Pmax=4, style=STYLES[seed % 5])
        h = tg.instance_from_inputs(base)
        core = tg.tg_solve_batch([h])[0]
        tg.tg_instance_set_stages(h, np.where(base.time_us == 0x7FFFFFFF, 0, base.time_us).astype(np.int32))
        a = tg.tg_solve_batch([h])[0]
        assert a.tobytes()[:24] == core.tobytes()[:24] and stages_of(a) == stages_of(core)
        st = gen.with_stages(base, seed)
        tg.tg_instance_set_stages(h, st.slow_us, st.q_stages)
        same(tg, st, h, tg.tg_solve_batch([h])[0], "switched on a live instance")
        tg.tg_instance_set_stages(h, None)
        b = tg.tg_solve_batch([h])[0]
        assert b.tobytes()[:24] == core.tobytes()[:24] and stages_of(b) == stages_of(core)
        h.destroy()


def test_stage_errors(tg):
    base = gen.random_small(8700, Lmax=6, Kmax=4, Pmax=3, style="mixed")
    st = gen.with_stages(base, 1)
    h = tg.instance_from_inputs(base)
    bad = st.slow_us.copy()
    bad[base.time_us != 0x7FFFFFFF] += 1 << 26                     # slow > time
    with pytest.raises(tg.TangramError) as e:
        tg.tg_instance_set_stages(h, bad)
    assert e.value.status == 3
    q = st.q_stages.copy()
    q[0, 0, 0] = 0
    with pytest.raises(tg.TangramError) as e:
        tg.tg_instance_set_stages(h, st.slow_us, q)
    assert e.value.status == 3
    tg.tg_instance_set_stages(h, st.slow_us, st.q_stages)
    with pytest.raises(tg.TangramError) as e:                      # not combinable with the footprint table
        tg.tg_instance_set_actmem(h, np.zeros_like(base.time_us))
    assert e.value.status == 2
    with pytest.raises(tg.TangramError) as e:
        tg.tg_prune(h)
    assert e.value.status == 2
    h.destroy()
    h = tg.instance_from_inputs(gen.with_actmem(base, 1, 0, 10))
    with pytest.raises(tg.TangramError) as e:
        tg.tg_instance_set_stages(h, st.slow_us)
    assert e.value.status == 2
    h.destroy()


def test_full_size_cfg3_with_stages(tg):
    """Full-size 70B-like config with multi-stage partial plans; stored result of the stages oracle
    (tests/golden/make_expected.py cfg3st)."""
    import json, os
    p = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "expected_cfg3st.json")
    e = json.load(open(p))["records"][0]
    inst = gen.with_stages(gen.config3(), 3)
    h = tg.instance_from_inputs(inst)
    g = tg.tg_solve_batch([h])[0]
    s = e["solve"]
    got = [int(g["iter_time_us"]), int(g["sum_us"]), int(g["bottleneck_us"]), int(g["island_mask"]), [list(t) for t in stages_of(g)]]
    assert got == [s["iter_time_us"], s["sum_us"], s["bottleneck_us"], s["island_mask"], s["stages"]]
    assert tg.tg_plan_pipeline_stages(h, g) == e["pipeline_stages"]
    assert rescore_stages(inst, stages_of(g))[:4] == (got[1], got[2], got[0], got[3])
    h.destroy()
