"""GPU parity of SURVEY.md §8(f) NEXT-1 (depth-aware activation memory, tg_instance_set_actmem) against
oracle.solve_depth: value and plan, bit-exact, through the C ABI."""
import numpy as np
import pytest

import oracle
import tg_inputs as gen
from test_gpu_parity import same, solve_all, STYLES
from test_oracle_depth import rescore_depth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_16907_b200 as tg
    tg.lib()
    return tg


@pytest.mark.parametrize("style", STYLES)
def test_random_small_with_actmem(tg, style):
    insts = [gen.with_actmem(gen.random_small(s + 70_000, Lmax=8, Kmax=5, Pmax=3, style=style), s) for s in range(300)]
    res = solve_all(tg, insts)
    differs = 0
    for inst, g in zip(insts, res):
        o = oracle.solve_depth(inst)
        same(o, g, inst.name)
        if o.feasible:
            differs += oracle.solve(inst).plan_key() != o.plan_key()     # oracle.solve ignores actmem_mb
    assert differs > 10, "the footprint should change some optima"


def test_mid_size_with_actmem(tg):
    """Several team sizes, ragged rows, row windows and per-level restaging of the cost rows."""
    insts = [gen.with_actmem(gen.config3(0, L=22, K=7), 1, 500, 6000), gen.with_actmem(gen.config4(0, L=18, K=8), 2, 2000, 20000),
             gen.with_actmem(gen.config5_one(3, L=20, K=6), 3, 2000, 20000), gen.with_actmem(gen.config2(), 4, 0, 2000)]
    for alone in (False, True):
        groups = [[i] for i in insts] if alone else [insts]
        for grp in groups:
            for inst, g in zip(grp, solve_all(tg, grp)):
                o = oracle.solve_depth(inst)
                same(o, g, inst.name)
                if o.feasible:
                    n = int(g["n_stages"])
                    st = [(int(g["stage_begin"][i]), int(g["stage_island"][i]), int(g["stage_plan"][i])) for i in range(n)]
                    assert rescore_depth(inst, st) == (int(g["sum_us"]), int(g["bottleneck_us"]), int(g["iter_time_us"]), int(g["island_mask"]))


def test_zero_footprint_and_removal(tg):
    base = gen.config2()
    h = tg.instance_from_inputs(base)
    core = tg.tg_solve_batch([h])[0].copy()
    tg.tg_instance_set_actmem(h, np.zeros_like(base.time_us))
    same(oracle.solve(base), tg.tg_solve_batch([h])[0], "zero footprint")
    heavy = gen.with_actmem(base, 9, 1000, 4000)
    tg.tg_instance_set_actmem(h, heavy.actmem_mb)
    same(oracle.solve_depth(heavy), tg.tg_solve_batch([h])[0], "heavy footprint")
    tg.tg_instance_set_actmem(h, None)
    assert tg.tg_solve_batch([h])[0].tobytes()[:24] == core.tobytes()[:24]      # iter, sum, T restored
    h.destroy()


def test_errors_with_actmem(tg):
    inst = gen.with_actmem(gen.config1(), 0)
    h = tg.instance_from_inputs(inst)
    bad = inst.actmem_mb.copy(); bad[2, 1, 0] = -1
    with pytest.raises(tg.TangramError) as e:
        tg.tg_instance_set_actmem(h, bad)
    assert e.value.status == 3
    h.destroy()


def test_full_size_cfg3_with_actmem(tg):
    """Full-size 70B-like config with a footprint; stored result of the depth oracle
    (tests/golden/make_expected.py cfg3d)."""
    import json, os
    p = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "expected_cfg3d.json")
    e = json.load(open(p))["records"][0]
    inst = gen.with_actmem(gen.config3(), 7, 500, 6000)
    g = solve_all(tg, [inst])[0]
    n = int(g["n_stages"])
    got = [int(g["iter_time_us"]), int(g["sum_us"]), int(g["bottleneck_us"]), int(g["island_mask"]),
           [[int(g["stage_begin"][i]), int(g["stage_island"][i]), int(g["stage_plan"][i])] for i in range(n)]]
    s = e["solve"]
    assert got == [s["iter_time_us"], s["sum_us"], s["bottleneck_us"], s["island_mask"], s["stages"]]
    assert s["iter_time_us"] >= e["core"]["iter_time_us"]
    st = [tuple(x) for x in got[4]]
    assert rescore_depth(inst, st) == (got[1], got[2], got[0], got[3])


def test_full_size_cfg4_with_actmem(tg):
    """The K = 16 depth-aware workload bench.py times as `cfg4d` (full-size MoE-like config with a footprint, the loader
    restaging its cost rows at each of 16 levels); stored result of the variant oracle
    (tests/golden/make_expected.py cfg4d) and of the core oracle for the same tables without the footprint."""
    import json, os
    here = os.path.dirname(os.path.abspath(__file__))
    e = json.load(open(os.path.join(here, "golden", "expected_cfg4d.json")))["records"][0]
    core = json.load(open(os.path.join(here, "golden", "expected_cfg4.json")))["records"][0]
    inst = gen.with_actmem(gen.config4(), 11, 300, 3000)
    g = solve_all(tg, [inst])[0]
    n = int(g["n_stages"])
    got = [int(g["iter_time_us"]), int(g["sum_us"]), int(g["bottleneck_us"]), int(g["island_mask"]),
           [[int(g["stage_begin"][i]), int(g["stage_island"][i]), int(g["stage_plan"][i])] for i in range(n)]]
    s = e["solve"]
    assert got == [s["iter_time_us"], s["sum_us"], s["bottleneck_us"], s["island_mask"], s["stages"]]
    assert s["iter_time_us"] >= core["solve"]["iter_time_us"]          # a footprint never improves the optimum
    st = [tuple(x) for x in got[4]]
    assert rescore_depth(inst, st) == (got[1], got[2], got[0], got[3])
