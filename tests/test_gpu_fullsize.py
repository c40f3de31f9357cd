"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (one
tg_solve_batch of resident instances).  Expected values were written by tests/golden/make_expected.py,
which calls only the CPU oracle (minutes of CPU time, hence stored).  Plus properties that hold at any
size: the independent re-scorer reproduces (sum, T, iter, mask) from the RAW tables; full sweep ==
windowed sweep."""
import json
import os

import numpy as np
import pytest

import tg_inputs as gen
from conftest import rescore

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))
I64MAX = (1 << 63) - 1


@pytest.fixture(scope="module")
def tg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_16907_b200 as tg
    tg.lib()
    return tg


def expected(name):
    p = os.path.join(HERE, "golden", f"expected_{name}.json")
    if not os.path.exists(p):
        pytest.fail(f"{p} missing: run tests/golden/make_expected.py {name}")
    with open(p) as f:
        return json.load(f)["records"]


def check(exp, g, what):
    if not exp["feasible"]:
        assert int(g["iter_time_us"]) == I64MAX and int(g["n_stages"]) == 0, what
        return
    n = int(g["n_stages"])
    got = [int(g["iter_time_us"]), int(g["sum_us"]), int(g["bottleneck_us"]), int(g["island_mask"]),
           [[int(g["stage_begin"][i]), int(g["stage_island"][i]), int(g["stage_plan"][i])] for i in range(n)]]
    want = [exp["iter_time_us"], exp["sum_us"], exp["bottleneck_us"], exp["island_mask"], exp["stages"]]
    assert got == want, what


def check_rescore(inst, g):
    n = int(g["n_stages"])
    st = [(int(g["stage_begin"][i]), int(g["stage_island"][i]), int(g["stage_plan"][i])) for i in range(n)]
    s, T, it, mask = rescore(inst, st)
    assert (s, T, it, mask) == (int(g["sum_us"]), int(g["bottleneck_us"]), int(g["iter_time_us"]), int(g["island_mask"]))


def rec(r):
    return {k: getattr(r, k) for k, _ in r._fields_}


@pytest.mark.parametrize("name", ["cfg3", "cfg4"])
def test_full_config_solve_and_single_dps(tg, name):
    exp = expected(name)[0]
    inst = gen.by_name(name)
    assert (inst.L, inst.K, inst.P, inst.m) == (exp["L"], exp["K"], exp["P"], exp["m"])
    h = tg.instance_from_inputs(inst)
    g = tg.tg_solve_batch([h])[0]
    check(exp["solve"], g, name)
    check_rescore(inst, g)
    for d in exp["dp_at"]:
        r = rec(tg.tg_dp_at(h, d["T"]))
        e = dict(d["res"])
        check(e, r, f"{name} dp_at T={d['T']}")
    h.destroy()


def test_full_sweep_matches_on_cfg3(tg):
    exp = expected("cfg3")[0]
    h = tg.instance_from_inputs(gen.config3())
    st = tg.TgSolveStats()
    g = tg.tg_solve_batch([h], flags=tg.TG_SOLVE_FULL_SWEEP, stats=st)[0]
    check(exp["solve"], g, "cfg3 full sweep")
    assert st.n_dp >= exp["solve"]["n_candidates"]
    h.destroy()


def test_cfg5_batch_1024(tg):
    """The whole throughput batch in ONE tg_solve_batch call; EVERY instance against its stored oracle result (value
    and plan, tests/golden/make_expected.py cfg5: all 1024 seeds) and against the re-scorer."""
    exp = {r["seed"]: r for r in expected("cfg5")}
    assert sorted(exp) == list(range(1024))
    insts = gen.config5(1024)
    hs = [tg.instance_from_inputs(i) for i in insts]
    res = tg.tg_solve_batch(hs)
    for h in hs:
        h.destroy()
    for seed, r in exp.items():
        assert insts[seed].m == r["m"]
        check(r["solve"], res[seed], f"cfg5 seed {seed}")
    for inst, g in zip(insts, res):
        assert int(g["iter_time_us"]) != I64MAX
        check_rescore(inst, g)


def test_more_full_size_seeds(tg):
    """Other seeds of the 70B-like and MoE-like configs (different island mixes, hence different threshold
    windows and row windows) in one batch; stored oracle results (tests/golden/make_expected.py cfg3x cfg4x)."""
    exp3 = {r["seed"]: r for r in expected("cfg3x")}
    exp4 = {r["seed"]: r for r in expected("cfg4x")}
    insts = [gen.config3(s) for s in exp3] + [gen.config4(s) for s in exp4]
    exps = list(exp3.values()) + list(exp4.values())
    hs = [tg.instance_from_inputs(i) for i in insts]
    res = tg.tg_solve_batch(hs)
    for h in hs:
        h.destroy()
    for inst, e, g in zip(insts, exps, res):
        check(e["solve"], g, inst.name)
        check_rescore(inst, g)
