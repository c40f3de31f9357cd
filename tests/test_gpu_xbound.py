"""GPU parity of SURVEY.md §8(f) NEXT-3(b) (transfers bounded by the threshold, tg_instance_set_transfer_bound)
against oracle.solve_variant: value and plan, bit-exact, through the C ABI; alone and with NEXT-1's footprint."""
import json
import os

import numpy as np
import pytest

import oracle
import tg_inputs as gen
from test_gpu_parity import same, solve_all, STYLES
from test_oracle_xbound import rescore_xbound

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_16907_b200 as tg
    tg.lib()
    return tg


def stages_of(g):
    n = int(g["n_stages"])
    return [(int(g["stage_begin"][i]), int(g["stage_island"][i]), int(g["stage_plan"][i])) for i in range(n)]


@pytest.mark.parametrize("style", STYLES)
def test_random_small_with_transfer_bound(tg, style):
    insts = [gen.with_transfer_bound(gen.random_small(s + 90_000, Lmax=8, Kmax=5, Pmax=3, style=style)) for s in range(300)]
    differs = 0
    for inst, g in zip(insts, solve_all(tg, insts)):
        o = oracle.solve_variant(inst)
        same(o, g, inst.name)
        if o.feasible:
            differs += oracle.solve(inst).plan_key() != o.plan_key()     # oracle.solve ignores the flag
    assert differs >= 3, "the bound should change some optima"


def test_random_small_with_transfer_bound_and_actmem(tg):
    insts = [gen.with_transfer_bound(gen.with_actmem(gen.random_small(s + 91_000, Lmax=8, Kmax=5, Pmax=3, style=STYLES[s % 5]), s))
             for s in range(300)]
    for inst, g in zip(insts, solve_all(tg, insts)):
        same(oracle.solve_variant(inst), g, inst.name)


def test_mid_size_with_transfer_bound(tg):
    """Every config family (their links are 160..2560 us, around the stage times: the bound binds), alone and batched,
    with and without the footprint."""
    insts = [gen.with_transfer_bound(gen.config3(0, L=22, K=7)), gen.with_transfer_bound(gen.config4(0, L=18, K=8)),
             gen.with_transfer_bound(gen.config5_one(3, L=20, K=6)), gen.with_transfer_bound(gen.config2()),
             gen.with_transfer_bound(gen.with_actmem(gen.config4(1, L=16, K=7), 2, 2000, 20000))]
    changed = 0
    for alone in (False, True):
        groups = [[i] for i in insts] if alone else [insts]
        for grp in groups:
            for inst, g in zip(grp, solve_all(tg, grp)):
                o = oracle.solve_variant(inst)
                same(o, g, inst.name)
                if o.feasible:
                    assert rescore_xbound(inst, stages_of(g)) == (int(g["sum_us"]), int(g["bottleneck_us"]),
                                                                  int(g["iter_time_us"]), int(g["island_mask"]))
                    if inst.actmem_mb is None:
                        changed += oracle.solve(inst).plan_key() != o.plan_key()
    assert changed >= 2


def test_switching_the_bound_on_and_off(tg):
    base = gen.config2()
    h = tg.instance_from_inputs(base)
    same(oracle.solve(base), tg.tg_solve_batch([h])[0], "off")
    tg.tg_instance_set_transfer_bound(h, True)
    same(oracle.solve_variant(gen.with_transfer_bound(base)), tg.tg_solve_batch([h])[0], "on")
    tg.tg_instance_set_transfer_bound(h, False)
    same(oracle.solve(base), tg.tg_solve_batch([h])[0], "off again")
    full = tg.tg_solve_batch([h], flags=tg.TG_SOLVE_FULL_SWEEP)[0]
    same(oracle.solve(base), full, "full sweep")
    tg.tg_instance_set_transfer_bound(h, True)
    same(oracle.solve_variant(gen.with_transfer_bound(base)), tg.tg_solve_batch([h], flags=tg.TG_SOLVE_FULL_SWEEP)[0], "on, full sweep")


def test_full_size_cfg3_with_transfer_bound(tg):
    """Full-size 70B-like config; stored result of the variant oracle (tests/golden/make_expected.py cfg3xb)."""
    p = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "expected_cfg3xb.json")
    e = json.load(open(p))["records"][0]
    inst = gen.with_transfer_bound(gen.config3())
    g = solve_all(tg, [inst])[0]
    got = [int(g["iter_time_us"]), int(g["sum_us"]), int(g["bottleneck_us"]), int(g["island_mask"]), [list(t) for t in stages_of(g)]]
    s = e["solve"]
    assert got == [s["iter_time_us"], s["sum_us"], s["bottleneck_us"], s["island_mask"], s["stages"]]
    assert s["iter_time_us"] >= e["core"]["iter_time_us"]
    assert rescore_xbound(inst, stages_of(g)) == (got[1], got[2], got[0], got[3])


def test_full_size_cfg4_with_transfer_bound(tg):
    """The K = 16 workload bench.py times as `cfg4xb`; stored result of the variant oracle
    (tests/golden/make_expected.py cfg4xb) and of the core oracle for the same tables without the bound."""
    here = os.path.dirname(os.path.abspath(__file__))
    e = json.load(open(os.path.join(here, "golden", "expected_cfg4xb.json")))["records"][0]
    core = json.load(open(os.path.join(here, "golden", "expected_cfg4.json")))["records"][0]
    inst = gen.with_transfer_bound(gen.config4())
    g = solve_all(tg, [inst])[0]
    got = [int(g["iter_time_us"]), int(g["sum_us"]), int(g["bottleneck_us"]), int(g["island_mask"]), [list(t) for t in stages_of(g)]]
    s = e["solve"]
    assert got == [s["iter_time_us"], s["sum_us"], s["bottleneck_us"], s["island_mask"], s["stages"]]
    assert s["iter_time_us"] >= core["solve"]["iter_time_us"]          # bounding the transfers never improves the optimum
    assert rescore_xbound(inst, stages_of(g)) == (got[1], got[2], got[0], got[3])


def test_reduce_and_candidates_on_variant_instances(tg):
    """tg_reduce never writes past its documented capacity NS*K although a variant instance has more thresholds (all
    depths / the transfer times); tg_candidates returns the whole list.  Expected lists: the transfer-bound list is the
    union of the oracle's finite depth-1 costs and finite off-diagonal transfers; with a footprint the count is the
    variant oracle's n_candidates and the list is sorted, distinct and contains every depth-1 cost."""
    for seed in range(12):
        base = gen.random_small(700 + seed, Lmax=3, Kmax=5, Pmax=3, style=STYLES[seed % 5])
        NS = base.L * (base.L + 1) // 2
        oc, _, ox, ocand = oracle.reduce(base)
        for variant in ("xb", "act", "both"):
            inst = base
            if variant in ("act", "both"):
                inst = gen.with_actmem(inst, seed, 0, 40)
            if variant in ("xb", "both"):
                inst = gen.with_transfer_bound(inst)
            h = tg.instance_from_inputs(inst)
            guard = np.full(NS * base.K + 64, -7, dtype=np.int32)            # room behind the documented capacity
            n = np.zeros(1, dtype=np.int32)
            import ctypes as C
            st = tg.lib().tg_reduce(h.handle, None, None, None, guard.ctypes.data, n.ctypes.data_as(C.POINTER(C.c_int32)), None)
            assert st == 0 and (guard[NS * base.K:] == -7).all(), "tg_reduce wrote past NS*K"
            c, argp, x, cand_r = tg.tg_reduce(h)
            cand = tg.tg_candidates(h).astype(np.int64)
            assert int(n[0]) == cand.size and np.array_equal(cand[:cand_r.size], cand_r.astype(np.int64))
            assert cand_r.size == min(cand.size, NS * base.K)
            assert (np.diff(cand) > 0).all()
            assert cand.size == oracle.solve_variant(inst).n_candidates
            assert np.array_equal(x.astype(np.int64), ox)
            if variant == "xb":                                               # depth-1 tables are the core tables
                assert np.array_equal(c.astype(np.int64), oc)
                fx = ox[(ox < (1 << 30)) & ~np.eye(base.K, dtype=bool)]
                assert np.array_equal(cand, np.union1d(ocand, fx))
            else:                                                             # depth 1 of the footprint: a subset of the list
                assert np.isin(c[c < (1 << 30)].astype(np.int64), cand).all()
            h.destroy()
