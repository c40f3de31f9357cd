"""GPU parity: every step of the CUDA path against the CPU oracle, bit-exact, through the C ABI
(paper_2606_16907_b200 is argument marshalling only).  Integer work: no tolerance anywhere."""
import numpy as np
import pytest

import oracle
import tg_inputs as gen
from conftest import rescore

pytestmark = pytest.mark.gpu

STYLES = ["mixed", "ties", "tightmem", "asym", "sparse"]


@pytest.fixture(scope="module")
def tg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_16907_b200 as tg
    tg.lib()
    return tg


def same(o, g, what=""):
    """o: oracle.Result, g: numpy record or TgResult"""
    feas = int(g["iter_time_us"]) != (1 << 63) - 1
    assert o.feasible == feas, what
    if not feas:
        assert int(g["n_stages"]) == 0
        return
    n = int(g["n_stages"])
    stages = [(int(g["stage_begin"][i]), int(g["stage_island"][i]), int(g["stage_plan"][i])) for i in range(n)]
    assert (o.iter_time_us, o.sum_us, o.bottleneck_us, o.island_mask) == \
           (int(g["iter_time_us"]), int(g["sum_us"]), int(g["bottleneck_us"]), int(g["island_mask"])), what
    assert o.stages == stages, what


def rec(r):
    return {k: getattr(r, k) for k, _ in r._fields_}


def solve_all(tg, insts, flags=0):
    hs = [tg.instance_from_inputs(i) for i in insts]
    res = tg.tg_solve_batch(hs, flags=flags)
    for h in hs:
        h.destroy()
    return res


def test_reduce_steps_1_to_3(tg):
    for inst in [gen.config1(), gen.config1(0, 10), gen.config2(), gen.random_small(5, style="sparse"),
                 gen.random_small(7, style="tightmem"), gen.config3(0, L=20, K=5)]:
        h = tg.instance_from_inputs(inst)
        c, argp, x, cand = tg.tg_reduce(h)
        oc, oargp, ox, ocand = oracle.reduce(inst)
        assert np.array_equal(c.astype(np.int64), oc)
        assert np.array_equal(argp, oargp)
        assert np.array_equal(x.astype(np.int64), ox)
        assert np.array_equal(cand.astype(np.int64), ocand)
        h.destroy()


@pytest.mark.parametrize("style", STYLES)
def test_random_small_batches(tg, style):
    insts = [gen.random_small(s, Lmax=9, Kmax=6, Pmax=3, style=style) for s in range(400)]
    res = solve_all(tg, insts)
    for inst, g in zip(insts, res):
        same(oracle.solve(inst), g, inst.name)


def test_full_sweep_equals_windowed(tg):
    insts = [gen.random_small(s + 900, Lmax=8, Kmax=5, Pmax=3, style=STYLES[s % 5]) for s in range(100)]
    a = solve_all(tg, insts)
    b = solve_all(tg, insts, flags=1)
    for inst, ga, gb in zip(insts, a, b):
        o = oracle.solve(inst)
        same(o, ga, inst.name)
        same(o, gb, inst.name + " full")


def test_config1_and_twins(tg):
    insts = [gen.config1(0, d) for d in (1, 10, 20)]
    for inst, g in zip(insts, solve_all(tg, insts)):
        same(oracle.solve(inst), g, inst.name)


def test_config2(tg):
    inst = gen.config2()
    g = solve_all(tg, [inst])[0]
    o = oracle.solve(inst)
    same(o, g, inst.name)
    st = [(int(g["stage_begin"][i]), int(g["stage_island"][i]), int(g["stage_plan"][i])) for i in range(int(g["n_stages"]))]
    s, T, it, mask = rescore(inst, st)
    assert (s, T, it, mask) == (int(g["sum_us"]), int(g["bottleneck_us"]), int(g["iter_time_us"]), int(g["island_mask"]))


def test_dp_at_single_threshold(tg):
    """Step 5 + 7 at one T against oracle.dp_at, including T = infinity and infeasible T."""
    for inst in [gen.config1(), gen.config2(), gen.random_small(11, style="asym"), gen.config3(0, L=24, K=7)]:
        h = tg.instance_from_inputs(inst)
        _, _, _, cand = oracle.reduce(inst)
        picks = [-1, int(cand[0]), int(cand[len(cand) // 3]), int(cand[len(cand) // 2]), int(cand[-1]), int(cand[-1]) + 5]
        for T in picks:
            o = oracle.dp_at(inst, T)
            g = rec(tg.tg_dp_at(h, T))
            same(o, g, f"{inst.name} T={T}")
        h.destroy()


def test_mid_size_scaled_configs(tg):
    """Scaled-down twins of configs 3-5 that the oracle still solves in seconds: several tiles per
    level, ragged last tile, L not a multiple of 4."""
    insts = [gen.config3(0, L=30, K=8), gen.config4(0, L=22, K=9), gen.config5_one(3, L=26, K=7),
             gen.config3(1, L=37, K=6), gen.config5_one(4, L=17, K=8)]
    for inst, g in zip(insts, solve_all(tg, insts)):
        same(oracle.solve(inst, n_threads=8), g, inst.name)


def test_extreme_shapes(tg):
    """Limits of the ABI: L = 1, L = 255 (TG_MAX_L), K = 16 (TG_MAX_K) with a tiny L, P = 255, m = 1 and
    m = 2^20, nothing feasible, only the whole-model slice feasible."""
    import numpy as np
    insts = []
    a = gen.random_small(1, Lmax=1, Kmax=1, Pmax=1); insts.append(a)
    b = gen.random_small(2, Lmax=6, Kmax=3, Pmax=2); b.m = 1 << 20; insts.append(b)
    c = gen.random_small(3, Lmax=6, Kmax=3, Pmax=2); c.m = 1; insts.append(c)
    d = gen.random_small(4, Lmax=6, Kmax=3, Pmax=2); d.time_us[:] = 0x7FFFFFFF; insts.append(d)
    e = gen.config3(0, L=6, K=3)   # only the whole model on island 1 is feasible
    keep = e.time_us[gen.slice_index(6, 0, 6), 1, :].copy()
    e.time_us[:] = 0x7FFFFFFF; e.time_us[gen.slice_index(6, 0, 6), 1, :] = keep; insts.append(e)
    insts.append(gen.config4(0, L=3, K=16))                       # 65536 masks, L not a multiple of 4
    for L, K, P in [(255, 2, 1), (5, 3, 255)]:                     # TG_MAX_L, TG_MAX_P
        NS = L * (L + 1) // 2
        idx = np.arange(NS * K * P).reshape(NS, K, P)
        aa, bb = gen.slice_bounds(L)
        t = ((bb - aa)[:, None, None] * gen.urand(9, 1, idx, 100, 900)).astype(np.int32)
        mm = gen.urand(9, 2, idx, 1, 50).astype(np.int32)
        insts.append(gen.Instance(f"L{L}K{K}P{P}", L, K, P, 4, t, mm, np.ones(K, np.int32), np.full(K, 25, np.int32),
                                  np.full((K, K), 50, np.int32), 32))
    for inst, g in zip(insts, solve_all(tg, insts)):
        same(oracle.solve(inst, n_threads=8), g, inst.name)
    for inst, g in zip(insts, solve_all(tg, insts, flags=1)):
        same(oracle.solve(inst, n_threads=8), g, inst.name + " full sweep")


@pytest.mark.parametrize("style", ["ties", "mixed", "tightmem"])
def test_threshold_search_stress(tg, style):
    """Branch-and-bound threshold search against the oracle's sweep on mid-size instances with every m,
    heavy ties and binding memory; teams and solo mode (one batch of 60, then each alone)."""
    insts = [gen.random_small(s + 20_000, Lmax=20, Kmax=8, Pmax=3, style=style) for s in range(60)]
    want = [oracle.solve(i, n_threads=8) for i in insts]
    for inst, o, g in zip(insts, want, solve_all(tg, insts)):
        same(o, g, inst.name)
    for inst, o in list(zip(insts, want))[:12]:
        same(o, solve_all(tg, [inst])[0], inst.name + " alone")


def test_more_instances_than_items_per_round(tg):
    """9000 instances in one call: more active instances than the scheduler's 8192 items per round."""
    insts = [gen.random_small(s + 40_000, Lmax=5, Kmax=3, Pmax=2, style=STYLES[s % 5]) for s in range(9000)]
    res = solve_all(tg, insts)
    for inst, g in zip(insts, res):
        same(oracle.solve(inst), g, inst.name)


def test_create_batch(tg):
    """tg_instance_create_batch == one tg_instance_create per instance; a bad table anywhere creates nothing."""
    insts = [gen.random_small(s + 95_000, Lmax=8, Kmax=5, Pmax=3, style=STYLES[s % 5]) for s in range(64)] + \
            [gen.config2(), gen.config3(0, L=20, K=6)]
    spec = lambda i: (i.L, i.K, i.P, i.m, i.time_us, i.mem_mb, i.island_gpus, i.island_cap_mb, i.bw_gbps, i.act_mb)
    hs = tg.tg_instance_create_batch([spec(i) for i in insts])
    assert len(hs) == len(insts) and all(h.handle for h in hs)
    res = tg.tg_solve_batch(hs)
    for inst, g in zip(insts, res):
        same(oracle.solve(inst), g, inst.name)
    for h in hs:
        h.destroy()
    assert tg.tg_instance_create_batch([]) == []
    bad = insts[5].copy()
    bad.time_us = bad.time_us.copy()
    bad.time_us[0, 0, 0] = -7
    with pytest.raises(tg.TangramError) as e:
        tg.tg_instance_create_batch([spec(i) for i in insts[:5]] + [spec(bad)] + [spec(i) for i in insts[6:9]])
    assert e.value.status == 3 and "instance 5" in str(e.value)
    shape = list(spec(insts[0]))
    shape[1] = 17                                  # K above TG_MAX_K
    with pytest.raises(tg.TangramError) as e:
        tg.tg_instance_create_batch([spec(insts[1]), tuple(shape)])
    assert e.value.status == 2 and "instance 1" in str(e.value)


def test_large_stage_times(tg):
    """Stage times up to TG_TIME_MAX = 2^25 us: candidate extraction leaves the shared-memory bitmap (keys < 2^20) for
    the radix sort; times just below and above the switch, and the largest allowed value."""
    insts = []
    for seed, scale in [(0, 10), (1, 300), (2, 3000)]:
        i = gen.config3(seed, L=14, K=5)
        valid = i.time_us != 0x7FFFFFFF
        i.time_us = np.where(valid, np.minimum(i.time_us.astype(np.int64) * scale, 1 << 25), 0x7FFFFFFF).astype(np.int32)
        i.name += f"_x{scale}"
        insts.append(i)
    j = gen.random_small(11, Lmax=6, Kmax=3, Pmax=2)
    j.time_us = np.where(j.time_us != 0x7FFFFFFF, (1 << 25) - (j.time_us % 7), 0x7FFFFFFF).astype(np.int32)
    insts.append(j)
    assert max(int(i.time_us[i.time_us != 0x7FFFFFFF].max()) for i in insts[:1]) < (1 << 20) <= \
        min(int(i.time_us[i.time_us != 0x7FFFFFFF].max()) for i in insts[1:])
    for inst, g in zip(insts, solve_all(tg, insts)):
        same(oracle.solve(inst), g, inst.name)
    for inst in insts:
        h = tg.instance_from_inputs(inst)
        cand = tg.tg_reduce(h)[3]
        assert np.array_equal(cand.astype(np.int64), oracle.reduce(inst)[3]), inst.name
        h.destroy()


@pytest.mark.parametrize("n", [1, 2, 4, 5, 8, 9, 63, 64, 65, 147, 148, 149, 300, 1024, 1025])
def test_batch_sizes_around_the_scheduling_modes(tg, n):
    """1-4 instances: every probe of the last round back-tracks; <= 8: a warp lays out an instance's probes; < 64: one thread
    per instance on CTA 0; 64..1024: queue mode (no rounds after the first); above: wide scheduling in rounds; items below /
    at / above the number of slots: team mode vs solo mode."""
    insts = [gen.random_small(s + 99_000 + 1000 * n, Lmax=8, Kmax=5, Pmax=3, style=STYLES[s % 5]) for s in range(n)]
    for inst, g in zip(insts, solve_all(tg, insts)):
        same(oracle.solve(inst), g, inst.name)


def test_loader_paths_in_one_batch(tg):
    """Cost-table loader: batches large enough for the many-cells-per-thread mode whose
    instances take every path of the kernel -- batched loads for P = 4 and P = 8, the cell-at-a-time path for
    another P, for a footprint table, and for an instance whose P differs from the first one's; chunk tails that
    end inside a row of the slice triangle."""
    p8 = [gen.config3(s, L=17 + s % 5, K=4 + s % 3) for s in range(150)]                      # P = 8 first
    p4 = [gen.config5_one(s, L=14 + s % 7, K=5 + s % 2) for s in range(150)]                  # P = 4 first
    odd = [gen.random_small(s + 12_000, Lmax=9, Kmax=6, Pmax=7, style=STYLES[s % 5]) for s in range(40)]
    foot = [gen.with_actmem(gen.config3(s, L=15, K=4), s, 500, 6000) for s in range(10)]
    for batch in (p8 + odd + p4[:20] + foot, p4 + odd + p8[:20] + foot, odd + p4 + p8):
        for inst, g in zip(batch, solve_all(tg, batch)):
            same(oracle.solve_depth(inst) if inst.actmem_mb is not None else oracle.solve(inst), g, inst.name)


@pytest.mark.parametrize("shape,P", [("config4", 8), ("config5_one", 4)])
def test_row_group_loader_on_uniform_batches(tg, shape, P):
    """Cost-table loader, the row-group form (tgLoadRowsKernel: a CTA reduces 8 start rows and writes the diagonal-major
    tables through a shared-memory tile): taken by a batch of plain instances of one P in {4, 8} that fills the GPU -- what
    the 1024-instance batch runs with P = 4.  Here 320 instances each of P = 8 and P = 4 with L = 11 ... 16, so the last row
    group of an instance is partial and instances of different L share one grid."""
    insts = [getattr(gen, shape)(s + 300, L=11 + s % 6, K=5 + s % 4) for s in range(320)]
    assert all(x.P == P for x in insts)
    for inst, g in zip(insts, solve_all(tg, insts)):
        same(oracle.solve(inst), g, inst.name)


def test_statistics_on_the_device_match_the_host_form(tg):
    """tg_solve_stats written to a DEVICE buffer (the call stays asynchronous; bench.py times it that way) against the HOST
    form of the same solve: a few instances run in rounds, so every count is deterministic."""
    import torch
    insts = [gen.config2(), gen.config3(0, L=20, K=5), gen.random_small(77, Lmax=9, Kmax=5, Pmax=3, style="ties")]
    hs = [tg.instance_from_inputs(i) for i in insts]
    host = tg.TgSolveStats()
    want = tg.tg_solve_batch(hs, stats=host)
    out = torch.empty(len(hs) * tg.RESULT_BYTES, dtype=torch.uint8, device="cuda")
    dev = torch.zeros(256, dtype=torch.uint8, device="cuda")
    tg.tg_solve_batch(hs, out=out, stats=dev)
    torch.cuda.synchronize()
    got = tg.stats_from_tensor(dev)
    for f in ("n_dp", "plans_dense", "states_live", "n_rounds", "error_flag", "relax_admissible", "states_windowed"):
        assert getattr(got, f) == getattr(host, f), f
    assert host.n_dp > 0 and host.error_flag == 0
    res = tg.results_from_tensor(out, len(hs))
    for inst, a, b in zip(insts, want, res):
        assert int(a["iter_time_us"]) == int(b["iter_time_us"]) and int(a["island_mask"]) == int(b["island_mask"])
        same(oracle.solve(inst), b, inst.name)
    for h in hs:
        h.destroy()
