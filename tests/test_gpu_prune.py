"""GPU parity of tg_prune (rules R1-R4) against oracle.prune: the pruned time
table and the per-rule counts, bit-exact; and solve(prune(x)) on the device against the oracle."""
import numpy as np
import pytest

import oracle
import tg_inputs as gen
from test_gpu_parity import same, solve_all, STYLES

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_16907_b200 as tg
    tg.lib()
    return tg


def cases():
    out = [gen.random_small(s + 8000, Lmax=9, Kmax=6, Pmax=7, style=STYLES[s % 5]) for s in range(60)]
    out += [gen.config1(), gen.config1(0, 10), gen.config2(), gen.config3(0, L=21, K=5), gen.config4(0, L=18, K=6)]
    return out


@pytest.mark.parametrize("mode,thr", [(0, 0), (1, 16384), (1, 3000), (1, 1500), (1, 1000), (2, 0), (2, 700), (2, 5000), (2, 1 << 25)])
def test_prune_table_and_counts(tg, mode, thr):
    for inst in cases():
        h = tg.instance_from_inputs(inst)
        counts = tg.tg_prune(h, mode, thr)
        t = tg.tg_instance_read_time(h)
        pr, ocounts = oracle.prune(inst, mode, thr)
        assert counts.tolist() == ocounts.tolist(), (inst.name, mode, thr)
        assert np.array_equal(t, pr.time_us.reshape(t.shape)), (inst.name, mode, thr)
        again = tg.tg_prune(h, mode, thr)                       # monotone; idempotent except R3, which
        pr2, ocounts2 = oracle.prune(pr, mode, thr)             # re-profiles the live table (DESIGN.md R-r3)
        assert again.tolist() == ocounts2.tolist()
        if mode != 1:
            assert again.tolist() == [0, 0, 0, 0]
        t2 = tg.tg_instance_read_time(h)
        assert np.array_equal(t2, pr2.time_us.reshape(t.shape)) and ((t == 0x7FFFFFFF) <= (t2 == 0x7FFFFFFF)).all()
        pr = pr2
        g = tg.tg_solve_batch([h])[0]                           # the pruned instance solves like the oracle's
        same(oracle.solve(pr), g, inst.name)
        h.destroy()


def cases_with_footprint():
    out = [gen.with_actmem(gen.random_small(s + 8500, Lmax=9, Kmax=6, Pmax=7, style=STYLES[s % 5]), s) for s in range(60)]
    out += [gen.with_actmem(gen.random_small(s + 8600, Lmax=6, Kmax=3, Pmax=40, style=STYLES[s % 5]), s) for s in range(5)]
    out += [gen.with_actmem(gen.config1(0, 10), 1, 0, 300), gen.with_actmem(gen.config2(), 4, 0, 2000),
            gen.with_actmem(gen.config3(0, L=21, K=5), 1, 500, 6000), gen.with_actmem(gen.config4(0, L=18, K=6), 2, 2000, 20000)]
    return out


@pytest.mark.parametrize("mode,thr", [(0, 0), (1, 3000), (1, 1000), (2, 700), (2, 1 << 25)])
def test_prune_with_footprint_table_and_counts(tg, mode, thr):
    """R1 at depth 1 and 3-way R2 (oracle.prune_depth); the pruned instance solves like the
    depth oracle on the oracle's pruned tables; removing the footprint afterwards leaves the core rules."""
    killed3 = 0
    for inst in cases_with_footprint():
        h = tg.instance_from_inputs(inst)
        counts = tg.tg_prune(h, mode, thr)
        t = tg.tg_instance_read_time(h)
        pr, ocounts = oracle.prune_depth(inst, mode, thr)
        assert counts.tolist() == ocounts.tolist(), (inst.name, mode, thr)
        assert np.array_equal(t, pr.time_us.reshape(t.shape)), (inst.name, mode, thr)
        killed3 += int(ocounts[0] + ocounts[1])
        same(oracle.solve_depth(pr), tg.tg_solve_batch([h])[0], inst.name)
        again = tg.tg_prune(h, mode, thr)
        pr2, ocounts2 = oracle.prune_depth(pr, mode, thr)
        assert again.tolist() == ocounts2.tolist()
        assert np.array_equal(tg.tg_instance_read_time(h), pr2.time_us.reshape(t.shape))
        tg.tg_instance_set_actmem(h, None)                      # footprint removed: the two-axis rules apply again
        core = pr2.copy(); core.actmem_mb = None
        after = tg.tg_prune(h, 0, 0)
        pr3, ocounts3 = oracle.prune(core, 0, 0)
        assert after.tolist() == ocounts3.tolist()
        assert np.array_equal(tg.tg_instance_read_time(h), pr3.time_us.reshape(t.shape))
        h.destroy()
    assert killed3 > 100


@pytest.mark.parametrize("mode,thr", [(0, 0), (1, 3000), (1, 1000), (2, 700), (2, 1 << 25)])
def test_prune_batch_equals_single_calls(tg, mode, thr):
    """tg_prune_batch: instances of every shape, with and without a footprint table, in one pass; row i of the counts
    and the tables as after tg_prune on instance i (oracle.prune / oracle.prune_depth); then the pruned batch solves
    like the oracle on the oracle's pruned tables."""
    insts = cases() + cases_with_footprint()
    hs = [tg.instance_from_inputs(i) for i in insts]
    counts = tg.tg_prune_batch(hs, mode, thr)
    assert counts.shape == (len(insts), 4)
    pruned = []
    for inst, h, c in zip(insts, hs, counts):
        pr, oc = (oracle.prune_depth if inst.actmem_mb is not None else oracle.prune)(inst, mode, thr)
        assert c.tolist() == oc.tolist(), (inst.name, mode, thr)
        t = tg.tg_instance_read_time(h)
        assert np.array_equal(t, pr.time_us.reshape(t.shape)), (inst.name, mode, thr)
        pruned.append(pr)
    for pr, g in zip(pruned, tg.tg_solve_batch(hs)):
        same(oracle.solve_depth(pr) if pr.actmem_mb is not None else oracle.solve(pr), g, pr.name)
    if mode != 1:                                               # idempotent (R3 re-profiles: DESIGN.md R-r3)
        assert not tg.tg_prune_batch(hs, mode, thr).any()
    assert tg.tg_prune_batch([], mode, thr).shape == (0, 4)
    with pytest.raises(tg.TangramError) as e:                   # the same instance twice
        tg.tg_prune_batch([hs[0], hs[1], hs[0]], mode, thr)
    assert e.value.status == 3
    for h in hs:
        h.destroy()


def test_prune_errors(tg):
    h = tg.instance_from_inputs(gen.config1())
    for mode, thr in [(3, 0), (1, 999), (1, 16385), (2, -1)]:
        with pytest.raises(tg.TangramError) as e:
            tg.tg_prune(h, mode, thr)
        assert e.value.status == 3
        with pytest.raises(tg.TangramError) as e:
            tg.tg_prune_batch([h], mode, thr)
        assert e.value.status == 3
    h.destroy()


def test_create_rejects_bad_tables(tg):
    inst = gen.config1()
    bad = inst.copy(); bad.time_us[3, 1, 0] = -5
    with pytest.raises(tg.TangramError) as e:
        tg.instance_from_inputs(bad)
    assert e.value.status == 3
    bad = inst.copy(); bad.time_us[3, 1, 0] = (1 << 25) + 1
    with pytest.raises(tg.TangramError):
        tg.instance_from_inputs(bad)
    bad = inst.copy(); bad.mem_mb[0, 0, 0] = -1
    with pytest.raises(tg.TangramError):
        tg.instance_from_inputs(bad)
    bad = inst.copy(); bad.bw_gbps[0, 1] = 0
    with pytest.raises(tg.TangramError):
        tg.instance_from_inputs(bad)
    bad = inst.copy(); bad.island_gpus[2] = 0
    with pytest.raises(tg.TangramError):
        tg.instance_from_inputs(bad)
    ok = inst.copy(); ok.time_us[:] = 0x7FFFFFFF                # nothing feasible is not an error
    g = solve_all(tg, [ok])[0]
    assert int(g["iter_time_us"]) == (1 << 63) - 1 and int(g["n_stages"]) == 0


def test_device_resident_tables_and_async_out(tg):
    """EITHER pointers: device tables in, device results out on a side stream."""
    import torch
    insts = [gen.config2(s) for s in range(3)]
    hs = [tg.instance_from_inputs(i, device_tables=True) for i in insts]
    st = torch.cuda.Stream()
    out = torch.empty(len(hs) * tg.RESULT_BYTES, dtype=torch.uint8, device="cuda")
    with torch.cuda.stream(st):
        tg.tg_solve_batch(hs, out=out, stream=st)
    st.synchronize()
    for inst, g in zip(insts, tg.results_from_tensor(out, len(hs))):
        same(oracle.solve(inst), g, inst.name)
    for h in hs:
        h.destroy()


@pytest.mark.parametrize("shape,L,K,n,footprint", [("config5_one", 12, 10, 200, False), ("config4", 12, 8, 220, False),
                                                     ("config5_one", 12, 10, 200, True), ("config4", 12, 8, 220, True)])
def test_prune_batch_that_fills_the_gpu(tg, shape, L, K, n, footprint):
    """The launch the 1024-instance batch takes: a batch with at least 4 CTAs per SM (here 200 x 4 and 220 x 3 CTAs of 4 and 2
    cells a thread on 148 SMs) is pruned from registers, several cells of a thread in flight (P = 4 and P = 8, with and
    without the footprint axis); the smaller batches above take one cell per thread.  Tables and counts against the oracle."""
    insts = [getattr(gen, shape)(5000 + s, L=L, K=K) for s in range(n)]
    if footprint:
        insts = [gen.with_actmem(x, s) for s, x in enumerate(insts)]
    assert insts[0].P == (4 if shape == "config5_one" else 8)
    orc = oracle.prune_depth if footprint else oracle.prune
    killed = 0
    for mode, thr in [(0, 0), (1, 3000)]:
        hs = [tg.instance_from_inputs(i) for i in insts]
        counts = tg.tg_prune_batch(hs, mode, thr)
        for inst, h, c in zip(insts, hs, counts):
            pr, oc = orc(inst, mode, thr)
            assert c.tolist() == oc.tolist(), (inst.name, mode, thr)
            t = tg.tg_instance_read_time(h)
            assert np.array_equal(t, pr.time_us.reshape(t.shape)), (inst.name, mode, thr)
            killed += int(oc[0] + oc[1])
        for h in hs:
            h.destroy()
    assert killed > 1000
