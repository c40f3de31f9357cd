"""tg_prune_batch_static: the pruning pass with its scratch in a file-scope device array of the library (no device
allocation in the call) against tg_prune_batch, the existing path -- per-rule counts and pruned tables bit-exact (integer
work), two calls in a row on the shared scratch, and the size limit.  Collected last on purpose (file name)."""
import numpy as np
import pytest

import tg_inputs as gen

pytestmark = pytest.mark.gpu

STYLES = ["mixed", "ties", "tightmem", "asym", "sparse"]


@pytest.fixture(scope="module")
def tg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_16907_b200 as tg
    tg.lib()
    return tg


def batch(seed0, n, with_footprint=False):
    out = [gen.random_small(seed0 + s, Lmax=9, Kmax=6, Pmax=7, style=STYLES[s % 5]) for s in range(n)]
    out += [gen.config1(0, 10), gen.config2(), gen.config3(0, L=21, K=5), gen.config4(0, L=18, K=6)]
    if with_footprint:
        out = [gen.with_actmem(x, i) for i, x in enumerate(out)]
    return out


def both(tg, insts, mode, thr):
    """(counts, tables) of the existing path and of the static-scratch path on two uploads of the same instances."""
    ha = [tg.instance_from_inputs(i) for i in insts]
    hb = [tg.instance_from_inputs(i) for i in insts]
    ca = tg.tg_prune_batch(ha, mode, thr)
    cb = tg.tg_prune_batch_static(hb, mode, thr)
    ta = [tg.tg_instance_read_time(h) for h in ha]
    tb = [tg.tg_instance_read_time(h) for h in hb]
    for h in ha + hb:
        h.destroy()
    return ca, cb, ta, tb


def test_static_scratch_matches_existing_path_two_calls_in_a_row(tg):
    # call 1 leaves its counters, caps and descriptors in the shared array; call 2 is a different batch (other sizes,
    # another mode) and must not see them
    plan = [(batch(9100, 40), 1, 1500), (batch(9200, 25, with_footprint=True), 0, 0), (batch(9300, 33), 2, 700),
            (batch(9100, 40), 1, 1500)]
    killed = 0
    for insts, mode, thr in plan:
        ca, cb, ta, tb = both(tg, insts, mode, thr)
        assert ca.shape == cb.shape == (len(insts), 4)
        assert np.array_equal(ca, cb), (mode, thr)
        for x, a, b in zip(insts, ta, tb):
            assert np.array_equal(a, b), (x.name, mode, thr)
        killed += int(cb.sum())
    assert killed > 0


def test_static_scratch_same_handles_twice(tg):
    # two calls in a row on the SAME instances: EXACT is idempotent, so the second call must count nothing
    insts = batch(9400, 30)
    hs = [tg.instance_from_inputs(i) for i in insts]
    ref = [tg.instance_from_inputs(i) for i in insts]
    first = tg.tg_prune_batch_static(hs, tg.TG_PRUNE_EXACT, 0)
    second = tg.tg_prune_batch_static(hs, tg.TG_PRUNE_EXACT, 0)
    want = tg.tg_prune_batch(ref, tg.TG_PRUNE_EXACT, 0)
    assert np.array_equal(first, want) and first.sum() > 0
    assert not second.any()
    for a, b in zip(hs, ref):
        assert np.array_equal(tg.tg_instance_read_time(a), tg.tg_instance_read_time(b))
        a.destroy(); b.destroy()


def test_static_scratch_limits(tg):
    assert tg.TG_PRUNE_STATIC_MAX_N == 1024
    one = gen.config1()
    hs = [tg.instance_from_inputs(one) for _ in range(tg.TG_PRUNE_STATIC_MAX_N + 1)]
    with pytest.raises(tg.TangramError) as ei:
        tg.tg_prune_batch_static(hs, tg.TG_PRUNE_EXACT, 0)
    assert "TG_PRUNE_STATIC_MAX_N" in str(ei.value)
    full = tg.tg_prune_batch_static(hs[:-1], tg.TG_PRUNE_EXACT, 0)          # exactly the maximum fits
    ref = tg.instance_from_inputs(one)
    assert np.array_equal(full, np.tile(tg.tg_prune(ref, tg.TG_PRUNE_EXACT, 0), (tg.TG_PRUNE_STATIC_MAX_N, 1)))
    assert tg.tg_prune_batch_static([], tg.TG_PRUNE_EXACT, 0).shape == (0, 4)
    with pytest.raises(tg.TangramError):
        tg.tg_prune_batch_static([hs[0], hs[0]], tg.TG_PRUNE_EXACT, 0)     # listed twice
    ref.destroy()
    for h in hs:
        h.destroy()
