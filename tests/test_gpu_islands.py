"""GPU parity of SURVEY.md §8(f) NEXT-4 (tg_islands_build) against the island oracle, exact on the
partition, the island attributes and the bandwidth matrix; the islands feed tg_instance_create."""
import numpy as np
import pytest

import oracle
import tg_inputs as gen

pytestmark = pytest.mark.gpu
EPS = (100, 50, 100)


@pytest.fixture(scope="module")
def tg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_16907_b200 as tg
    tg.lib()
    return tg


def same(tg, prof, eps):
    got = tg.tg_islands_build(*prof, *eps)
    want = oracle.islands(*prof, *eps)
    for g, w in zip(got, want):
        assert np.array_equal(g, w)
    return got


def test_table_3_clusters_and_random_clusters(tg):
    for name, k in (("C1", 2), ("C2", 2), ("C3", 4)):
        assert same(tg, gen.cluster_profile(name), EPS)[1].size == k
    for seed in range(400):
        same(tg, gen.random_cluster(seed, nmax=12 + (seed % 4) * 8), (EPS, (0, 0, 0), (1000, 1000, 1000))[seed % 3])


def test_largest_cluster_and_errors(tg):
    n = 64
    idx = np.arange(n)
    prof = ((4 + 4 * (idx % 2)).astype(np.int32), (100 + idx % 3).astype(np.int32), np.full(n, 80000, np.int32),
            np.full(n, 600, np.int32), (50 + gen.urand(1, 3, idx[:, None] * n + idx[None, :], 0, 60)).astype(np.int32))
    same(tg, prof, EPS)
    with pytest.raises(tg.TangramError) as e:
        tg.tg_islands_build(*(np.concatenate([a, a[:1]]) for a in prof[:4]), np.ones((65, 65), np.int32), *EPS)
    assert e.value.status == 2
    bad = prof[4].copy()
    bad[0, 1] = 0
    with pytest.raises(tg.TangramError) as e:
        tg.tg_islands_build(*prof[:4], bad, *EPS)
    assert e.value.status == 3


def test_islands_feed_the_composition_search(tg):
    """C3 -> 4 islands -> a planning instance on them (synthetic cost tables) -> same result as the oracle."""
    of, ig, ic, bw = tg.tg_islands_build(*gen.cluster_profile("C3"), *EPS)
    base = next(b for b in (gen.random_small(s, Lmax=8, Kmax=4, Pmax=3, style="mixed") for s in range(77, 400)) if b.K == ig.size)
    inst = base.copy()
    inst.island_gpus, inst.bw_gbps = ig.astype(np.int32), bw.astype(np.int32)
    h = tg.instance_from_inputs(inst)
    g = tg.tg_solve_batch([h])[0]
    o = oracle.solve(inst)
    assert (o.iter_time_us, o.sum_us, o.bottleneck_us, o.island_mask) == \
           (int(g["iter_time_us"]), int(g["sum_us"]), int(g["bottleneck_us"]), int(g["island_mask"]))
    h.destroy()
