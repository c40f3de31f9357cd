"""Pins for the oracle other than brute force: closed forms, special cases that reduce to textbook
results, invariants (SURVEY.md §8(c) "what pins each part"; test pins P-single, P-drop, P-balance,
P-cover of SURVEY.md §4).  None of these re-types the oracle's recurrence."""
import numpy as np
import pytest

import oracle
import tg_inputs as gen
from conftest import rescore

INVALID = 0x7FFFFFFF
STYLES = ["mixed", "ties", "tightmem", "asym", "sparse"]


def mk(L, K, P, m, time, mem=None, cap=None, bw=None, act=0, gpus=None):
    NS = L * (L + 1) // 2
    time = np.asarray(time, dtype=np.int32).reshape(NS, K, P)
    mem = np.zeros((NS, K, P), np.int32) if mem is None else np.asarray(mem, np.int32).reshape(NS, K, P)
    cap = np.full(K, 1000, np.int32) if cap is None else np.asarray(cap, np.int32)
    bw = np.full((K, K), 100, np.int32) if bw is None else np.asarray(bw, np.int32)
    gpus = np.ones(K, np.int32) if gpus is None else np.asarray(gpus, np.int32)
    return gen.Instance("hand", L, K, P, m, time, mem, gpus, cap, bw, act)


def linear_instance(L, K, u, m, act=0):
    """identical islands, t([a,b)) = (b-a)*u, one plan, no memory pressure"""
    a, b = gen.slice_bounds(L)
    t = np.repeat(((b - a) * u)[:, None, None], K, axis=1)
    return mk(L, K, 1, m, t, act=act)


# ---- K = 1: reproduces the parallelizer's own plan (pin P-single) -----------------
@pytest.mark.parametrize("seed", range(40))
def test_single_island_closed_form(seed):
    inst = gen.random_small(seed, Lmax=9, Kmax=1, Pmax=4, style=STYLES[seed % 5])
    assert inst.K == 1
    whole = inst.time_us[gen.slice_index(inst.L, 0, inst.L), 0, :].astype(np.int64)
    memw = inst.mem_mb[gen.slice_index(inst.L, 0, inst.L), 0, :]
    ok = (whole != INVALID) & (memw <= inst.island_cap_mb[0])
    r = oracle.solve(inst)
    if not ok.any():
        assert not r.feasible
        return
    best = whole[ok].min()
    p = int(np.nonzero(ok & (whole == best))[0][0])
    assert r.iter_time_us == inst.m * best
    assert r.stages == [(0, 0, p)] and r.island_mask == 1 and r.bottleneck_us == best


# ---- m = 1: plain shortest path; the sweep must return the SMALLEST T attaining it ----------------------
@pytest.mark.parametrize("seed", range(60))
def test_m1_equals_f_inf_and_smallest_T(seed):
    inst = gen.random_small(seed + 300, Lmax=7, Kmax=4, Pmax=2, style=STYLES[seed % 5])
    inst.m = 1
    r = oracle.solve(inst)
    finf = oracle.dp_at(inst, -1, want_plan=False)
    assert r.feasible == finf.feasible
    if not r.feasible:
        return
    assert r.iter_time_us == finf.sum_us == r.sum_us
    _, _, _, cand = oracle.reduce(inst)
    lower = [int(T) for T in cand if T < r.bottleneck_us]
    for T in lower[-3:]:                      # no smaller candidate attains f_inf
        q = oracle.dp_at(inst, T, want_plan=False)
        assert (not q.feasible) or q.sum_us > finf.sum_us


# ---- identical islands, linear times, x = 0: iter = L*u + (m-1)*ceil(L/n)*u, n = min(K, L) ----------------
@pytest.mark.parametrize("L,K,u,m", [(8, 3, 10, 8), (7, 4, 3, 5), (5, 5, 7, 64), (4, 6, 11, 2), (9, 2, 1, 16), (6, 1, 5, 9)])
def test_identical_islands_closed_form(L, K, u, m):
    r = oracle.solve(linear_instance(L, K, u, m))
    n = min(K, L)
    assert r.iter_time_us == L * u + (m - 1) * (-(-L // n)) * u
    assert r.sum_us == L * u
    # lowest-mask tie-break: the n lowest islands ... or fewer if a shallower pipeline ties
    assert r.island_mask == (1 << r.n_stages) - 1


# ---- all x equal: the boundary lane is redundant, lane-less (a,S) recurrence gives the optimum ------------
@pytest.mark.parametrize("seed", range(60))
def test_equal_transfers_match_laneless_recurrence(seed):
    inst = gen.random_small(seed + 700, Lmax=7, Kmax=5, Pmax=3, style=STYLES[seed % 5])
    bwv = 1 + seed % 7
    inst.bw_gbps = np.full((inst.K, inst.K), bwv, np.int32)
    xc = -((-inst.act_mb * 1000) // bwv)
    r = oracle.solve(inst)
    ll = oracle.laneless_iter(inst, xc)
    assert (r.iter_time_us if r.feasible else oracle.INT64_MAX) == ll


# ---- transfer table: 64 MB at 25/100/400 GB/s -> 2560/640/160 us ---------------------------
def test_transfer_units():
    inst = gen.config1()
    _, _, x, _ = oracle.reduce(inst)
    assert x.tolist() == [[0, 2560, 640], [2560, 0, 160], [640, 160, 0]]
    inst.act_mb = 1
    inst.bw_gbps = np.array([[1, 3, 7], [1000, 1, 999], [1001, 333, 1]], np.int32)
    _, _, x, _ = oracle.reduce(inst)
    assert x.tolist() == [[0, 334, 143], [1, 0, 2], [1, 4, 0]]     # integer ceil, directional


# ---- hand-worked two-island instance with a directional link (catches a transposed x) -------------------
def test_hand_worked_direction_of_transfer():
    # L=2, K=2, P=1.  slices: s0=[0,1) s1=[0,2) s2=[1,2).  island0: 10,100,10 ; island1: 10,100,10
    t = [[10, 10], [100, 100], [10, 10]]
    bw = [[1, 1000], [1, 1]]          # 0 -> 1 fast (1 us per MB*1000/1000), 1 -> 0 slow
    inst = mk(2, 2, 1, 1, t, bw=bw, act=1)
    r = oracle.solve(inst)
    # plans: (k0=0,k1=1): 10+10+x[0][1]=1 -> 21 ; (1,0): 10+10+1000 = 1020 ; single stage: 100
    assert (r.iter_time_us, r.stages) == (21, [(0, 0, 0), (1, 1, 0)])
    inst.bw_gbps = np.array(bw, np.int32).T.copy()
    r = oracle.solve(inst)
    assert (r.iter_time_us, r.stages) == (21, [(0, 1, 0), (1, 0, 0)])


# ---- invariants (north_star; SURVEY.md §4 pins P-drop, P-balance, P-cover) -----------------------------------
def _add_island(inst, seed, useless=False):
    """append one island (new highest label)"""
    o = inst.copy()
    NS, K, P = inst.time_us.shape
    idx = np.arange(NS * P).reshape(NS, 1, P)
    a, b = gen.slice_bounds(inst.L)
    if useless:
        t = np.full((NS, 1, P), INVALID, np.int64)
    else:
        t = (b - a)[:, None, None] * gen.urand(seed, 77, idx, 50, 1500)
    o.time_us = np.concatenate([inst.time_us, t.astype(np.int32)], axis=1)
    o.mem_mb = np.concatenate([inst.mem_mb, np.zeros((NS, 1, P), np.int32)], axis=1)
    o.island_gpus = np.append(inst.island_gpus, 1).astype(np.int32)
    o.island_cap_mb = np.append(inst.island_cap_mb, 10 ** 6).astype(np.int32)
    bw = np.full((K + 1, K + 1), 13, np.int32)
    bw[:K, :K] = inst.bw_gbps
    o.bw_gbps = bw
    o.K = K + 1
    return o


@pytest.mark.parametrize("seed", range(80))
def test_adding_an_island_never_worsens(seed):
    inst = gen.random_small(seed + 1200, Lmax=7, Kmax=4, Pmax=2, style=STYLES[seed % 5])
    r0 = oracle.solve(inst)
    r1 = oracle.solve(_add_island(inst, seed))
    if r0.feasible:
        assert r1.feasible and r1.iter_time_us <= r0.iter_time_us
    # a useless island (eliminated) changes neither value nor plan
    r2 = oracle.solve(_add_island(inst, seed, useless=True))
    assert r2.plan_key() == r0.plan_key()


@pytest.mark.parametrize("seed", range(60))
def test_relabelling_islands_keeps_the_optimum(seed):
    inst = gen.random_small(seed + 2000, Lmax=7, Kmax=5, Pmax=2, style=STYLES[seed % 5])
    perm = np.argsort(gen.mix64(seed, 99, np.arange(inst.K)))       # new label i = old island perm[i]
    o = inst.copy()
    o.time_us = inst.time_us[:, perm, :].copy()
    o.mem_mb = inst.mem_mb[:, perm, :].copy()
    o.island_cap_mb = inst.island_cap_mb[perm].copy()
    o.island_gpus = inst.island_gpus[perm].copy()
    o.bw_gbps = inst.bw_gbps[np.ix_(perm, perm)].copy()
    r0, r1 = oracle.solve(inst), oracle.solve(o)
    assert r0.feasible == r1.feasible
    if r0.feasible:
        assert (r0.iter_time_us, r0.bottleneck_us) == (r1.iter_time_us, r1.bottleneck_us)
        # the permuted plan is a valid plan of the original instance with the same score
        back = [(a, int(perm[k]), p) for a, k, p in r1.stages]
        s, T, it, _ = rescore(inst, back)
        assert (it, T) == (r0.iter_time_us, r0.bottleneck_us)


def test_permuting_identical_islands_changes_nothing():
    inst = gen.random_small(31, Lmax=7, Kmax=4, Pmax=2, style="mixed")
    inst = _add_island(inst, 5)
    K = inst.K
    # make islands K-1 and 0 identical twins, symmetric links
    inst.time_us[:, K - 1, :] = inst.time_us[:, 0, :]
    inst.mem_mb[:, K - 1, :] = inst.mem_mb[:, 0, :]
    inst.island_cap_mb[K - 1] = inst.island_cap_mb[0]
    inst.bw_gbps = np.minimum(inst.bw_gbps, inst.bw_gbps.T)
    inst.bw_gbps[K - 1, :] = inst.bw_gbps[0, :]; inst.bw_gbps[:, K - 1] = inst.bw_gbps[:, 0]
    o = inst.copy()
    sw = list(range(K)); sw[0], sw[K - 1] = K - 1, 0
    o.time_us = inst.time_us[:, sw, :].copy(); o.mem_mb = inst.mem_mb[:, sw, :].copy()
    o.bw_gbps = inst.bw_gbps[np.ix_(sw, sw)].copy(); o.island_cap_mb = inst.island_cap_mb[sw].copy()
    r0, r1 = oracle.solve(inst), oracle.solve(o)
    assert r0.plan_key() == r1.plan_key()       # the instance is literally the same


@pytest.mark.parametrize("seed", range(40))
def test_monotone_in_T_and_m_and_scaling(seed):
    inst = gen.random_small(seed + 3000, Lmax=7, Kmax=4, Pmax=2, style=STYLES[seed % 5])
    _, _, _, cand = oracle.reduce(inst)
    prev = None
    for T in cand:                                                    # f_T non-increasing in T
        q = oracle.dp_at(inst, int(T), want_plan=False)
        f = q.sum_us if q.feasible else oracle.INF
        assert prev is None or f <= prev
        prev = f
    its = []
    for m in (1, 2, 3, 8, 64):                                        # iter non-decreasing in m
        o = inst.copy(); o.m = m
        r = oracle.solve(o)
        its.append(r.iter_time_us)
    assert its == sorted(its)
    # multiplying every time by q multiplies iter by q when transfers are zero
    o = inst.copy(); o.act_mb = 0
    r0 = oracle.solve(o)
    o.time_us = np.where(o.time_us == INVALID, INVALID, o.time_us.astype(np.int64) * 3).astype(np.int32)
    r1 = oracle.solve(o)
    if r0.feasible:
        assert r1.iter_time_us == 3 * r0.iter_time_us and r1.stages == r0.stages


@pytest.mark.parametrize("seed", range(40))
def test_large_m_minimises_the_bottleneck_first(seed):
    """P-balance: for m large the optimum's T* is the min-max bottleneck =
    the lowest feasible candidate threshold."""
    inst = gen.random_small(seed + 4000, Lmax=7, Kmax=4, Pmax=2, style=STYLES[seed % 5])
    inst.m = 1 << 20
    r = oracle.solve(inst)
    if not r.feasible:
        return
    _, _, _, cand = oracle.reduce(inst)
    lowest = next(int(T) for T in cand if oracle.dp_at(inst, int(T), want_plan=False).feasible)
    assert r.bottleneck_us == lowest


@pytest.mark.parametrize("name", ["cfg1", "cfg2"])
def test_named_configs_rescore_and_cover(name):
    inst = gen.by_name(name)
    r = oracle.solve(inst)
    full = oracle.solve(inst, full_sweep=True)
    assert r.plan_key() == full.plan_key()
    s, T, it, mask = rescore(inst, r.stages)
    assert (s, T, it, mask) == (r.sum_us, r.bottleneck_us, r.iter_time_us, r.island_mask)
    assert r.stages[0][0] == 0 and len({k for _, k, _ in r.stages}) == r.n_stages
