"""Seeded synthetic planning instances shaped like TANGRAM's workloads.

This module only *draws inputs* (cost / memory tables, islands, bandwidths).  It
holds none of the method's arithmetic: no table reduction, no transfer times, no
DP, no pruning.  The oracle (`oracle/`) and the CUDA library
(`paper_2606_16907_b200/`) both consume the byte buffers produced here, so
generator arithmetic can never cause a parity failure.

Recipe: DESIGN.md "Input recipe" (concretises BASELINE.json:configs[0..4];
SURVEY.md §8(d)).  The paper's profiled cost tables (§6.1
:276-290) are not available; these synthetic tables stand in for them.

RNG: counter-based 64-bit mixer on (seed, stream, element index), so any element
can be reproduced in isolation.  u(lo,hi) = lo + r mod (hi-lo+1).
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

TG_INVALID = 0x7FFFFFFF
TG_TIME_MAX = 1 << 25

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)
_C1 = np.uint64(0x9E3779B97F4A7C15)
_C2 = np.uint64(0xBF58476D1CE4E5B9)
_C3 = np.uint64(0x94D049BB133111EB)

# RNG stream ids
S_NOISE, S_GEN, S_NGPU, S_BW, S_MISC = 1, 2, 3, 4, 5


def mix64(seed: int, stream: int, idx) -> np.ndarray:
    """SplitMix64-style finaliser of (seed, stream, idx) -> uint64 array."""
    idx = np.asarray(idx, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = (np.uint64(seed) * _C1 + np.uint64(stream) * _C2 + np.uint64(0x2545F4914F6CDD1D)) & _M64
        z = z + idx * _C3 + _C1
        z ^= z >> np.uint64(30)
        z *= _C2
        z ^= z >> np.uint64(27)
        z *= _C3
        z ^= z >> np.uint64(31)
    return z


def urand(seed: int, stream: int, idx, lo: int, hi: int) -> np.ndarray:
    r = mix64(seed, stream, idx)
    return (np.int64(lo) + (r % np.uint64(hi - lo + 1)).astype(np.int64))


def n_slices(L: int) -> int:
    return L * (L + 1) // 2


def slice_index(L: int, a: int, b: int) -> int:
    """s(a,b) = a(2L-a+1)/2 + (b-a-1): a-major, b ascending."""
    return a * (2 * L - a + 1) // 2 + (b - a - 1)


def slice_bounds(L: int):
    a = np.concatenate([np.full(L - i, i, dtype=np.int64) for i in range(L)])
    b = np.concatenate([np.arange(i + 1, L + 1, dtype=np.int64) for i in range(L)])
    return a, b


@dataclass
class Instance:
    name: str
    L: int
    K: int
    P: int
    m: int
    time_us: np.ndarray       # [NS, K, P] int32, TG_INVALID = no such plan
    mem_mb: np.ndarray        # [NS, K, P] int32
    island_gpus: np.ndarray   # [K] int32
    island_cap_mb: np.ndarray  # [K] int32
    bw_gbps: np.ndarray       # [K, K] int32 sender-major
    act_mb: int
    meta: dict = field(default_factory=dict)
    actmem_mb: np.ndarray = None   # [NS, K, P] int32 or None: MB per in-flight microbatch (NEXT-1, depth-aware memory)
    transfer_bound: bool = False   # NEXT-3(b): transfers count toward the bottleneck (x <= T as well)
    act_mb_b: np.ndarray = None    # [L+1] int32 or None: activation MB crossing boundary b = 1..L-1 (NEXT-3(b), per-boundary sizes)
    slow_us: np.ndarray = None     # [NS, K, P] int32 or None: slowest internal stage of the partial plan (NEXT-2)
    q_stages: np.ndarray = None    # [NS, K, P] int32 or None: its number of internal pipeline stages (NEXT-2)

    def copy(self) -> "Instance":
        return Instance(self.name, self.L, self.K, self.P, self.m, self.time_us.copy(),
                        self.mem_mb.copy(), self.island_gpus.copy(), self.island_cap_mb.copy(),
                        self.bw_gbps.copy(), self.act_mb, dict(self.meta),
                        None if self.actmem_mb is None else self.actmem_mb.copy(), self.transfer_bound,
                        None if self.act_mb_b is None else self.act_mb_b.copy(),
                        None if self.slow_us is None else self.slow_us.copy(),
                        None if self.q_stages is None else self.q_stages.copy())


def _cdiv(a, b):
    return -((-a) // b)


GEN3 = [(1, 40), (2, 80), (4, 180)]
GEN4 = [(1, 40), (2, 80), (3, 141), (4, 180)]
BW_CHOICES = np.array([25, 50, 100, 400], dtype=np.int64)
E_BY_TP = [950, 900, 820, 700]


def _bw_matrix(seed: int, K: int) -> np.ndarray:
    bw = np.full((K, K), 400, dtype=np.int64)
    for j in range(K):
        for k in range(j + 1, K):
            v = BW_CHOICES[int(urand(seed, S_BW, j * K + k, 0, 3))]
            bw[j, k] = bw[k, j] = v
    return bw.astype(np.int32)


def _build_tables(seed, L, K, P, w, pm1, pm2, am, speed, ngpu, plans):
    """plans: list of dicts with keys
         deg   : degree that must divide n (validity)
         d1,d2 : memory shard degree of pm1 / pm2; int, or 'n' for the island's GPU count
         tm,e,af : per-mille time multiplier, efficiency, activation factor
         extra : per-slice extra microseconds array [NS] or 0
    time = ceil(W*noise*tm / (v*n*e*1000)) + extra ;  mem = ceil(PM1/d1)+ceil(PM2/d2)+ceil(AM*af/1000)+500
    """
    NS = n_slices(L)
    a, b = slice_bounds(L)
    pw = np.concatenate([[0], np.cumsum(w)]).astype(np.int64)
    p1 = np.concatenate([[0], np.cumsum(pm1)]).astype(np.int64)
    p2 = np.concatenate([[0], np.cumsum(pm2)]).astype(np.int64)
    pa = np.concatenate([[0], np.cumsum(am)]).astype(np.int64)
    W = pw[b] - pw[a]
    PM1 = p1[b] - p1[a]
    PM2 = p2[b] - p2[a]
    AM = pa[b] - pa[a]
    time = np.empty((NS, K, P), dtype=np.int64)
    mem = np.empty((NS, K, P), dtype=np.int64)
    sidx = np.arange(NS, dtype=np.int64)
    for k in range(K):
        v, n = int(speed[k]), int(ngpu[k])
        for p, pl in enumerate(plans):
            noise = urand(seed, S_NOISE, (sidx * K + k) * P + p, 900, 1100)
            t = _cdiv(W * noise * pl["tm"], v * n * pl["e"] * 1000)
            ex = pl.get("extra", 0)
            t = t + ex
            d1 = n if pl["d1"] == "n" else pl["d1"]
            d2 = n if pl["d2"] == "n" else pl["d2"]
            mm = _cdiv(PM1, d1) + _cdiv(PM2, d2) + _cdiv(AM * pl["af"], 1000) + 500
            if n % pl["deg"] != 0:
                t = np.full(NS, TG_INVALID, dtype=np.int64)
            time[:, k, p] = t
            mem[:, k, p] = mm
    assert time[time != TG_INVALID].max() <= TG_TIME_MAX
    return time.astype(np.int32), mem.astype(np.int32)


def config1(seed: int = 0, cap_div: int = 1) -> Instance:
    """Tiny, brute-force-checkable (BASELINE.json:configs[0]).  cap_div=10 gives the
    'tiny-mem' twin whose memory caps bind."""
    L, K, P, m = 8, 3, 2, 8
    ngpu = np.array([2, 4, 2]); speed = np.array([1, 2, 4]); gb = np.array([40, 80, 180])
    w = np.full(L, 1000); pm = np.full(L, 1500); z = np.zeros(L, dtype=np.int64)
    plans = [dict(deg=1, d1=1, d2=1, tm=1000, e=900, af=1000),
             dict(deg=1, d1="n", d2=1, tm=1000, e=800, af=1000)]
    t, mm = _build_tables(seed, L, K, P, w, pm, z, z, speed, ngpu, plans)
    bw = np.array([[400, 25, 100], [25, 400, 400], [100, 400, 400]], dtype=np.int32)
    return Instance(f"cfg1_tiny_s{seed}" + ("" if cap_div == 1 else f"_capdiv{cap_div}"), L, K, P, m, t, mm,
                    ngpu.astype(np.int32), (gb * 1000 // cap_div).astype(np.int32), bw, 64,
                    dict(speed=speed.tolist()))


def _tp_plans():
    return [dict(deg=tp, d1=tp, d2=1, tm=1000, e=E_BY_TP[i], af=1000) for i, tp in enumerate([1, 2, 4, 8])]


def _islands(seed, K, gens, nlo, nhi):
    g = urand(seed, S_GEN, np.arange(K), 0, len(gens) - 1)
    n = urand(seed, S_NGPU, np.arange(K), nlo, nhi)
    speed = np.array([gens[int(i)][0] for i in g]); gb = np.array([gens[int(i)][1] for i in g])
    return speed, gb, n


def config2(seed: int = 0) -> Instance:
    """Dense 7B-like (BASELINE.json:configs[1])."""
    L, K, P, m = 32, 6, 4, 16
    speed, gb, n = _islands(seed, K, GEN3, 1, 8)
    cm = np.ones(L, dtype=np.int64); cm[0] = cm[-1] = 2
    w = 1000 * cm; pm = 1500 * cm; z = np.zeros(L, dtype=np.int64)
    t, mm = _build_tables(seed, L, K, P, w, pm, z, z, speed, n, _tp_plans())
    return Instance(f"cfg2_7b_s{seed}", L, K, P, m, t, mm, n.astype(np.int32), (gb * 1000).astype(np.int32),
                    _bw_matrix(seed, K), 64, dict(speed=speed.tolist()))


def config3(seed: int = 0, L: int = 80, K: int = 12) -> Instance:
    """Dense 70B-like (BASELINE.json:configs[2])."""
    P, m = 8, 32
    speed, gb, n = _islands(seed, K, GEN4, 2, 8)
    w = np.full(L, 4000); pm = np.full(L, 6000); am = np.full(L, 800); z = np.zeros(L, dtype=np.int64)
    plans = [dict(deg=tp, d1=tp, d2=1, tm=1000, e=E_BY_TP[i], af=1000 // tp) for i, tp in enumerate([1, 2, 4, 8])]
    plans += [dict(deg=1, d1="n", d2=1, tm=1150, e=950, af=1000),      # TP1 + ZeRO
              dict(deg=2, d1="n", d2=1, tm=1150, e=900, af=500),       # TP2 + ZeRO
              dict(deg=1, d1=1, d2=1, tm=1330, e=950, af=400),         # TP1 + recompute
              dict(deg=2, d1="n", d2=1, tm=1530, e=900, af=200)]       # TP2 + ZeRO + recompute
    t, mm = _build_tables(seed, L, K, P, w, pm, z, am, speed, n, plans)
    return Instance(f"cfg3_70b_s{seed}", L, K, P, m, t, mm, n.astype(np.int32), (gb * 1000).astype(np.int32),
                    _bw_matrix(seed, K), 64, dict(speed=speed.tolist()))


def config4(seed: int = 0, L: int = 64, K: int = 16) -> Instance:
    """MoE 8-expert-like (BASELINE.json:configs[3])."""
    P, m = 8, 64
    speed, gb, n = _islands(seed, K, GEN4, 1, 8)
    moe = (np.arange(L) % 2 == 1)
    w = np.where(moe, 2000, 1000); pm_attn = np.where(moe, 0, 1500); pm_moe = np.where(moe, 12000, 0)
    am = np.full(L, 400)
    a, b = slice_bounds(L)
    pmoe = np.concatenate([[0], np.cumsum(moe.astype(np.int64))])
    nmoe = pmoe[b] - pmoe[a]
    a2a = _cdiv(256 * 1000, 600)  # 427 us per MoE layer
    plans = []
    for i, ep in enumerate([1, 2, 4, 8]):
        for rc in (0, 1):
            plans.append(dict(deg=ep, d1=1, d2=ep, tm=1330 if rc else 1000, e=[900, 880, 860, 840][i],
                              af=400 if rc else 1000, extra=(nmoe * a2a if ep > 1 else 0)))
    t, mm = _build_tables(seed, L, K, P, w, pm_attn, pm_moe, am, speed, n, plans)
    return Instance(f"cfg4_moe_s{seed}", L, K, P, m, t, mm, n.astype(np.int32), (gb * 1000).astype(np.int32),
                    _bw_matrix(seed, K), 64, dict(speed=speed.tolist()))


def config5_one(seed: int, L: int = 48, K: int = 10) -> Instance:
    """One instance of the throughput batch (BASELINE.json:configs[4])."""
    P = 4
    m = [4, 8, 16, 32, 64][seed % 5]
    speed, gb, n = _islands(seed, K, GEN4, 1, 8)
    cm = np.ones(L, dtype=np.int64); cm[0] = cm[-1] = 2
    w = 2250 * cm; pm = 3375 * cm; z = np.zeros(L, dtype=np.int64)
    t, mm = _build_tables(seed, L, K, P, w, pm, z, z, speed, n, _tp_plans())
    return Instance(f"cfg5_batch_s{seed}", L, K, P, m, t, mm, n.astype(np.int32), (gb * 1000).astype(np.int32),
                    _bw_matrix(seed, K), 64, dict(speed=speed.tolist()))


def config5(n_inst: int = 1024, first_seed: int = 0, L: int = 48, K: int = 10):
    return [config5_one(first_seed + i, L, K) for i in range(n_inst)]


def random_small(seed: int, Lmax: int = 8, Kmax: int = 5, Pmax: int = 3, style: str = "mixed") -> Instance:
    """Randomised small instance for brute-force / parity suites.
    style: 'mixed' | 'ties' (few distinct values) | 'tightmem' | 'asym' (asymmetric bandwidth)
           | 'sparse' (many invalid entries)"""
    r = lambda i, lo, hi: int(urand(seed, S_MISC, i, lo, hi))
    L = r(0, 1, Lmax); K = r(1, 1, Kmax); P = r(2, 1, Pmax); m = [1, 2, 4, 8, 64][r(3, 0, 4)]
    NS = n_slices(L)
    a, b = slice_bounds(L)
    ln = (b - a)[:, None, None]
    idx = np.arange(NS * K * P).reshape(NS, K, P)
    spd = urand(seed, S_GEN, np.arange(K), 1, 4)[None, :, None]
    if style == "ties":
        t = ln * 10 * urand(seed, S_NOISE, idx, 1, 2)
    else:
        t = _cdiv(ln * 1000 * urand(seed, S_NOISE, idx, 700, 1300), spd * 1000)
    mm = ln * 100 * urand(seed, S_NOISE + 10, idx, 1, 4)
    cap = urand(seed, S_NGPU + 10, np.arange(K), 2, 12) * (100 if style == "tightmem" else 400)
    if style == "sparse":
        kill = urand(seed, S_NOISE + 20, idx, 0, 2) == 0
        t = np.where(kill, TG_INVALID, t)
    bw = urand(seed, S_BW, np.arange(K * K), 1, 40).reshape(K, K)
    if style != "asym":
        bw = np.minimum(bw, bw.T)
    act = r(4, 0, 3) * 32
    return Instance(f"rand_{style}_s{seed}", L, K, P, m, t.astype(np.int32), mm.astype(np.int32),
                    urand(seed, S_NGPU, np.arange(K), 1, 8).astype(np.int32), cap.astype(np.int32),
                    bw.astype(np.int32), act)


def with_actmem(inst: Instance, seed: int, lo: int = 0, hi: int = 60) -> Instance:
    """Adds a per-plan activation footprint (MB per in-flight microbatch) proportional to the slice length."""
    o = inst.copy()
    NS, K, P = inst.time_us.shape
    a, b = slice_bounds(inst.L)
    idx = np.arange(NS * K * P).reshape(NS, K, P)
    o.actmem_mb = ((b - a)[:, None, None] * urand(seed, S_MISC + 30, idx, lo, hi)).astype(np.int32)
    o.name = inst.name + "_act"
    return o


def length_classes(inst: Instance):
    """Signature classes of a model of identical layers (NEXT-3(a)): the class of a slice is its length, and the class
    tables are the rows of the slices that start at layer 0.  Returns (class_of_slice [NS], class_time [L,K,P],
    class_mem [L,K,P], the expanded Instance these define)."""
    L = inst.L
    a, b = slice_bounds(L)
    class_of = (b - a - 1).astype(np.int32)
    rows = np.array([slice_index(L, 0, d) for d in range(1, L + 1)])
    ct, cm = inst.time_us[rows].copy(), inst.mem_mb[rows].copy()
    o = inst.copy()
    o.time_us, o.mem_mb = ct[class_of], cm[class_of]
    o.name = inst.name + "_cls"
    return class_of, ct, cm, o


def with_transfer_bound(inst: Instance) -> Instance:
    """Same tables, transfers bounded by the threshold as well (NEXT-3(b))."""
    o = inst.copy()
    o.transfer_bound = True
    o.name = inst.name + "_xb"
    return o


def with_boundary_act(inst: Instance, seed: int, sizes=(16, 64, 256)) -> Instance:
    """NEXT-3(b): the activation crossing boundary b has one of a few sizes (MB), e.g. narrow after an attention block,
    wide after an MoE block or the embedding (the paper prints no activation sizes)."""
    o = inst.copy()
    b = np.arange(inst.L + 1)
    o.act_mb_b = np.asarray(sizes, dtype=np.int64)[urand(seed, S_MISC + 60, b, 0, len(sizes) - 1)].astype(np.int32)
    o.name = inst.name + "_ab"
    return o


def with_stages(inst: Instance, seed: int, qmax: int = 4) -> Instance:
    """NEXT-2: every entry becomes a partial plan of q = u(1, min(qmax, slice length)) internal pipeline stages whose
    slowest stage is between an even split and 1.6 x it: slow = min(time, ceil(time / q * u(1000, 1600) / 1000)); q = 1 keeps
    slow = time.  The paper prints no figures for the internal stages of a parallelizer's plan."""
    o = inst.copy()
    NS, K, P = inst.time_us.shape
    a, b = slice_bounds(inst.L)
    idx = np.arange(NS * K * P).reshape(NS, K, P)
    q = 1 + (urand(seed, S_MISC + 40, idx, 0, qmax - 1) % np.minimum(qmax, (b - a))[:, None, None])
    t = inst.time_us.astype(np.int64)
    even = -(-t // q)
    slow = np.minimum(t, -(-(even * urand(seed, S_MISC + 41, idx, 1000, 1600)) // 1000))
    slow = np.where(q == 1, t, slow)
    slow = np.where(inst.time_us == TG_INVALID, 0, slow)
    o.slow_us = slow.astype(np.int32)
    o.q_stages = q.astype(np.int32)
    o.name = inst.name + "_st"
    return o


# ---- NEXT-4: cluster profiles for the island construction (PAPER.md:177 per-GPU attributes, given per node) -------------
# GPU types of Tab. 3: (relative compute, memory MB, intra-node link GB/s: PCIe 32, NVLink 300/600/900).
# The paper prints no bandwidth figures: nodes bought together share a dedicated interconnect, modelled as
# 100 GB/s between nodes of one type and 25 GB/s across types.
GPU_TYPES = {"T4": (65, 16000, 32), "V100-16": (125, 16000, 32), "V100-32": (125, 32000, 300),
             "A100-80": (312, 80000, 600), "H100NVL": (835, 94000, 900)}
CLUSTERS = {"C1": [("T4", 4, 4), ("V100-16", 4, 4)],                                   # (type, nodes, GPUs per node)
            "C2": [("A100-80", 2, 4), ("H100NVL", 4, 2)],
            "C3": [("T4", 1, 4), ("V100-16", 1, 4), ("V100-32", 1, 8), ("A100-80", 1, 4)]}


def cluster_profile(name: str, same: int = 100, cross: int = 25):
    """(gpus, comp, mem_mb, intra, inter [N,N]) of an evaluation cluster of PAPER.md Tab. 3."""
    gp, cp, mm, ib, ty = [], [], [], [], []
    for t, nodes, g in CLUSTERS[name]:
        c, m, b = GPU_TYPES[t]
        for _ in range(nodes):
            gp.append(g); cp.append(c); mm.append(m); ib.append(b); ty.append(t)
    n = len(gp)
    inter = np.array([[0 if i == j else (same if ty[i] == ty[j] else cross) for j in range(n)] for i in range(n)], dtype=np.int32)
    return (np.array(gp, np.int32), np.array(cp, np.int32), np.array(mm, np.int32), np.array(ib, np.int32), inter)


def random_cluster(seed: int, nmax: int = 12):
    """A random cluster: 2-nmax nodes drawn from a few GPU types with a few percent of spread, asymmetric links."""
    n = int(urand(seed, S_MISC + 50, 0, 2, nmax))
    idx = np.arange(n)
    types = list(GPU_TYPES.values())
    t = urand(seed, S_MISC + 51, idx, 0, len(types) - 1)
    gp = 1 << urand(seed, S_MISC + 52, t, 1, 3)                                       # GPUs per node follow the type
    comp = np.array([types[i][0] for i in t]) * urand(seed, S_MISC + 53, idx, 97, 103) // 100
    mem = np.array([types[i][1] for i in t]) * urand(seed, S_MISC + 54, idx, 99, 101) // 100
    intra = np.array([types[i][2] for i in t])
    pair = idx[:, None] * n + idx[None, :]
    inter = np.where(t[:, None] == t[None, :], urand(seed, S_MISC + 55, pair, 80, 120), urand(seed, S_MISC + 56, pair, 10, 90))
    np.fill_diagonal(inter, 0)
    return (gp.astype(np.int32), comp.astype(np.int32), mem.astype(np.int32), intra.astype(np.int32), inter.astype(np.int32))


def by_name(name: str, seed: int = 0):
    return {"cfg1": config1, "cfg2": config2, "cfg3": config3, "cfg4": config4}[name](seed)
