"""TEST INFRASTRUCTURE — ctypes front end of the CPU oracle (oracle/tangram_oracle.cpp).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this.  It never imports the CUDA package and the CUDA package never imports it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_DIR, "tangram_oracle.cpp")
_SRC_DEPTH = os.path.join(_DIR, "tangram_oracle_depth.cpp")   # NEXT-1 variant, separate translation unit
_SRC_STAGES = os.path.join(_DIR, "tangram_oracle_stages.cpp")  # NEXT-2 variant, separate translation unit
_SRC_ISLANDS = os.path.join(_DIR, "tangram_oracle_islands.cpp")  # NEXT-4 front end, separate translation unit
# TG_ORACLE_LIB / TG_ORACLE_CXXFLAGS: an instrumented build beside the plain one (the CPU suite under
# AddressSanitizer + UBSan:  TG_ORACLE_LIB=oracle/libtangram_oracle_asan.so TG_ORACLE_CXXFLAGS="-fsanitize=address,undefined
# -fno-sanitize-recover=all -g" LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 pytest -m "not gpu")
_SO = os.path.abspath(os.environ.get("TG_ORACLE_LIB", os.path.join(_DIR, "libtangram_oracle.so")))
MAXK = 16
INF = 1 << 30
INT64_MAX = (1 << 63) - 1


def build(force: bool = False) -> str:
    srcs = [f for f in (_SRC, _SRC_DEPTH, _SRC_STAGES, _SRC_ISLANDS) if os.path.exists(f)]
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < max(os.path.getmtime(f) for f in srcs):
        tmp = _SO + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-pthread"] + os.environ.get("TG_ORACLE_CXXFLAGS", "").split() +
                              ["-o", tmp] + srcs)
        os.replace(tmp, _SO)
    return _SO


class _Res(C.Structure):
    _fields_ = [("iter_time_us", C.c_int64), ("sum_us", C.c_int64), ("bottleneck_us", C.c_int64),
                ("n_stages", C.c_int32), ("island_mask", C.c_uint32), ("n_dp_run", C.c_int32),
                ("n_candidates", C.c_int32), ("stage_begin", C.c_int32 * MAXK),
                ("stage_island", C.c_int32 * MAXK), ("stage_plan", C.c_int32 * MAXK)]


@dataclass
class Result:
    iter_time_us: int
    sum_us: int
    bottleneck_us: int
    n_stages: int
    island_mask: int
    stages: list          # [(begin, island, plan)]
    n_dp_run: int = 0
    n_candidates: int = 0
    first_island: int = -1

    @property
    def feasible(self) -> bool:
        return self.iter_time_us != INT64_MAX

    def plan_key(self):
        return (self.iter_time_us, self.sum_us, self.bottleneck_us, self.island_mask, tuple(self.stages))


_lib = None
_I32P = C.POINTER(C.c_int32)
_I64P = C.POINTER(C.c_int64)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_laneless_iter.restype = C.c_int64
    return _lib


def _p32(a):
    return a.ctypes.data_as(_I32P)


def _args(inst):
    t = np.ascontiguousarray(inst.time_us, dtype=np.int32)
    mm = np.ascontiguousarray(inst.mem_mb, dtype=np.int32)
    cap = np.ascontiguousarray(inst.island_cap_mb, dtype=np.int32)
    bw = np.ascontiguousarray(inst.bw_gbps, dtype=np.int32)
    keep = (t, mm, cap, bw)
    return keep, (C.c_int(inst.L), C.c_int(inst.K), C.c_int(inst.P), C.c_int(inst.m), _p32(t), _p32(mm),
                  _p32(cap), _p32(bw), C.c_int(inst.act_mb))


def _conv(r: _Res) -> Result:
    n = r.n_stages
    return Result(r.iter_time_us, r.sum_us, r.bottleneck_us, n, r.island_mask,
                  [(r.stage_begin[i], r.stage_island[i], r.stage_plan[i]) for i in range(n)],
                  r.n_dp_run, r.n_candidates, r.stage_island[0])


def solve(inst, full_sweep: bool = False, n_threads: int = 1) -> Result:
    keep, a = _args(inst)
    r = _Res()
    lib().orc_solve(*a, C.c_int(int(full_sweep)), C.c_int(n_threads), C.byref(r))
    return _conv(r)


def bruteforce(inst):
    keep, a = _args(inst)
    r = _Res()
    n = C.c_int64(0)
    lib().orc_bruteforce(*a, C.byref(r), C.byref(n))
    return _conv(r), n.value


def dp_at(inst, T: int, want_plan: bool = True) -> Result:
    """DP at one threshold (T < 0: infinity).  sum_us = f_T; infeasible -> feasible == False."""
    keep, a = _args(inst)
    r = _Res()
    lib().orc_dp_at(*a, C.c_int64(T), C.c_int(int(want_plan)), C.byref(r))
    return _conv(r)


def laneless_iter(inst, xc: int) -> int:
    keep, a = _args(inst)
    return lib().orc_laneless_iter(*a[:7], C.c_int64(xc))


def reduce(inst):
    """-> c [NS,K] int64 (2^30 none), argp [NS,K] int32, x [K,K] int64, candidates int64[]"""
    keep, a = _args(inst)
    NS = inst.L * (inst.L + 1) // 2
    c = np.empty((NS, inst.K), dtype=np.int64)
    argp = np.empty((NS, inst.K), dtype=np.int32)
    x = np.empty((inst.K, inst.K), dtype=np.int64)
    cand = np.empty(NS * inst.K, dtype=np.int64)
    n = lib().orc_reduce(a[0], a[1], a[2], a[4], a[5], a[6], a[7], a[8], c.ctypes.data_as(_I64P),
                         _p32(argp), x.ctypes.data_as(_I64P), cand.ctypes.data_as(_I64P))
    return c, argp, x, cand[:n].copy()


def prune(inst, mode: int = 0, threshold: int = 0):
    """Returns (pruned copy of inst, counts[4]).  inst itself is not modified."""
    out = inst.copy()
    t = np.ascontiguousarray(out.time_us, dtype=np.int32)
    mm = np.ascontiguousarray(out.mem_mb, dtype=np.int32)
    cap = np.ascontiguousarray(out.island_cap_mb, dtype=np.int32)
    counts = np.zeros(4, dtype=np.int64)
    lib().orc_prune(C.c_int(out.L), C.c_int(out.K), C.c_int(out.P), _p32(t), _p32(mm), _p32(cap),
                    C.c_int(mode), C.c_int64(threshold), counts.ctypes.data_as(_I64P))
    out.time_us = t
    return out, counts


def _args_depth(inst):
    keep, a = _args(inst)
    am = np.ascontiguousarray(inst.actmem_mb, dtype=np.int32)
    return (keep, am), a[:6] + (_p32(am),) + a[6:]


def solve_depth(inst) -> Result:
    """NEXT-1: depth-aware activation memory (inst.actmem_mb [NS,K,P])."""
    keep, a = _args_depth(inst)
    r = _Res()
    lib().orc_depth_solve(*a, C.byref(r))
    return _conv(r)


def bruteforce_depth(inst) -> Result:
    keep, a = _args_depth(inst)
    r = _Res()
    lib().orc_depth_bruteforce(*a, C.byref(r))
    return _conv(r)


def _args_variant(inst):
    keep, a = _args(inst)
    am = None if inst.actmem_mb is None else np.ascontiguousarray(inst.actmem_mb, dtype=np.int32)
    amp = C.cast(None, _I32P) if am is None else _p32(am)
    return (keep, am), a[:6] + (amp,) + a[6:] + (C.c_int(1 if getattr(inst, "transfer_bound", False) else 0),)


def solve_variant(inst, n_threads: int = 0) -> Result:
    """Variants of SURVEY §8(f): NEXT-1 depth-aware memory (inst.actmem_mb) and NEXT-3(b) transfers bounded by
    T (inst.transfer_bound), alone or together; with neither this is the core definition.
    n_threads > 0: the same arithmetic with the schedule of the core oracle's solve (bisection for the lowest feasible
    threshold, blocks of n_threads DPs) -- for the K = 16 configs."""
    keep, a = _args_variant(inst)
    r = _Res()
    if n_threads > 0:
        lib().orc_variant_solve_mt(*a, C.c_int(n_threads), C.byref(r))
    else:
        lib().orc_variant_solve(*a, C.byref(r))
    return _conv(r)


def _args_variant_b(inst):
    keep, a = _args_variant(inst)                      # (..., act_mb, xbound)
    ab = None if getattr(inst, "act_mb_b", None) is None else np.ascontiguousarray(inst.act_mb_b, dtype=np.int32)
    abp = C.cast(None, _I32P) if ab is None else _p32(ab)
    return (keep, ab), a[:-1] + (abp, a[-1])


def solve_variant_b(inst) -> Result:
    """Variant oracle with per-boundary activation sizes (inst.act_mb_b [L+1] or None), NEXT-3(b) second half."""
    keep, a = _args_variant_b(inst)
    r = _Res()
    lib().orc_variant_solve_b(*a, C.byref(r))
    return _conv(r)


def bruteforce_variant_b(inst) -> Result:
    keep, a = _args_variant_b(inst)
    r = _Res()
    lib().orc_variant_bruteforce_b(*a, C.byref(r))
    return _conv(r)


def bruteforce_variant(inst) -> Result:
    keep, a = _args_variant(inst)
    r = _Res()
    lib().orc_variant_bruteforce(*a, C.byref(r))
    return _conv(r)


def prune_depth(inst, mode: int = 0, threshold: int = 0):
    """tg_prune on an instance with a footprint table (3-way dominance).  Returns (pruned copy, counts[4])."""
    out = inst.copy()
    t = np.ascontiguousarray(out.time_us, dtype=np.int32)
    mm = np.ascontiguousarray(out.mem_mb, dtype=np.int32)
    am = np.ascontiguousarray(out.actmem_mb, dtype=np.int32)
    cap = np.ascontiguousarray(out.island_cap_mb, dtype=np.int32)
    counts = np.zeros(4, dtype=np.int64)
    lib().orc_prune_depth(C.c_int(out.L), C.c_int(out.K), C.c_int(out.P), _p32(t), _p32(mm), _p32(am), _p32(cap),
                          C.c_int(mode), C.c_int64(threshold), counts.ctypes.data_as(_I64P))
    out.time_us = t
    return out, counts


def _args_stages(inst):
    keep, a = _args(inst)
    sl = np.ascontiguousarray(inst.slow_us, dtype=np.int32)
    qs = None if getattr(inst, "q_stages", None) is None else np.ascontiguousarray(inst.q_stages, dtype=np.int32)
    qp = C.cast(None, _I32P) if qs is None else _p32(qs)
    return (keep, sl, qs), a[:6] + (_p32(sl), qp) + a[6:]


def solve_stages(inst):
    """NEXT-2: multi-stage partial plans (inst.slow_us [NS,K,P] slowest internal stage, inst.q_stages [NS,K,P] or None).
    Returns (Result, total pipeline stages of the plan)."""
    keep, a = _args_stages(inst)
    r = _Res()
    tot = C.c_int32(0)
    lib().orc_stages_solve(*a, C.byref(r), C.byref(tot))
    return _conv(r), tot.value


def bruteforce_stages(inst):
    keep, a = _args_stages(inst)
    r = _Res()
    tot = C.c_int32(0)
    n = C.c_int64(0)
    lib().orc_stages_bruteforce(*a, C.byref(r), C.byref(tot), C.byref(n))
    return _conv(r), tot.value, n.value


def islands(gpus, comp, mem_mb, intra, inter, eps_c: int, eps_m: int, eps_i: int):
    """NEXT-4: island construction from per-node profiles (tolerances in permille).
    Returns (island_of_node [N], island_gpus [K], island_cap_mb [K], bw [K,K])."""
    g, c, mm, b = (np.ascontiguousarray(a, dtype=np.int32) for a in (gpus, comp, mem_mb, intra))
    e = np.ascontiguousarray(inter, dtype=np.int32)
    N = g.size
    of = np.zeros(N, dtype=np.int32)
    ig, ic, bw = np.zeros(N, dtype=np.int32), np.zeros(N, dtype=np.int32), np.zeros(N * N, dtype=np.int32)
    K = C.c_int32(0)
    lib().orc_islands(C.c_int(N), _p32(g), _p32(c), _p32(mm), _p32(b), _p32(e), C.c_int(eps_c), C.c_int(eps_m), C.c_int(eps_i),
                      _p32(of), C.byref(K), _p32(ig), _p32(ic), _p32(bw))
    k = K.value
    return of, ig[:k].copy(), ic[:k].copy(), bw[:k * k].reshape(k, k).copy()


def hw_threads() -> int:
    return lib().orc_hw_threads()
