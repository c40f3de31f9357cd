"""Thin Python binding of libtangram (include/tangram.h): argument marshalling only.

Every step of the path — cost-table loader, candidate thresholds, per-T wavefront DP, sweep
reduction, back-tracker, pruning — runs in the CUDA kernels of `csrc/`.  There is no CPU fallback:
if the shared library is missing or no CUDA device is present the calls raise.

Names follow the C ABI: tg_instance_create, tg_instance_destroy, tg_solve_batch, tg_solve_batch_ex,
tg_prune, tg_reduce, tg_dp_at, tg_instance_read_time, tg_last_error, tg_version.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_DIR, "libtangram.so")

TG_MAX_K = 16
TG_INVALID = 0x7FFFFFFF
TG_INF = 1 << 30
INT64_MAX = (1 << 63) - 1
TG_SOLVE_DEFAULT, TG_SOLVE_FULL_SWEEP = 0, 1
TG_PRUNE_EXACT, TG_PRUNE_IMBALANCE, TG_PRUNE_BOTTLENECK = 0, 1, 2
STATUS = {0: "TG_OK", 1: "TG_ERR_NULL", 2: "TG_ERR_SHAPE", 3: "TG_ERR_RANGE", 4: "TG_ERR_OOM", 5: "TG_ERR_CUDA"}


class TgResult(C.Structure):
    _fields_ = [("iter_time_us", C.c_int64), ("sum_us", C.c_int64), ("bottleneck_us", C.c_int32),
                ("n_stages", C.c_int32), ("island_mask", C.c_uint32), ("n_thresholds_run", C.c_uint32),
                ("stage_begin", C.c_int32 * TG_MAX_K), ("stage_island", C.c_int32 * TG_MAX_K),
                ("stage_plan", C.c_int32 * TG_MAX_K)]

    @property
    def feasible(self) -> bool:
        return self.iter_time_us != INT64_MAX

    @property
    def stages(self):
        return [(self.stage_begin[i], self.stage_island[i], self.stage_plan[i]) for i in range(self.n_stages)]


class TgSolveStats(C.Structure):
    _fields_ = [("n_dp", C.c_uint64), ("plans_dense", C.c_uint64), ("states_live", C.c_uint64),
                ("n_rounds", C.c_uint64), ("n_barriers", C.c_uint64), ("n_items_global_c", C.c_uint64),
                ("error_flag", C.c_uint64), ("relax_admissible", C.c_uint64), ("states_windowed", C.c_uint64),
                ("cyc_stage", C.c_uint64), ("cyc_levels", C.c_uint64), ("cyc_level_barrier", C.c_uint64),
                ("cyc_grid_wait", C.c_uint64), ("cyc_scheduler", C.c_uint64), ("cyc_backtrack", C.c_uint64)]

    CYC = ("cyc_stage", "cyc_levels", "cyc_level_barrier", "cyc_grid_wait", "cyc_scheduler", "cyc_backtrack")


RESULT_BYTES = C.sizeof(TgResult)
RESULT_DTYPE = np.dtype([("iter_time_us", "<i8"), ("sum_us", "<i8"), ("bottleneck_us", "<i4"), ("n_stages", "<i4"),
                         ("island_mask", "<u4"), ("n_thresholds_run", "<u4"), ("stage_begin", "<i4", (TG_MAX_K,)),
                         ("stage_island", "<i4", (TG_MAX_K,)), ("stage_plan", "<i4", (TG_MAX_K,))])
assert RESULT_DTYPE.itemsize == RESULT_BYTES == 224


class TangramError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{STATUS.get(status, status)}: {msg}")
        self.status = status


_lib = None
EXPORTS = ["tg_instance_create", "tg_instance_create_classes", "tg_instance_create_batch", "tg_instance_set_actmem", "tg_instance_set_transfer_bound", "tg_instance_set_boundary_act", "tg_instance_set_stages", "tg_plan_pipeline_stages", "tg_instance_destroy", "tg_solve_batch", "tg_solve_batch_ex", "tg_prune", "tg_prune_batch", "tg_prune_batch_static",
           "tg_reduce", "tg_candidates", "tg_dp_at", "tg_instance_read_time", "tg_islands_build", "tg_release_cached_memory", "tg_last_solver_kernel_ms", "tg_last_loader_kernel_ms", "tg_last_error", "tg_version"]


def lib():
    """Loads libtangram.so; raises if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            # not a fallback: the same CUDA library, compiled on first use (nvcc, sm_100a); raises if that fails
            from . import build as _build
            _build.build()
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_16907_b200.build`")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64, u32 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint32
        L.tg_instance_create.argtypes = [i32, i32, i32, i32, vp, vp, vp, vp, vp, i32, C.POINTER(vp)]
        L.tg_instance_create_classes.argtypes = [i32, i32, i32, i32, i32, vp, vp, vp, vp, vp, vp, i32, C.POINTER(vp)]
        L.tg_instance_create_batch.argtypes = [i32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
        L.tg_instance_set_transfer_bound.argtypes = [vp, i32]
        L.tg_instance_set_stages.argtypes = [vp, vp, vp]
        L.tg_instance_set_boundary_act.argtypes = [vp, vp]
        L.tg_plan_pipeline_stages.argtypes = [vp, vp, C.POINTER(i32)]
        L.tg_instance_destroy.argtypes = [vp]
        L.tg_instance_set_actmem.argtypes = [vp, vp]
        L.tg_solve_batch.argtypes = [C.POINTER(vp), i32, vp, vp]
        L.tg_solve_batch_ex.argtypes = [C.POINTER(vp), i32, vp, u32, vp, vp]
        L.tg_prune.argtypes = [vp, C.c_int, i64, C.POINTER(i64), vp]
        L.tg_prune_batch.argtypes = [C.POINTER(vp), i32, C.c_int, i64, C.POINTER(i64), vp]
        L.tg_prune_batch_static.argtypes = [C.POINTER(vp), i32, C.c_int, i64, C.POINTER(i64), vp]
        L.tg_reduce.argtypes = [vp, vp, vp, vp, vp, C.POINTER(i32), vp]
        L.tg_candidates.argtypes = [vp, vp, i64, C.POINTER(i32), vp]
        L.tg_dp_at.argtypes = [vp, i64, vp, vp]
        L.tg_instance_read_time.argtypes = [vp, vp]
        L.tg_islands_build.argtypes = [i32, vp, vp, vp, vp, vp, i32, i32, i32, vp, C.POINTER(i32), vp, vp, vp]
        L.tg_last_solver_kernel_ms.argtypes = [C.POINTER(C.c_float)]
        L.tg_last_loader_kernel_ms.argtypes = [C.POINTER(C.c_float)]
        L.tg_last_error.restype = C.c_char_p
        L.tg_version.restype = i32
        for name in EXPORTS:
            if name not in ("tg_last_error", "tg_version"):
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def tg_last_error() -> str:
    return lib().tg_last_error().decode()


def tg_version() -> int:
    return lib().tg_version()


def _check(st: int):
    if st != 0:
        raise TangramError(st, tg_last_error())


def _ptr(a):
    """Address of a numpy array (host) or torch tensor (host or device); None -> NULL."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return a.ctypes.data
    if isinstance(a, int):
        return a
    assert a.is_contiguous()
    return a.data_ptr()


def _stream_ptr(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return stream if isinstance(stream, int) else stream.cuda_stream


class Instance:
    """Owner of one tg_instance handle."""

    def __init__(self, handle: int, L: int, K: int, P: int, m: int):
        self.handle, self.L, self.K, self.P, self.m = handle, L, K, P, m
        self.NS = L * (L + 1) // 2

    def destroy(self):
        if self.handle:
            lib().tg_instance_destroy(self.handle)
            self.handle = 0

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def tg_instance_create(L, K, P, m, time_us, mem_mb, island_gpus, island_cap_mb, bw_gbps, act_mb) -> Instance:
    """Tables: int32 numpy arrays (host) or int32 torch tensors (host or device), C-contiguous."""
    def prep(a):
        if isinstance(a, np.ndarray):
            return np.ascontiguousarray(a, dtype=np.int32)
        return a
    arrs = [prep(a) for a in (time_us, mem_mb, island_gpus, island_cap_mb, bw_gbps)]
    h = C.c_void_p(0)
    _check(lib().tg_instance_create(L, K, P, m, *[_ptr(a) for a in arrs], act_mb, C.byref(h)))
    return Instance(h.value, L, K, P, m)


def tg_instance_create_classes(L, K, P, m, class_of_slice, class_time_us, class_mem_mb, island_gpus, island_cap_mb,
                               bw_gbps, act_mb) -> Instance:
    """NEXT-3(a): tables per signature class ([NC,K,P]) and the class of every slice ([NS])."""
    def prep(a):
        return np.ascontiguousarray(a, dtype=np.int32) if isinstance(a, np.ndarray) else a
    arrs = [prep(a) for a in (class_of_slice, class_time_us, class_mem_mb, island_gpus, island_cap_mb, bw_gbps)]
    nc = int(arrs[1].shape[0])
    h = C.c_void_p(0)
    _check(lib().tg_instance_create_classes(L, K, P, m, nc, *[_ptr(a) for a in arrs], act_mb, C.byref(h)))
    return Instance(h.value, L, K, P, m)


def tg_instance_create_batch(specs) -> list:
    """specs: sequence of (L, K, P, m, time_us, mem_mb, island_gpus, island_cap_mb, bw_gbps, act_mb), tables as in
    tg_instance_create.  One synchronisation for the whole batch; all or nothing."""
    n = len(specs)
    if n == 0:
        return []
    def prep(a):
        return np.ascontiguousarray(a, dtype=np.int32) if isinstance(a, np.ndarray) else a
    keep = [[prep(a) for a in s[4:9]] for s in specs]           # keeps converted copies alive during the call
    I32 = C.c_int32 * n
    PP = C.c_void_p * n
    scal = [I32(*[int(s[j]) for s in specs]) for j in (0, 1, 2, 3)]
    acts = I32(*[int(s[9]) for s in specs])
    ptrs = [PP(*[_ptr(k[j]) for k in keep]) for j in range(5)]
    out = PP()
    _check(lib().tg_instance_create_batch(C.c_int32(n), *scal, *ptrs, acts, out))
    return [Instance(out[i], int(s[0]), int(s[1]), int(s[2]), int(s[3])) for i, s in enumerate(specs)]


def tg_instance_set_actmem(inst: Instance, actmem_mb):
    """NEXT-1: per-plan MB per in-flight microbatch ([NS,K,P] int32 numpy array or torch tensor); None removes it."""
    a = np.ascontiguousarray(actmem_mb, dtype=np.int32) if isinstance(actmem_mb, np.ndarray) else actmem_mb
    _check(lib().tg_instance_set_actmem(inst.handle, _ptr(a)))


def tg_instance_set_boundary_act(inst: Instance, act_mb_b):
    """NEXT-3(b): activation MB crossing boundary b ([L+1] int32; entries 1..L-1 used); None restores the scalar size."""
    a = np.ascontiguousarray(act_mb_b, dtype=np.int32) if isinstance(act_mb_b, np.ndarray) else act_mb_b
    _check(lib().tg_instance_set_boundary_act(inst.handle, _ptr(a)))


def tg_instance_set_stages(inst: Instance, slow_us, n_stages=None):
    """NEXT-2: slowest internal stage and internal stage count per entry ([NS,K,P] int32); slow_us None removes them."""
    a = np.ascontiguousarray(slow_us, dtype=np.int32) if isinstance(slow_us, np.ndarray) else slow_us
    q = np.ascontiguousarray(n_stages, dtype=np.int32) if isinstance(n_stages, np.ndarray) else n_stages
    _check(lib().tg_instance_set_stages(inst.handle, _ptr(a), _ptr(q)))


def tg_plan_pipeline_stages(inst: Instance, result) -> int:
    """Total pipeline stages of a plan: `result` is a TgResult or one record of the RESULT_DTYPE array."""
    if isinstance(result, TgResult):
        r = result
    else:
        r = TgResult.from_buffer_copy(np.asarray(result).tobytes())
    n = C.c_int32(0)
    _check(lib().tg_plan_pipeline_stages(inst.handle, C.addressof(r), C.byref(n)))
    return n.value


def tg_instance_set_transfer_bound(inst: Instance, on: bool):
    """NEXT-3(b): transfers count toward the bottleneck (x <= T as well)."""
    _check(lib().tg_instance_set_transfer_bound(inst.handle, C.c_int32(1 if on else 0)))


def tg_instance_destroy(inst: Instance):
    inst.destroy()


def _handles(instances):
    arr = (C.c_void_p * len(instances))(*[i.handle for i in instances])
    return arr


def tg_solve_batch(instances, out=None, stream=None, flags: int = TG_SOLVE_DEFAULT, stats=None):
    """Solves the batch.  `out`: a uint8 CUDA tensor of len(instances)*224 bytes (asynchronous on
    `stream`), or None for a host result array (synchronous).  Returns `out`, or a numpy structured
    array of RESULT_DTYPE when out is None.  `stats`: optional TgSolveStats (host: filled on return, the call then
    synchronises) or a uint8 CUDA tensor of at least sizeof(TgSolveStats) bytes (written asynchronously on `stream`; read it
    with stats_from_tensor after synchronising)."""
    n = len(instances)
    h = _handles(instances)
    sp = _stream_ptr(stream)
    host = None
    if out is None:
        host = np.zeros(n, dtype=RESULT_DTYPE)
        optr = host.ctypes.data
    else:
        optr = _ptr(out)
    sptr = None if stats is None else (C.addressof(stats) if isinstance(stats, TgSolveStats) else _ptr(stats))
    _check(lib().tg_solve_batch_ex(h, n, optr, flags, sptr, sp))
    return host if out is None else out


def stats_from_tensor(t) -> "TgSolveStats":
    """TgSolveStats from the device buffer a tg_solve_batch(..., stats=<CUDA tensor>) call wrote (after synchronising)."""
    return TgSolveStats.from_buffer_copy(bytes(t[:C.sizeof(TgSolveStats)].cpu().numpy().tobytes()))


def tg_solve_batch_ex(instances, out, flags, stats, stream=None):
    return tg_solve_batch(instances, out, stream, flags, stats)


def tg_dp_at(inst: Instance, T: int, stream=None) -> TgResult:
    r = TgResult()
    _check(lib().tg_dp_at(inst.handle, T, C.addressof(r), _stream_ptr(stream)))
    return r


def tg_reduce(inst: Instance, stream=None):
    """-> c [NS,K] int32 (2^30 none), argp [NS,K] int32 (-1 none), x [K,K] int32, candidates int32[]"""
    c = np.empty((inst.NS, inst.K), dtype=np.int32)
    argp = np.empty((inst.NS, inst.K), dtype=np.int32)
    x = np.empty((inst.K, inst.K), dtype=np.int32)
    cand = np.empty(inst.NS * inst.K, dtype=np.int32)
    n = C.c_int32(0)
    _check(lib().tg_reduce(inst.handle, c.ctypes.data, argp.ctypes.data, x.ctypes.data, cand.ctypes.data,
                           C.byref(n), _stream_ptr(stream)))
    return c, argp, x, cand[:min(n.value, cand.size)].copy()


def tg_candidates(inst: Instance, stream=None) -> np.ndarray:
    """The instance's candidate thresholds as the solver sees them (all depths, transfer times under the bound)."""
    n = C.c_int32(0)
    _check(lib().tg_candidates(inst.handle, None, 0, C.byref(n), _stream_ptr(stream)))
    cand = np.empty(max(n.value, 1), dtype=np.int32)
    _check(lib().tg_candidates(inst.handle, cand.ctypes.data, cand.size, C.byref(n), _stream_ptr(stream)))
    return cand[:n.value].copy()


def tg_prune(inst: Instance, mode: int = TG_PRUNE_EXACT, threshold: int = 0, stream=None) -> np.ndarray:
    counts = (C.c_int64 * 4)()
    _check(lib().tg_prune(inst.handle, mode, threshold, counts, _stream_ptr(stream)))
    return np.array(list(counts), dtype=np.int64)


def tg_prune_batch(instances, mode: int = TG_PRUNE_EXACT, threshold: int = 0, stream=None) -> np.ndarray:
    """tg_prune over distinct instances in one pass; returns counts [n, 4]."""
    n = len(instances)
    counts = (C.c_int64 * (4 * max(n, 1)))()
    _check(lib().tg_prune_batch(_handles(instances), n, mode, threshold, counts, _stream_ptr(stream)))
    return np.array(list(counts), dtype=np.int64)[:4 * n].reshape(n, 4)


TG_PRUNE_STATIC_MAX_N = 1024


def tg_prune_batch_static(instances, mode: int = TG_PRUNE_EXACT, threshold: int = 0, stream=None) -> np.ndarray:
    """tg_prune_batch without any device allocation: scratch in the library's file-scope device array; at most
    TG_PRUNE_STATIC_MAX_N instances.  Returns counts [n, 4]."""
    n = len(instances)
    counts = (C.c_int64 * (4 * max(n, 1)))()
    _check(lib().tg_prune_batch_static(_handles(instances), n, mode, threshold, counts, _stream_ptr(stream)))
    return np.array(list(counts), dtype=np.int64)[:4 * n].reshape(n, 4)


def tg_islands_build(node_gpus, node_compute, node_mem_mb, node_intra_bw, inter_bw, eps_c: int, eps_m: int, eps_i: int):
    """NEXT-4: islands from per-node profiles.  Returns (island_of_node [N], island_gpus [K], island_cap_mb [K], bw [K,K])."""
    g, c, mm, ib = (np.ascontiguousarray(a, dtype=np.int32) for a in (node_gpus, node_compute, node_mem_mb, node_intra_bw))
    e = np.ascontiguousarray(inter_bw, dtype=np.int32)
    n = g.size
    of, ig, ic, bw = (np.zeros(n, np.int32), np.zeros(n, np.int32), np.zeros(n, np.int32), np.zeros(n * n, np.int32))
    k = C.c_int32(0)
    _check(lib().tg_islands_build(n, g.ctypes.data, c.ctypes.data, mm.ctypes.data, ib.ctypes.data, e.ctypes.data, eps_c, eps_m, eps_i,
                                  of.ctypes.data, C.byref(k), ig.ctypes.data, ic.ctypes.data, bw.ctypes.data))
    return of, ig[:k.value].copy(), ic[:k.value].copy(), bw[:k.value * k.value].reshape(k.value, k.value).copy()


def tg_release_cached_memory():
    _check(lib().tg_release_cached_memory())


def tg_instance_read_time(inst: Instance) -> np.ndarray:
    t = np.empty((inst.NS, inst.K, inst.P), dtype=np.int32)
    _check(lib().tg_instance_read_time(inst.handle, t.ctypes.data))
    return t


def tg_last_solver_kernel_ms() -> float:
    ms = C.c_float(0)
    _check(lib().tg_last_solver_kernel_ms(C.byref(ms)))
    return ms.value


def tg_last_loader_kernel_ms() -> float:
    ms = C.c_float(0)
    _check(lib().tg_last_loader_kernel_ms(C.byref(ms)))
    return ms.value


def results_from_tensor(out, n: int) -> np.ndarray:
    """Device result tensor -> numpy structured array (synchronises)."""
    return np.frombuffer(out.cpu().numpy().tobytes(), dtype=RESULT_DTYPE, count=n)


def instance_from_inputs(inst, device_tables: bool = False) -> Instance:
    """Convenience: build from a tg_inputs.Instance-like object (fields L,K,P,m,time_us,...)."""
    if device_tables:
        import torch
        t = torch.from_numpy(np.ascontiguousarray(inst.time_us, dtype=np.int32)).cuda()
        mm = torch.from_numpy(np.ascontiguousarray(inst.mem_mb, dtype=np.int32)).cuda()
        return tg_instance_create(inst.L, inst.K, inst.P, inst.m, t, mm, inst.island_gpus, inst.island_cap_mb,
                                  inst.bw_gbps, inst.act_mb)
    h = tg_instance_create(inst.L, inst.K, inst.P, inst.m, inst.time_us, inst.mem_mb, inst.island_gpus,
                           inst.island_cap_mb, inst.bw_gbps, inst.act_mb)
    if getattr(inst, "actmem_mb", None) is not None:
        tg_instance_set_actmem(h, inst.actmem_mb)
    if getattr(inst, "transfer_bound", False):
        tg_instance_set_transfer_bound(h, True)
    if getattr(inst, "act_mb_b", None) is not None:
        tg_instance_set_boundary_act(h, inst.act_mb_b)
    if getattr(inst, "slow_us", None) is not None:
        tg_instance_set_stages(h, inst.slow_us, getattr(inst, "q_stages", None))
    return h
