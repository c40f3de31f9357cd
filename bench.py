#!/usr/bin/env python
"""bench.py — throughput of the TANGRAM composition search on B200 (contract: see DESIGN.md §Measurement).

A step = one tg_solve_batch over the workload's synthetic instances (whole hot path: loader,
candidate thresholds, DP at T=inf, windowed per-T wavefront DPs, sweep reduction, back-track).
metric  = slice/island plans evaluated per second, "plans evaluated" of one DP(T) being the dense
          relaxation count NS*K*2^(K-1), summed over the DPs the solver ran.
value   = device-timed (CUDA events on the launching stream), instances resident in HBM.
e2e     = same metric through the C ABI with HOST tables: tg_instance_create (H2D) + tg_solve_batch
          with a host result buffer (D2H) inside the timed region.
roofline= the persistent solver kernel: algorithmic bytes (every live DP state written once and read
          once, 8 B per state) / its own event-timed duration, against the measured HBM copy peak.
`--impl reference` times the CPU oracle (oracle/, test infrastructure) on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "slice_island_plans_evaluated_per_sec"
UNIT = "plans/s"


# dram__bytes_read.sum + dram__bytes_write.sum of ONE tgSolveKernel launch from the committed ncu capture
# (profiles/); only valid for the windowed run of the workload as captured (cfg5: 1024 instances)
NCU_TRAFFIC_BYTES = {("cfg4", False): (0.170e9, "profiles/r1c_ncu_cfg4_solver.md"),
                     ("cfg5", False): (1.341e9, "profiles/r1c_ncu_cfg5_solver.md")}


def make_workload(name: str, rank: int, n_inst: int, n_make: int = None):
    """Seeded synthetic instances (DESIGN.md input recipe).  Rank r takes its own seeds (weak scaling).
    n_make: build only the first n_make instances of the workload (the CPU arm's bounded sample); the
    description stays that of the whole workload."""
    import tg_inputs as gen
    if name == "cfg4":
        return [gen.config4(rank)], "cfg4 MoE-like L=64 K=16 P=8 m=64 (BASELINE.json configs[3]), 1 instance/GPU"
    if name == "cfg3":
        return [gen.config3(rank)], "cfg3 70B-like L=80 K=12 P=8 m=32 (configs[2]), 1 instance/GPU"
    if name == "cfg2":
        return [gen.config2(rank)], "cfg2 7B-like L=32 K=6 P=4 m=16 (configs[1]), 1 instance/GPU"
    if name == "cfg4d":   # cfg4 with a per-plan activation footprint
        return [gen.with_actmem(gen.config4(rank), 11 + rank, 300, 3000)], \
            "cfg4 MoE-like L=64 K=16 P=8 m=64 + depth-aware activation memory (NEXT-1), 1 instance/GPU"
    if name == "cfg3d":
        return [gen.with_actmem(gen.config3(rank), 7 + rank, 500, 6000)], \
            "cfg3 70B-like L=80 K=12 P=8 m=32 + depth-aware activation memory (NEXT-1), 1 instance/GPU"
    if name == "cfg4xb":  # cfg4 with the boundary transfers bounded by the threshold
        return [gen.with_transfer_bound(gen.config4(rank))], \
            "cfg4 MoE-like L=64 K=16 P=8 m=64 + transfers as pipeline slots (NEXT-3(b)), 1 instance/GPU"
    if name == "cfg3xb":
        return [gen.with_transfer_bound(gen.config3(rank))], \
            "cfg3 70B-like L=80 K=12 P=8 m=32 + transfers as pipeline slots (NEXT-3(b)), 1 instance/GPU"
    if name == "cfg5":
        from paper_2606_16907_b200.shard import weak_seeds
        return [gen.config5_one(sd) for sd in weak_seeds(n_inst, rank)[:n_make]], \
            f"cfg5 throughput batch: {n_inst} instances L=48 K=10 P=4 m in {{4..64}} (configs[4]) per GPU"
    raise SystemExit(f"unknown workload {name}")


def dense_plans(inst) -> int:
    return inst.L * (inst.L + 1) // 2 * inst.K * (1 << (inst.K - 1))


class ClockSampler:
    """SM clocks and throttle reasons sampled during the timed region (profiling recipe's clocks line).
    Sampled in-process through NVML (the library nvidia-smi itself queries): spawning nvidia-smi ten times a
    second from a thread of the timed process stalled the launching thread for tens of ms now and then.
    Falls back to the nvidia-smi command line when the NVML binding is not importable."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
    BITS = [("hw_slowdown", 0x8), ("hw_thermal_slowdown", 0x40), ("sw_thermal_slowdown", 0x20), ("sw_power_cap", 0x4)]

    def __init__(self, index: int):
        self.rows, self.stop, self.index = [], threading.Event(), index
        self.active = threading.Event()      # set while the timed region runs: only those samples are kept
        self.nvml = self.handle = None
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            try:
                self.handle = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + str(torch.cuda.get_device_properties(index).uuid)).encode())
            except Exception:
                self.handle = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.reasons_fn = getattr(pynvml, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
                pynvml.nvmlDeviceGetCurrentClocksThrottleReasons
            self.max_sm = int(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
            self.nvml = pynvml
        except Exception:
            self.nvml = None
        self.th = threading.Thread(target=self._run, daemon=True)
        self.th.start()                      # started before the warm-up: the first queries initialise driver state and are slow

    def _sample_nvml(self):
        n = self.nvml
        sm = int(n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM))
        mask = int(self.reasons_fn(self.handle))
        self.rows.append([str(sm), str(self.max_sm)] + ["Active" if mask & bit else "Not Active" for _, bit in self.BITS])

    def _sample_smi(self):
        o = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                            "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout.strip()
        if o:
            self.rows.append([c.strip() for c in o.splitlines()[0].split(",")])

    def _run(self):
        while not self.stop.is_set():
            try:
                if self.nvml is not None:
                    self._sample_nvml()
                else:
                    self._sample_smi()
            except Exception:
                pass
            if not self.active.is_set():
                self.rows.clear()            # priming samples outside the timed region are dropped
            self.stop.wait(0.05 if self.nvml is not None else 0.25)

    def __enter__(self):
        self.rows.clear()
        self.active.set()
        return self

    def __exit__(self, *a):
        try:
            if self.nvml is not None and not self.rows:
                self._sample_nvml()          # a timed region shorter than the sampling period: sample before it closes
        except Exception:
            pass
        self.active.clear()
        self.stop.set()
        self.th.join(timeout=6)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["clock query unavailable"]}
        sm = sorted(int(r[0]) for r in self.rows if r[0].isdigit())
        names = [n for n, _ in self.BITS]
        reasons = [n for i, n in enumerate(names) if any(r[2 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": int(self.rows[0][1]) if self.rows[0][1].isdigit() else None,
                "reasons": reasons, "samples": len(self.rows), "source": "nvml" if self.nvml is not None else "nvidia-smi"}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def oracle_sample(insts, workload: str, threads: int, seconds: float = 10.0):
    """Bounded sample of the workload on the CPU oracle, as it stands: `threads` host threads run single DP(T)
    calls (oracle.dp_at releases the GIL inside the C++ library) over thresholds spread over the upper half of the
    candidate lists (feasible region) of the first instances, until about `seconds` of wall time have passed
    (every thread finishes the DP it is in; at least one DP per thread).  Returns (plans, seconds, text)."""
    import oracle
    sample_insts = insts[:min(len(insts), 4)]
    work = []                                        # (instance, T) in a fixed order: thread i takes i, i+threads, ...
    for inst in sample_insts:
        _, _, _, cand = oracle.reduce(inst)
        half = len(cand) // 2
        work.append([(inst, int(cand[half + (i * (half - 1)) // max(1, threads - 1)])) for i in range(threads)])
    done = [0.0] * threads
    t0 = time.perf_counter()

    def worker(i):
        r = 0
        while True:
            inst, T = work[r % len(work)][(i + r // len(work)) % threads]
            oracle.dp_at(inst, T, False)
            done[i] += dense_plans(inst)
            r += 1
            if time.perf_counter() - t0 >= seconds:
                return

    ths = [threading.Thread(target=worker, args=(i,)) for i in range(threads)]
    for t in ths:
        t.start()
    for t in ths:
        t.join()
    dt = time.perf_counter() - t0
    n_dp = sum(round(d / dense_plans(sample_insts[0])) for d in done)
    return sum(done), dt, (f"{n_dp} single-threshold DPs (oracle.dp_at) over {len(sample_insts)} instance(s) from {sample_insts[0].name}, "
                           f"{threads} threads, {dt:.1f} s of wall time")


def run_reference(args):
    """Reference arm = the CPU oracle (this tier has no reference implementation)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    insts, desc = make_workload(args.workload, 0, args.n_inst, 4)
    cores = max(1, min(oracle.hw_threads(), args.cpu_threads))
    per_step = max(2.0, min(10.0, 100.0 / max(1, args.steps)))        # the whole run stays within a few minutes
    for _ in range(min(args.warmup, 1)):
        oracle_sample(insts, args.workload, cores, 1.0)
    plans = secs = 0.0
    sample = ""
    for _ in range(args.steps):
        p, dt, sample = oracle_sample(insts, args.workload, cores, per_step)
        plans += p
        secs += dt
    v = plans / secs
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": min(args.warmup, 1), "ms_per_step": secs / args.steps * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": {"workload": desc, "l2": "n/a (CPU)"},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2606_16907_b200 as tg
    tg.lib()  # fail loudly if the CUDA library is missing
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    insts, desc = make_workload(args.workload, rank, args.n_inst)
    n = len(insts)
    stream = torch.cuda.current_stream()
    flags = tg.TG_SOLVE_FULL_SWEEP if args.full_sweep else tg.TG_SOLVE_DEFAULT
    handles = [tg.instance_from_inputs(i) for i in insts]            # resident in HBM
    out = torch.empty(n * tg.RESULT_BYTES, dtype=torch.uint8, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2
    st = tg.TgSolveStats()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    clk = ClockSampler(local)
    def warm_step(w):                                                 # the warm-up steps are the timed steps, untimed
        flush.fill_(w & 0xff)
        tg.tg_solve_batch(handles, out=out, flags=flags, stats=st)
        torch.cuda.synchronize()

    for w in range(args.warmup - 1):
        warm_step(w)
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kern_ms, load_ms, plans, states, n_dp = [], [], 0, 0, 0
    cyc = [0] * 8
    relax = 0
    with clk:
        if args.warmup > 0:
            warm_step(args.warmup - 1)                                # last warm-up step with the clock sampler already running
        for s in range(args.steps):
            flush.fill_(s & 0xff)                                     # evict L2 between timed steps
            ev[s][0].record(stream)
            tg.tg_solve_batch(handles, out=out, flags=flags, stats=st)   # stats on host => synchronises
            ev[s][1].record(stream)
            torch.cuda.synchronize()
            kern_ms.append(tg.tg_last_solver_kernel_ms())
            load_ms.append(tg.tg_last_loader_kernel_ms())
            plans += st.plans_dense
            states += st.states_live
            n_dp += st.n_dp
            assert st.error_flag == 0, "solver error flag"
            cyc = [c + int(v) for c, v in zip(cyc, st.cyc)]
            relax += int(st.relax_admissible)
        barrier()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = sum(step_ms)
    # ---- end to end: host tables -> create (H2D) -> solve -> host results (D2H) ----
    h2d = sum(i.time_us.nbytes + i.mem_mb.nbytes + i.bw_gbps.nbytes + 8 * i.K +
              (i.actmem_mb.nbytes if i.actmem_mb is not None else 0) for i in insts)
    d2h = n * tg.RESULT_BYTES
    e2e_steps = max(1, min(args.steps, 3))
    # inputs of the end-to-end leg wait in PINNED host memory
    pinned = [[torch.from_numpy(np.ascontiguousarray(a, dtype=np.int32)).pin_memory()
               for a in (i.time_us, i.mem_mb, i.island_gpus, i.island_cap_mb, i.bw_gbps)] for i in insts]
    pinned_act = [torch.from_numpy(np.ascontiguousarray(i.actmem_mb, dtype=np.int32)).pin_memory()
                  if i.actmem_mb is not None else None for i in insts]
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        hs = tg.tg_instance_create_batch([(i.L, i.K, i.P, i.m, *pp, i.act_mb) for i, pp in zip(insts, pinned)])
        for h, pa, i in zip(hs, pinned_act, insts):
            if pa is not None:
                tg.tg_instance_set_actmem(h, pa)
            if i.transfer_bound:
                tg.tg_instance_set_transfer_bound(h, True)
        res = tg.tg_solve_batch(hs, out=None, flags=flags)            # host result buffer: D2H + sync inside
        for h in hs:
            h.destroy()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    prune_info = None
    if args.with_prune:
        # step 0 of the path, outside every timed region above: tg_prune_batch(EXACT) once on a fresh copy of the
        # workload (the pass mutates its instances); wall clock of the call, which synchronises
        hs = tg.tg_instance_create_batch([(i.L, i.K, i.P, i.m, *pp, i.act_mb) for i, pp in zip(insts, pinned)])
        for h, pa in zip(hs, pinned_act):
            if pa is not None:
                tg.tg_instance_set_actmem(h, pa)
        flush.fill_(1)
        torch.cuda.synchronize()
        tp = time.perf_counter()
        killed = tg.tg_prune_batch(hs, tg.TG_PRUNE_EXACT, 0)
        prune_ms = (time.perf_counter() - tp) * 1e3
        for h in hs:
            h.destroy()
        prune_info = {"call": "tg_prune_batch(EXACT)", "wall_ms": prune_ms, "killed_r1_r2": killed.sum(0)[:2].tolist(),
                      "entries": int(sum(i.time_us.size for i in insts))}
    from paper_2606_16907_b200.shard import aggregate
    (plans_all, plans_e2e, ndp_all), (total_ms, e2e_s) = aggregate(
        [float(plans), float(plans) / args.steps * e2e_steps, float(n_dp)], [total_ms, e2e_s], device="cuda")
    if rank == 0:
        peak, peak_src = peaks()
        km = sum(kern_ms) / len(kern_ms)
        alg_bytes = states / args.steps * 8.0                          # live state: 4 B written + 4 B read
        achieved = alg_bytes / (km * 1e-3) / 1e9
        inst0 = insts[0]
        load_bytes = sum(i.time_us.shape[0] * i.K * ((12 * i.P + 9 * i.K) if i.actmem_mb is not None else (8 * i.P + 9)) for i in insts)
        ncu_traffic = NCU_TRAFFIC_BYTES.get((args.workload, args.full_sweep), (None, None))
        if args.workload == "cfg5" and n != 1024:
            ncu_traffic = (None, None)
        line = {"metric": METRIC, "value": plans_all / (total_ms * 1e-3), "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_ms / args.steps,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
                "config": {"workload": desc, "sweep": "full" if args.full_sweep else "exact branch-and-bound over thresholds",
                           "l2": "256 MB buffer written between timed steps", "instances_per_gpu": n,
                           "dps_per_step": ndp_all / args.steps / world,
                           "planning_ms_per_instance": total_ms / args.steps / n},
                "clocks": clk.summary(),
                "e2e": {"value": plans_e2e / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                        "ms_per_step": e2e_s / e2e_steps * 1e3},
                "gpu_launches": 3 * args.steps,   # tgLoadKernel + tgPrepareKernel + tgSolveKernel per tg_solve_batch
                "roofline": {"bound": "hbm", "kernel": "tgSolveKernel", "achieved": achieved, "peak": peak, "unit": "GB/s",
                             "frac": achieved / peak, "traffic": ncu_traffic[0], "traffic_source": ncu_traffic[1],
                             "peak_source": peak_src,
                             "kernel_ms": km, "step_ms": [round(x, 3) for x in step_ms],
                             "kernel_ms_steps": [round(x, 3) for x in kern_ms],
                             "algorithmic_bytes_per_launch": alg_bytes,
                             "us_per_dp": km * 1e3 / (n_dp / args.steps),
                             "alu": {"relaxations_per_launch": relax / args.steps,
                                     "achieved_Trelax_s": relax / args.steps / (km * 1e-3) / 1e12,
                                     "peak_Trelax_s": 148 * 64 * 1.965e9 / 1e12,
                                     "frac": relax / args.steps / (km * 1e-3) / (148 * 64 * 1.965e9)},
                             # step 1 of the path (cost-table loader): 8*P bytes read and 9 bytes written per (slice, island) cell
                             "loader": {"kernel": "tgLoadKernel", "kernel_ms": sum(load_ms) / len(load_ms),
                                        "algorithmic_bytes_per_launch": float(load_bytes),
                                        "achieved": load_bytes / (sum(load_ms) / len(load_ms) * 1e-3) / 1e9, "unit": "GB/s",
                                        "frac": load_bytes / (sum(load_ms) / len(load_ms) * 1e-3) / 1e9 / peak,
                                        "note": "a few MB: bound by launch latency, not by HBM" if load_bytes < (32 << 20) else "HBM stream"},
                             "cta_cycle_shares": dict(zip(["stage", "unused1", "unused2", "dp_levels", "level_barrier_wait",
                                                           "grid_wait", "scheduler", "backtrack"],
                                                          [round(c / max(1, sum(cyc)), 4) for c in cyc]))}}
        if prune_info is not None:
            line["prune"] = prune_info
        if not args.no_cpu_baseline:
            import oracle
            cores = max(1, min(oracle.hw_threads(), args.cpu_threads))
            p, dt, sample = oracle_sample(insts, args.workload, cores)
            line["cpu_baseline"] = {"value": p / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                                    "seconds": dt}
        print(json.dumps(line), flush=True)
    for h in handles:
        h.destroy()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4", choices=["cfg2", "cfg3", "cfg4", "cfg5", "cfg3d", "cfg4d", "cfg3xb", "cfg4xb"])
    ap.add_argument("--n-inst", type=int, default=1024, help="instances per GPU of the cfg5 batch")
    ap.add_argument("--full-sweep", action="store_true", help="run the DP at every candidate T")
    ap.add_argument("--cpu-threads", type=int, default=8)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--with-prune", action="store_true", help="also run tg_prune_batch once on a fresh copy of the workload (untimed legs unchanged)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
