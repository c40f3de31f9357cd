#!/usr/bin/env python
"""bench.py — throughput of the TANGRAM composition search on B200 (contract: see DESIGN.md §Measurement).

A step = one tg_solve_batch over the workload's synthetic instances (whole hot path: loader, transfer table, candidate
thresholds, exact threshold search, per-T wavefront DPs, sweep reduction, back-track).
metric   = slice/island plans evaluated per second, "plans evaluated" of one DP(T) being the dense relaxation count
           NS*K*2^(K-1), summed over the DPs the solver ran.
value    = device-timed (CUDA events on the launching stream), instances resident in HBM; headline workload cfg4 (the
           config north_star's roofline target is quoted on).
config.secondary = the 1024-instance batch (cfg5) measured in the same run: planning time per instance, its own
           roofline, loader roofline and end-to-end leg (the other half of BASELINE.json's metric).
e2e      = same metric through the C ABI with pinned HOST tables: tg_instance_create_batch (H2D) + tg_solve_batch with a
           host result buffer (D2H) inside the timed region; a large batch goes up in sub-batches whose upload overlaps
           the previous sub-batch's solve; one untimed end-to-end step first (the upload path has first-call costs).
roofline = the persistent solver kernel against what binds it: admissible add-min relaxations per second (counted by
           the kernel) over the integer-ALU peak; the dense-table byte figure of SURVEY §8(d) is kept as
           hbm_algorithmic_frac, next to the DRAM fraction ncu measured (nulled when the kernels changed since).
verified = the last timed step's results equal the stored oracle results (tests/golden/), value and plan.
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


def kernel_sources_sha() -> str:
    """Fingerprint of the solver kernel's sources (tg_solve.cuh, tg_common.cuh): an ncu figure of that kernel is quoted only
    while they are the ones that were profiled."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2606_16907_b200", "csrc")
    for f in ("tg_common.cuh", "tg_solve.cuh"):
        with open(os.path.join(d, f), "rb") as fh:
            h.update(f.encode() + b"\0" + fh.read())
    return h.hexdigest()[:16]


def ncu_traffic(workload: str, n_inst: int, full_sweep: bool):
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE tgSolveKernel launch, from the committed ncu capture listed in
    profiles/ncu_traffic.json (written beside the capture, with the fingerprint of the kernel sources at that time).
    Returns (bytes, source) -- (None, why) when there is no capture of this workload or the kernels changed since."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    if full_sweep or not os.path.exists(p):
        return None, "no ncu capture of this configuration"
    with open(p) as f:
        rec = json.load(f).get(workload)
    if rec is None or (workload == "cfg5" and n_inst != rec.get("instances", 1024)):
        return None, "no ncu capture of this configuration"
    if rec["kernel_sources_sha"] != kernel_sources_sha():
        return None, f"stale: {rec['source']} was captured with other kernel sources ({rec['kernel_sources_sha']})"
    return float(rec["dram_bytes_per_launch"]), rec["source"]


GOLDEN = {"cfg3": "expected_cfg3.json", "cfg4": "expected_cfg4.json", "cfg5": "expected_cfg5.json", "cfg3d": "expected_cfg3d.json",
          "cfg4d": "expected_cfg4d.json", "cfg3xb": "expected_cfg3xb.json", "cfg4xb": "expected_cfg4xb.json"}


def golden_records(workload: str):
    """Stored oracle results of the workload (tests/golden/, written by make_expected.py from oracle/ only): seed -> solve."""
    f = GOLDEN.get(workload)
    p = os.path.join(ROOT, "tests", "golden", f) if f else None
    if not p or not os.path.exists(p):
        return {}
    with open(p) as fh:
        recs = json.load(fh)["records"]
    return {int(r.get("seed", 0)): r["solve"] for r in recs}


def verify_results(workload: str, seeds, res) -> object:
    """Compares what the timed steps returned with the stored oracle results (value and plan).  True / False, or a
    string when no stored result covers these seeds (other ranks of a weak-scaling run)."""
    gold = golden_records(workload)
    if not gold or any(sd not in gold for sd in seeds):
        return "no stored oracle result for these seeds"
    for sd, g in zip(seeds, res):
        e = gold[sd]
        n = int(g["n_stages"])
        got = [int(g["iter_time_us"]), int(g["sum_us"]), int(g["bottleneck_us"]), int(g["island_mask"]),
               [[int(g["stage_begin"][i]), int(g["stage_island"][i]), int(g["stage_plan"][i])] for i in range(n)]]
        if got != [e["iter_time_us"], e["sum_us"], e["bottleneck_us"], e["island_mask"], e["stages"]]:
            return False
    return True


def make_workload(name: str, rank: int, n_inst: int, n_make: int = None):
    """Seeded synthetic instances (DESIGN.md input recipe).  Rank r takes its own seeds (weak scaling).
    n_make: build only the first n_make instances of the workload (the CPU arm's bounded sample); the
    description stays that of the whole workload.  Returns (instances, description, seeds)."""
    import tg_inputs as gen
    if name == "cfg4":
        return [gen.config4(rank)], "cfg4 MoE-like L=64 K=16 P=8 m=64 (BASELINE.json configs[3]), 1 instance/GPU", [rank]
    if name == "cfg3":
        return [gen.config3(rank)], "cfg3 70B-like L=80 K=12 P=8 m=32 (configs[2]), 1 instance/GPU", [rank]
    if name == "cfg2":
        return [gen.config2(rank)], "cfg2 7B-like L=32 K=6 P=4 m=16 (configs[1]), 1 instance/GPU", [rank]
    if name == "cfg4d":   # cfg4 with a per-plan activation footprint
        return [gen.with_actmem(gen.config4(rank), 11 + rank, 300, 3000)], \
            "cfg4 MoE-like L=64 K=16 P=8 m=64 + depth-aware activation memory (NEXT-1), 1 instance/GPU", [rank]
    if name == "cfg3d":
        return [gen.with_actmem(gen.config3(rank), 7 + rank, 500, 6000)], \
            "cfg3 70B-like L=80 K=12 P=8 m=32 + depth-aware activation memory (NEXT-1), 1 instance/GPU", [rank]
    if name == "cfg4xb":  # cfg4 with the boundary transfers bounded by the threshold
        return [gen.with_transfer_bound(gen.config4(rank))], \
            "cfg4 MoE-like L=64 K=16 P=8 m=64 + transfers as pipeline slots (NEXT-3(b)), 1 instance/GPU", [rank]
    if name == "cfg3xb":
        return [gen.with_transfer_bound(gen.config3(rank))], \
            "cfg3 70B-like L=80 K=12 P=8 m=32 + transfers as pipeline slots (NEXT-3(b)), 1 instance/GPU", [rank]
    if name == "cfg5":
        from paper_2606_16907_b200.shard import weak_seeds
        seeds = list(weak_seeds(n_inst, rank))[:n_make]
        return [gen.config5_one(sd) for sd in seeds], \
            f"cfg5 throughput batch: {n_inst} instances L=48 K=10 P=4 m in {{4..64}} (configs[4]) per GPU", seeds
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
        self.entered = False                 # samples of every timed region of the run (headline and secondary) are kept
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
            if not self.active.is_set() and not self.entered:
                self.rows.clear()            # priming samples before the first timed region are dropped
            elif not self.active.is_set() and self.rows:
                self.rows.pop()              # between two timed regions: not part of either
            self.stop.wait(0.05 if self.nvml is not None else 0.25)

    def __enter__(self):
        if not self.entered:
            self.rows.clear()
            self.entered = True
        self.active.set()
        return self

    def __exit__(self, *a):
        try:
            if self.nvml is not None and not self.rows:
                self._sample_nvml()          # a timed region shorter than the sampling period: sample before it closes
        except Exception:
            pass
        self.active.clear()                  # (the sampler thread keeps running: a later timed region re-enters)

    def close(self):
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


def oracle_sample(insts, workload: str, seeds, threads: int, seconds: float = 10.0):
    """Bounded sample of the workload on the CPU oracle, as it stands: `threads` host threads run single DP(T)
    calls (oracle.dp_at releases the GIL inside the C++ library) until about `seconds` of wall time have passed (every
    thread finishes the DP it is in; at least one DP per thread).  The thresholds are the ones a search evaluates: candidates
    from 20 below to 200 above the optimum's bottleneck T* of the first instances (T* from the stored oracle result, the
    same region the GPU's branch and bound works in, so both sides meet the same admissible-edge density); without a
    stored result, the upper half of the candidate list.  Returns (plans, seconds, text)."""
    import oracle
    gold = golden_records(workload)
    sample_insts = insts[:min(len(insts), 4)]
    work, where = [], "upper half of the candidate list"
    for inst, sd in zip(sample_insts, seeds):
        _, _, _, cand = oracle.reduce(inst)
        if sd in gold and gold[sd].get("feasible", True) and getattr(inst, "actmem_mb", None) is None:
            star = int(np.searchsorted(cand, gold[sd]["bottleneck_us"]))
            lo, hi = max(0, star - 20), min(len(cand) - 1, star + 200)
            where = "candidates T*-20 .. T*+200 of the stored optimum"
        else:
            lo, hi = len(cand) // 2, len(cand) - 1
        work.append([(inst, int(cand[lo + (i * (hi - lo)) // max(1, threads - 1)])) for i in range(threads)])
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
    return sum(done), dt, (f"{n_dp} single-threshold DPs (oracle.dp_at, {where}) over {len(sample_insts)} instance(s) from "
                           f"{sample_insts[0].name}, {threads} threads, {dt:.1f} s of wall time")


def run_reference(args):
    """Reference arm = the CPU oracle (this tier has no reference implementation)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    insts, desc, seeds = make_workload(args.workload, 0, args.n_inst, 4)
    cores = max(1, min(oracle.hw_threads(), args.cpu_threads))
    per_step = max(2.0, min(10.0, 100.0 / max(1, args.steps)))        # the whole run stays within a few minutes
    for _ in range(min(args.warmup, 1)):
        oracle_sample(insts, args.workload, seeds, cores, 1.0)
    plans = secs = 0.0
    sample = ""
    for _ in range(args.steps):
        p, dt, sample = oracle_sample(insts, args.workload, seeds, cores, per_step)
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


ALU_PEAK = 148 * 64 * 1.965e9      # add-min per second: 148 SMs x 4 SMSPs x 16 int lanes x 1.965 GHz


def measure_workload(tg, torch, args, workload, rank, world, barrier, clk=None):
    """Times `args.steps` tg_solve_batch calls over the resident instances of one workload (after `args.warmup` untimed
    ones), checks the last step's results against the stored oracle results, and measures the end-to-end leg from pinned
    host tables.  Returns the rank's raw numbers."""
    import contextlib
    insts, desc, seeds = make_workload(workload, rank, args.n_inst)
    n = len(insts)
    stream = torch.cuda.current_stream()
    flags = tg.TG_SOLVE_FULL_SWEEP if args.full_sweep else tg.TG_SOLVE_DEFAULT
    handles = [tg.instance_from_inputs(i) for i in insts]            # resident in HBM
    out = torch.empty(n * tg.RESULT_BYTES, dtype=torch.uint8, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2
    st_dev = torch.zeros(256, dtype=torch.uint8, device="cuda")   # tg_solve_stats, written on the device: the timed call stays asynchronous

    def warm_step(w):                                                 # the warm-up steps are the timed steps, untimed
        flush.fill_(w & 0xff)
        tg.tg_solve_batch(handles, out=out, flags=flags, stats=st_dev)
        torch.cuda.synchronize()

    for w in range(args.warmup - 1):
        warm_step(w)
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    R = {"desc": desc, "n": n, "kern_ms": [], "load_ms": [], "plans": 0, "states_dense": 0, "states_windowed": 0, "n_dp": 0,
         "relax": 0, "cyc": [0] * len(tg.TgSolveStats.CYC), "global_c": 0}
    with (clk if clk is not None else contextlib.nullcontext()):
        if args.warmup > 0:
            warm_step(args.warmup - 1)                                # last warm-up step with the clock sampler already running
        for s in range(args.steps):
            flush.fill_(s & 0xff)                                     # evict L2 between timed steps
            ev[s][0].record(stream)
            tg.tg_solve_batch(handles, out=out, flags=flags, stats=st_dev)   # results and statistics stay on the device: no host round trip inside the timed region
            ev[s][1].record(stream)
            torch.cuda.synchronize()
            st = tg.stats_from_tensor(st_dev)
            R["kern_ms"].append(tg.tg_last_solver_kernel_ms())
            R["load_ms"].append(tg.tg_last_loader_kernel_ms())
            R["plans"] += st.plans_dense
            R["states_dense"] += st.states_live
            R["states_windowed"] += st.states_windowed
            R["n_dp"] += st.n_dp
            R["global_c"] += st.n_items_global_c
            assert st.error_flag == 0, "solver error flag"
            R["cyc"] = [c + int(getattr(st, f)) for c, f in zip(R["cyc"], tg.TgSolveStats.CYC)]
            R["relax"] += int(st.relax_admissible)
        barrier()
    R["step_ms"] = [a.elapsed_time(b) for a, b in ev]
    # the timed steps returned the right answer: last step's results against the stored oracle results (value and plan)
    R["verified"] = verify_results(workload, seeds, tg.results_from_tensor(out, n))
    # ---- end to end: pinned host tables -> create (H2D) -> solve -> host results (D2H), wall clock ----
    R["h2d"] = sum(i.time_us.nbytes + i.mem_mb.nbytes + i.bw_gbps.nbytes + 8 * i.K +
                   (i.actmem_mb.nbytes if i.actmem_mb is not None else 0) for i in insts)
    R["d2h"] = n * tg.RESULT_BYTES
    R["e2e_steps"] = max(1, min(args.steps, 3))
    pinned = [[torch.from_numpy(np.ascontiguousarray(a, dtype=np.int32)).pin_memory()
               for a in (i.time_us, i.mem_mb, i.island_gpus, i.island_cap_mb, i.bw_gbps)] for i in insts]
    pinned_act = [torch.from_numpy(np.ascontiguousarray(i.actmem_mb, dtype=np.int32)).pin_memory()
                  if i.actmem_mb is not None else None for i in insts]

    def create(lo, hi):
        hs = tg.tg_instance_create_batch([(i.L, i.K, i.P, i.m, *pp, i.act_mb) for i, pp in zip(insts[lo:hi], pinned[lo:hi])])
        for h, pa, i in zip(hs, pinned_act[lo:hi], insts[lo:hi]):
            if pa is not None:
                tg.tg_instance_set_actmem(h, pa)
            if i.transfer_bound:
                tg.tg_instance_set_transfer_bound(h, True)
        return hs

    # a large batch goes up in sub-batches: while one is solved (on a side stream) the next one's tables are uploaded by
    # a second host thread (the uploads run on the legacy default stream, the side stream does not synchronise with it)
    n_sub = args.e2e_sub if n >= 64 * args.e2e_sub else 1
    cuts = [(q * n) // n_sub for q in range(n_sub + 1)]
    side = torch.cuda.Stream()
    e2e_res = None
    e2e_warm = 1 if args.warmup > 0 else 0   # the upload path has its own first-call costs (pool growth, module loading: 70-1000 ms once)
    for it in range(e2e_warm + R["e2e_steps"]):
        if it == e2e_warm:
            torch.cuda.synchronize()
            barrier()
            t0 = time.perf_counter()
        parts, made = [], [None]
        nxt = create(cuts[0], cuts[1])
        for q in range(n_sub):
            hs, th = nxt, None
            if q + 1 < n_sub:
                th = threading.Thread(target=lambda a=cuts[q + 1], b=cuts[q + 2]: made.__setitem__(0, create(a, b)))
                th.start()
            parts.append(tg.tg_solve_batch(hs, out=None, flags=flags, stream=side))   # host result buffer: D2H + sync inside
            if th is not None:
                th.join()
                nxt = made[0]
            for h in hs:
                h.destroy()
        e2e_res = np.concatenate(parts)
    torch.cuda.synchronize()
    R["e2e_s"] = time.perf_counter() - t0
    R["e2e_sub_batches"] = n_sub
    R["e2e_verified"] = verify_results(workload, seeds, e2e_res)
    if args.with_prune:
        # step 0 of the path, outside every timed region above: tg_prune_batch(EXACT) once on a fresh copy of the
        # workload (the pass mutates its instances); wall clock of the call, which synchronises
        hs = create(0, n)
        flush.fill_(1)
        torch.cuda.synchronize()
        tp = time.perf_counter()
        killed = tg.tg_prune_batch(hs, tg.TG_PRUNE_EXACT, 0)
        prune_ms = (time.perf_counter() - tp) * 1e3
        for h in hs:
            h.destroy()
        R["prune"] = {"call": "tg_prune_batch(EXACT)", "wall_ms": prune_ms, "killed_r1_r2": killed.sum(0)[:2].tolist(),
                      "entries": int(sum(i.time_us.size for i in insts))}
    R["load_bytes"] = sum(i.time_us.shape[0] * i.K * ((12 * i.P + 9 * i.K) if i.actmem_mb is not None else (8 * i.P + 9)) for i in insts)
    R["insts"], R["seeds"] = insts, seeds
    for h in handles:
        h.destroy()
    del flush, out
    return R


def summarize(R, args, workload, world, peak, peak_src, agg):
    """One workload's numbers as they go into the JSON line.  agg = (plans_all, plans_e2e, ndp_all, total_ms, e2e_s):
    sums over the ranks and max-over-ranks times."""
    plans_all, plans_e2e, ndp_all, total_ms, e2e_s = agg
    steps, n = args.steps, R["n"]
    km = sum(R["kern_ms"]) / len(R["kern_ms"])
    lm = sum(R["load_ms"]) / len(R["load_ms"])
    relax = R["relax"] / steps
    dense_bytes = R["states_dense"] / steps * 8.0          # every state of the dense valid table written once, read once
    win_bytes = R["states_windowed"] / steps * 8.0         # the states the kernel really writes and reads (row windows)
    traffic, traffic_src = ncu_traffic(workload, n, args.full_sweep)
    cyc_tot = max(1, sum(R["cyc"]))
    roof = {
        # what binds: the solver is bound by integer add-min issue (and by the latency of its short dependent chains), not by
        # DRAM -- the wavefronts of the windowed tables stay in L2 (profiles/)
        "bound": "alu", "kernel": "tgSolveKernel", "achieved": relax / (km * 1e-3) / 1e12, "peak": ALU_PEAK / 1e12,
        "unit": "T add-min/s", "frac": relax / (km * 1e-3) / ALU_PEAK,
        "peak_source": "derived: 148 SMs x 64 int32 lanes x 1.965 GHz (DESIGN.md 7.5), one VIADDMNMX per relaxation",
        "relaxations_per_launch": relax, "kernel_ms": km, "kernel_ms_steps": [round(x, 3) for x in R["kern_ms"]],
        "step_ms": [round(x, 3) for x in R["step_ms"]], "us_per_dp": km * 1e3 / (R["n_dp"] / steps),
        "traffic": traffic, "traffic_source": traffic_src,
        "dram_frac_measured": (traffic / (km * 1e-3) / 1e9 / peak) if traffic else None,
        "hbm_peak": peak, "hbm_peak_source": peak_src,
        # the dense-table figure SURVEY 8(d) defines (8 B per state of the dense valid table of every DP, whether or not the
        # windowed kernel touches it) and the same for the states the kernel does touch -- neither is achieved DRAM bandwidth
        "hbm_algorithmic_frac": dense_bytes / (km * 1e-3) / 1e9 / peak, "hbm_algorithmic_bytes_per_launch": dense_bytes,
        "hbm_windowed_frac": win_bytes / (km * 1e-3) / 1e9 / peak, "hbm_windowed_bytes_per_launch": win_bytes,
        "dps_on_l2_cost_rows": R["global_c"] / steps,
        # step 1 of the path (cost-table loader): 8*P bytes read and 9 bytes written per (slice, island) cell -- the kernel
        # of the path that IS HBM-bound on the batched workload
        "loader": {"bound": "hbm", "kernel": "tgLoadRowsKernel" if R["load_bytes"] >= (32 << 20) else "tgLoadKernel", "kernel_ms": lm, "algorithmic_bytes_per_launch": float(R["load_bytes"]),
                   "achieved": R["load_bytes"] / (lm * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                   "frac": R["load_bytes"] / (lm * 1e-3) / 1e9 / peak,
                   "note": "a few MB: bound by launch latency, not by HBM" if R["load_bytes"] < (32 << 20) else "HBM stream"},
        "cta_cycle_shares": {f[4:]: round(c / cyc_tot, 4) for f, c in zip(TgCyc, R["cyc"])}}
    return {"workload": R["desc"], "value": plans_all / (total_ms * 1e-3), "unit": UNIT, "ms_per_step": total_ms / steps,
            "instances_per_gpu": n, "dps_per_step": ndp_all / steps / world, "planning_ms_per_instance": total_ms / steps / n,
            "verified": R["verified"],
            "e2e": {"value": plans_e2e / e2e_s, "unit": UNIT, "h2d_bytes_per_step": R["h2d"], "d2h_bytes_per_step": R["d2h"],
                    "ms_per_step": e2e_s / R["e2e_steps"] * 1e3, "sub_batches": R["e2e_sub_batches"], "verified": R["e2e_verified"]},
            "roofline": roof, **({"prune": R["prune"]} if "prune" in R else {})}


TgCyc = ()


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2606_16907_b200 as tg
    global TgCyc
    tg.lib()  # fail loudly if the CUDA library is missing
    TgCyc = tg.TgSolveStats.CYC
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    from paper_2606_16907_b200.shard import aggregate
    clk = ClockSampler(local)
    names = [args.workload] + ([args.secondary] if args.secondary and args.secondary != args.workload and not args.full_sweep else [])
    parts = []
    for q, name in enumerate(names):
        R = measure_workload(tg, torch, args, name, rank, world, barrier, clk)
        total_ms = sum(R["step_ms"])
        (plans_all, plans_e2e, ndp_all), (total_ms, e2e_s) = aggregate(
            [float(R["plans"]), float(R["plans"]) / args.steps * R["e2e_steps"], float(R["n_dp"])], [total_ms, R["e2e_s"]], device="cuda")
        parts.append((name, R, (plans_all, plans_e2e, ndp_all, total_ms, e2e_s)))
    clk.close()
    if rank == 0:
        peak, peak_src = peaks()
        S = [summarize(R, args, name, world, peak, peak_src, agg) for name, R, agg in parts]
        main = S[0]
        line = {"metric": METRIC, "value": main["value"], "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": main["ms_per_step"],
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
                "verified": main["verified"],
                "config": {"workload": main["workload"], "sweep": "full" if args.full_sweep else "exact branch-and-bound over thresholds",
                           "l2": "256 MB buffer written between timed steps", "instances_per_gpu": main["instances_per_gpu"],
                           "dps_per_step": main["dps_per_step"], "planning_ms_per_instance": main["planning_ms_per_instance"]},
                "clocks": clk.summary(), "e2e": main["e2e"],
                # tgLoadKernel + tgPrepareKernel + tgSolveKernel + tgPoisonOnErrorKernel per tg_solve_batch, every workload timed
                "gpu_launches": 4 * args.steps * len(S),
                "roofline": main["roofline"]}
        if "prune" in main:
            line["prune"] = main["prune"]
        if len(S) > 1:
            # the other half of BASELINE.json's metric ("planning time per instance"): the 1024-instance batch in the same run
            line["config"]["secondary"] = S[1]
        if not args.no_cpu_baseline:
            import oracle
            cores = max(1, min(oracle.hw_threads(), args.cpu_threads))
            R0 = parts[0][1]
            p, dt, sample = oracle_sample(R0["insts"], args.workload, R0["seeds"], cores)
            line["cpu_baseline"] = {"value": p / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                                    "seconds": dt}
        print(json.dumps(line), flush=True)
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
    ap.add_argument("--secondary", default="cfg5", help="second workload measured in the same run and reported under "
                    "config.secondary (default: the 1024-instance batch); '' = none")
    ap.add_argument("--e2e-sub", type=int, default=3, help="sub-batches of the end-to-end leg of a large batch (upload of one "
                    "overlaps the solve of the previous)")
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
