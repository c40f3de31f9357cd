#!/usr/bin/env python
"""Writes tests/golden/expected_<cfg>.json: the CPU oracle's result (value AND plan) on the full-size
configs of BASELINE.json, which take the oracle minutes and so cannot be recomputed inside the test run.
Calls ONLY oracle/ and the seeded input generator; never the CUDA path.

    python tests/golden/make_expected.py cfg3 cfg4 cfg5 cfg3x cfg4x cfg3d cfg3xb cfg3st cfg4d cfg4xb   (cfg5 = all 1024 seeds, about 35 min on 8 cores)

Also stores oracle.dp_at results at fixed quantile thresholds (single-DP parity for tg_dp_at)."""
import json
import os
import sys
import time

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle            # noqa: E402
import tg_inputs as gen  # noqa: E402

CFG5_SEEDS = list(range(1024))                                  # every instance of the throughput batch
DP_QUANTILES = [0.35, 0.5, 0.8]                                 # thresholds for the single-DP records


def rec(r):
    return {"iter_time_us": r.iter_time_us, "sum_us": r.sum_us, "bottleneck_us": r.bottleneck_us,
            "island_mask": r.island_mask, "stages": [list(s) for s in r.stages], "n_dp_run": r.n_dp_run,
            "n_candidates": r.n_candidates, "feasible": r.feasible}


def one(inst, threads, with_dp):
    t0 = time.time()
    out = {"name": inst.name, "L": inst.L, "K": inst.K, "P": inst.P, "m": inst.m, "solve": rec(oracle.solve(inst, n_threads=threads))}
    if with_dp:
        _, _, _, cand = oracle.reduce(inst)
        out["dp_at"] = []
        for T in [-1] + [int(cand[int(q * (len(cand) - 1))]) for q in DP_QUANTILES]:
            out["dp_at"].append({"T": T, "res": rec(oracle.dp_at(inst, T, want_plan=True))})
    out["oracle_seconds"] = round(time.time() - t0, 1)
    return out


def main():
    threads = max(1, min(8, oracle.hw_threads()))
    for name in sys.argv[1:]:
        if name == "cfg3":
            data = [one(gen.config3(), threads, True)]
        elif name == "cfg4":
            data = [one(gen.config4(), threads, True)]
        elif name == "cfg3x":      # more seeds of the 70B-like config
            data = [dict(one(gen.config3(s), threads, False), seed=s) for s in (1, 2, 3, 4)]
        elif name == "cfg4x":      # a second MoE-like instance
            data = [dict(one(gen.config4(1), threads, False), seed=1)]
        elif name == "cfg3d":      # NEXT-1: the 70B-like config with a per-plan activation footprint (depth oracle)
            inst = gen.with_actmem(gen.config3(), 7, 500, 6000)
            t0 = time.time()
            data = [{"name": inst.name, "L": inst.L, "K": inst.K, "P": inst.P, "m": inst.m,
                     "solve": rec(oracle.solve_depth(inst)), "core": rec(oracle.solve(inst, n_threads=threads)),
                     "oracle_seconds": round(time.time() - t0, 1)}]
        elif name == "cfg3xb":     # NEXT-3(b): the 70B-like config with transfers bounded by the threshold (variant oracle)
            inst = gen.with_transfer_bound(gen.config3())
            t0 = time.time()
            data = [{"name": inst.name, "L": inst.L, "K": inst.K, "P": inst.P, "m": inst.m,
                     "solve": rec(oracle.solve_variant(inst)), "core": rec(oracle.solve(inst, n_threads=threads)),
                     "oracle_seconds": round(time.time() - t0, 1)}]
        elif name == "cfg3st":     # NEXT-2: the 70B-like config with multi-stage partial plans (stages oracle)
            inst = gen.with_stages(gen.config3(), 3)
            t0 = time.time()
            r, tq = oracle.solve_stages(inst)
            data = [{"name": inst.name, "L": inst.L, "K": inst.K, "P": inst.P, "m": inst.m, "solve": rec(r),
                     "pipeline_stages": tq, "oracle_seconds": round(time.time() - t0, 1)}]
        elif name in ("cfg4d", "cfg4xb"):   # the K = 16 variant workloads bench.py times: threaded variant oracle (same arithmetic)
            inst = gen.with_actmem(gen.config4(), 11, 300, 3000) if name == "cfg4d" else gen.with_transfer_bound(gen.config4())
            t0 = time.time()
            data = [{"name": inst.name, "L": inst.L, "K": inst.K, "P": inst.P, "m": inst.m,
                     "solve": rec(oracle.solve_variant(inst, n_threads=threads)),
                     "oracle_seconds": round(time.time() - t0, 1)}]
        elif name == "cfg5":
            data = [dict(one(gen.config5_one(s), threads, False), seed=s) for s in CFG5_SEEDS]
        else:
            raise SystemExit(f"unknown config {name}")
        with open(os.path.join(HERE, f"expected_{name}.json"), "w") as f:
            if len(data) > 64:     # the 1024-record batch: one compact record per line
                f.write('{"written_by": "tests/golden/make_expected.py (CPU oracle only)", "records": [\n')
                f.write(",\n".join(json.dumps(d, separators=(",", ":")) for d in data))
                f.write("\n]}\n")
            else:
                json.dump({"written_by": "tests/golden/make_expected.py (CPU oracle only)", "records": data}, f, indent=1)
        print(name, "done", [d["oracle_seconds"] for d in data], flush=True)


if __name__ == "__main__":
    main()
