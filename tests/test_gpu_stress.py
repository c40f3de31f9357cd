"""Repeat-run determinism of the persistent solver: its grid and team barriers are hand-rolled (release-arrive /
acquire-poll on monotone counters), the items of a round come from an atomic queue and the best state of a DP is folded
with 64-bit atomicMin -- none of which a race detector has seen (compute-sanitizer is closed on this pool).  300
back-to-back solves of the 70B-like config, the MoE-like config and a 300-instance mix, alternating between two streams
with asynchronous device results: every result must be bit-identical to the first, which must equal the stored oracle
result."""
import json
import os

import numpy as np
import pytest

import tg_inputs as gen

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))


def test_300_back_to_back_solves_are_bit_identical():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_16907_b200 as tg
    tg.lib()
    mix = [gen.config5_one(s, L=20 + s % 9, K=4 + s % 5) for s in range(300)]
    sets = {"cfg3": [gen.config3()], "cfg4": [gen.config4()], "mix": mix}
    hs = {k: [tg.instance_from_inputs(i) for i in v] for k, v in sets.items()}
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    reps = 300
    outs = {k: torch.zeros(reps, len(v) * tg.RESULT_BYTES, dtype=torch.uint8, device="cuda") for k, v in hs.items()}
    for it in range(reps):
        st = streams[it & 1]
        with torch.cuda.stream(st):
            for k in ("cfg3", "cfg4", "mix"):
                tg.tg_solve_batch(hs[k], out=outs[k][it], stream=st)          # device results, no statistics: fully asynchronous
    torch.cuda.synchronize()
    for k in hs:
        o = outs[k].cpu().numpy()
        res = o.view(tg.RESULT_DTYPE).reshape(reps, len(hs[k]))
        # n_thresholds_run is a diagnostic of the search schedule; everything else is the result
        cols = [c for c in tg.RESULT_DTYPE.names if c != "n_thresholds_run"]
        for c in cols:
            assert (res[c] == res[c][0:1]).all(), f"{k}: field {c} differs between runs"
        if k != "mix":   # (a batch of >= 64 instances runs in queue mode: the number of DPs per instance follows the queue's backlog)
            assert (res["n_thresholds_run"] == res["n_thresholds_run"][0:1]).all(), f"{k}: the search schedule differs between runs"
    for name in ("cfg3", "cfg4"):
        e = json.load(open(os.path.join(HERE, "golden", f"expected_{name}.json")))["records"][0]["solve"]
        g = outs[name][0].cpu().numpy().view(tg.RESULT_DTYPE)[0]
        n = int(g["n_stages"])
        assert [int(g["iter_time_us"]), int(g["bottleneck_us"]), int(g["island_mask"]),
                [[int(g["stage_begin"][i]), int(g["stage_island"][i]), int(g["stage_plan"][i])] for i in range(n)]] == \
               [e["iter_time_us"], e["bottleneck_us"], e["island_mask"], e["stages"]]
    for v in hs.values():
        for h in v:
            h.destroy()
