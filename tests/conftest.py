import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def rescore(inst, stages):
    """Independent re-scorer: recompute (sum, T, iter, mask) of a plan straight from the RAW tables.
    Shares nothing with the oracle's DP or the CUDA path (SURVEY.md §8(c) pins)."""
    INVALID = 0x7FFFFFFF
    L, K, m = inst.L, inst.K, inst.m
    n = len(stages)
    assert n >= 1 and stages[0][0] == 0
    total, T, mask = 0, 0, 0
    for i, (a, k, p) in enumerate(stages):
        b = stages[i + 1][0] if i + 1 < n else L
        assert 0 <= a < b <= L
        s = a * (2 * L - a + 1) // 2 + (b - a - 1)
        t = int(inst.time_us[s, k, p])
        assert t != INVALID, "plan uses a dead entry"
        assert int(inst.mem_mb[s, k, p]) <= int(inst.island_cap_mb[k]), "plan overflows memory"
        assert not (mask >> k) & 1, "island used twice"
        mask |= 1 << k
        total += t
        T = max(T, t)
        if i + 1 < n:
            kn = stages[i + 1][1]
            bw = int(inst.bw_gbps[k, kn])
            total += -((-inst.act_mb * 1000) // bw)
    return total, T, total + (m - 1) * T, mask
