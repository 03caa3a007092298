"""Full-DEPTH parity on a B200 (-m gpu): the reduced form of `python bench.py --verify 2,3` that the driver runs.
BASELINE.json configs 2 and 3 on the whole 48-layer Qwen3-30B-A3B-shaped stack through wisp_stack_forward (the launch
configuration bench.py times): prefill of 2048 tokens + 16 decode steps at batch 1 and 4, pools of 4 GiB (C = 9), 8 GiB (C = 18)
and all-resident, LRU and LFU at 8 GiB.  (a) trace == oracle/paging.py on the GPU's ids, (b) every step's x_L byte-identical to
the all-resident run, (c)/(d) teacher-forced against oracle/moe_forward.py on sampled (step, layer) pairs.
The full-length runs (256 steps, 4/8/16/32 GiB, Mixtral shape) are `bench.py --verify 2,3,4`; their summary is committed
under profiles/."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

pytestmark = pytest.mark.gpu


def _host_ram_ok(shape):
    with open("/proc/meminfo") as fh:
        avail = next(int(l.split()[1]) * 1024 for l in fh if l.startswith("MemAvailable"))
    return avail * 0.8 > shape.n_layers * shape.n_experts * shape.expert_bytes


def test_config3_full_depth_prefill_then_decode_across_budgets():
    import bench
    import synth_inputs as si
    q = si.QWEN3
    if not _host_ram_ok(q):
        pytest.skip("not enough host RAM for the 54 GiB pinned master")
    steps = 16
    samples = tuple((s, l) for s in (0, steps - 1) for l in (0, q.n_layers // 2, q.n_layers - 1))
    runs = [("all-resident", q.n_experts), ("8 GiB", 18), ("4 GiB", 9)]
    s = bench.verify_stack(q, runs, steps=steps, batches=(1, 4), prefill_tokens=2048, samples=samples, policies=("lru", "lfu"))
    assert s["byte_identical"] and s["trace_equal"], s
    assert s["max_rel_err"] <= 2e-2 and s["oracle_samples"] == 2 * len(samples)
    assert all(r["misses"] == r["oracle_misses"] and r["pool_bytes_equal_master"] for r in s["runs"])
    # the budgets really page: the small pools fault more than the all-resident one
    by = {(r["pool"], r["policy"], r["batch"]): r["misses"] for r in s["runs"]}
    assert by[("4 GiB", "lru", 1)] > by[("8 GiB", "lru", 1)] >= by[("all-resident", "lru", 1)]
