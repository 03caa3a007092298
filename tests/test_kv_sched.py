"""The harness-side KV-reservation scheduler (paper_2606_21868_b200/kv_sched.py, the one bench.py drives) against a
hand-stepped case (tests/golden/hand_kv_schedule.txt) and, step by step, against the oracle's model
(oracle/mvwsa.py:KVScheduler).  SURVEY.md 8(c) O5; G12."""
import random

from golden_util import read_golden
from oracle import mvwsa
from paper_2606_21868_b200.kv_sched import KvRequest, KvReservationScheduler

G = read_golden("hand_kv_schedule.txt")
ints = lambda v: [int(t) for t in v.split()]


def _run_harness(kappa, specs, log=None, ledger=None):
    reqs = [KvRequest(i, p, t) for i, (p, t) in enumerate(specs)]
    sch = KvReservationScheduler(kappa, reqs, reserve=(ledger.append if ledger is not None else None))
    admits, prefills, used, decoded, preempt_tick, tick = [], [], [], [], [], 0
    while sch.waiting or sch.running:
        for r, n in sch.admit():
            admits.append(r.rid); prefills.append(n)
        assert sch.running, "admission floor violated"
        before = sch.preemptions
        run = sch.grow_for_decode()
        tick += 1
        if sch.preemptions > before:
            preempt_tick.append(tick)
        decoded.append([r.rid for r in run])
        sch.finish_tick()
        used.append(sch.used)
        assert sch.used <= sch.kappa
    return sch, admits, prefills, used, decoded, preempt_tick


def _run_oracle(kappa, specs):
    sch = mvwsa.KVScheduler(kappa=kappa, block_tokens=16)
    sch.waiting.extend(mvwsa.Request(i, prompt=p, target=t) for i, (p, t) in enumerate(specs))
    admits, prefills, used, decoded = [], [], [], []
    while sch.waiting or sch.running:
        for r, n in sch.admit():
            admits.append(r.rid); prefills.append(n)
        done = sch.decode_tick()
        decoded.append([r.rid for r in done])
        used.append(sch.used)
    return sch, admits, prefills, used, decoded


def test_hand_stepped_schedule_both_implementations():
    specs = [(48, 4), (64, 4), (40, 2)]
    want_dec = [[int(x) for x in t.split(",")] for t in G["decoded_per_tick"].split()]
    ledger = []
    h, admits, prefills, used, decoded, ptick = _run_harness(10, specs, ledger=ledger)
    assert admits == ints(G["admit_order"]) and prefills == ints(G["prefill_tokens"])
    assert used == ints(G["used_after_tick"]) and decoded == want_dec
    assert h.preemptions == int(G["preemptions"]) and ptick == [int(G["preempt_tick"])]
    assert h.reprefill_tokens == int(G["reprefill_tokens"]) and h.peak == int(G["peak_used"])
    assert sum(ledger) == 0 and min(_prefix(ledger)) >= 0 and max(_prefix(ledger)) == h.peak   # what wisp_kv_reserve saw
    o, o_admits, o_prefills, o_used, o_decoded = _run_oracle(10, specs)
    assert (o_admits, o_prefills, o_used, o_decoded) == (admits, prefills, used, decoded)
    assert (o.preemptions, o.reprefill_tokens, o.peak) == (h.preemptions, h.reprefill_tokens, h.peak)


def _prefix(xs):
    out, acc = [], 0
    for x in xs:
        acc += x
        out.append(acc)
    return out


def test_harness_equals_oracle_model_on_random_workloads():
    rng = random.Random(5)
    for _ in range(60):
        n = rng.randint(1, 6)
        specs = [(rng.randint(1, 400), rng.randint(1, 60)) for _ in range(n)]
        floor = max(-(-(p + t) // 16) for p, t in specs)               # one full request always fits (Eq. 4, W = 1)
        kappa = rng.randint(floor, floor + 40)
        h, *hrest = _run_harness(kappa, specs)
        o, *orest = _run_oracle(kappa, specs)
        assert tuple(hrest[:4]) == tuple(orest)
        assert (h.preemptions, h.reprefill_tokens, h.peak) == (o.preemptions, o.reprefill_tokens, o.peak)
        assert all(r.gen == r.target for r in h.done) and len(h.done) == n


def test_window_peak_survives_a_request_finishing_mid_window():
    """p of Eq. 6 is the PEAK occupancy of the window, not the level when the controller looks."""
    reqs = [KvRequest(0, 160, 2), KvRequest(1, 160, 40)]
    sch = KvReservationScheduler(100, reqs)
    sch.reset_window()
    sch.admit()
    for _ in range(5):
        sch.grow_for_decode(); sch.finish_tick()
    assert len(sch.done) == 1 and sch.used == 11          # request 0 left; request 1 holds ceil(165/16) blocks
    assert sch.window_peak == 22                          # 10 + 10 at admission, +1 each when both crossed 160 -> 161 tokens in tick 1
    sch.reset_window()
    assert sch.window_peak == sch.used
    sch.set_kappa(50)
    assert sch.kappa == 50
