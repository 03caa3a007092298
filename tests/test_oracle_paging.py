"""Pins for oracle O4 (Algorithm 1): SURVEY.md §8(c) P3, P4, P7, P9."""
import random

import pytest

from golden_util import num, read_golden
from oracle import mvwsa
from oracle.paging import ASCENDING, HITS_FIRST, HIT, LFU, LRU, MISS, RESIZE_DROP, RESIZE_MOVE, PagerLayer

TR = read_golden("hand_paging_trace.txt")
STEPS = [{1, 4}, {1, 2}, {3, 5}, {1, 2}, {2, 3}, {0, 4}]


def _parse_step(txt):
    misses, slots, tau = (p.strip() for p in txt.split("|"))
    m = []
    for tok in misses.split():
        e, rest = tok.split(">")
        s, ev = rest.split("/")
        m.append((int(e), int(s), -1 if ev == "-" else int(ev)))
    sl = [None if t == "-" else int(t) for t in slots.split()]
    ta = [int(t) for t in tau.split()] if tau else None
    return m, sl, ta


@pytest.mark.parametrize("name,policy", [("lru", LRU), ("lfu", LFU)])
def test_p4_hand_trace(name, policy):
    sec = TR[name]
    p = PagerLayer(C=3, E=6, policy=policy)
    for i, R in enumerate(STEPS):
        ev = p.step(R)
        m, sl, ta = _parse_step(sec[f"step{i}"])
        assert [(e.expert, e.slot, e.evicted) for e in ev if e.kind == MISS] == m
        assert p.slots() == sl
        if ta is not None:
            assert p.tau == ta
        assert [e.expert for e in ev] == sorted(R)
        p.check_invariants()
    assert p.hits == num(sec["hits"]) and p.misses == num(sec["misses"])
    if "evictions" in sec:
        assert p.evictions == num(sec["evictions"])


def test_p4_overflow_waves():
    sec = TR["overflow"]
    p = PagerLayer(C=2, E=6, policy=LRU)
    ev = p.step([0, 1, 2, 3, 5])
    m, sl, ta = _parse_step(sec["step0"])
    assert [(e.expert, e.slot, e.evicted) for e in ev if e.kind == MISS] == m
    assert [e.wave for e in ev] == [0, 0, 1, 1, 2]
    assert p.slots() == sl and p.tau == ta
    ev = p.step([3, 5])
    _, sl, ta = _parse_step(sec["step1"])
    assert sum(e.kind == HIT for e in ev) == num(sec["step1_hits"]) and p.slots() == sl and p.tau == ta


def test_g25_hits_first_hand_trace():
    """G25, stepped by hand in tests/golden/hand_paging_trace.txt [hits_first]."""
    sec = TR["hits_first"]
    steps = [{4, 5}, {0, 1, 5}, {1, 5}]
    p = PagerLayer(C=2, E=6, policy=LRU, wave_order=HITS_FIRST)
    for i, R in enumerate(steps):
        ev = p.step(R)
        m, sl, ta = _parse_step(sec[f"step{i}"])
        assert [(e.expert, e.slot, e.evicted) for e in ev if e.kind == MISS] == m
        assert p.slots() == sl and p.tau == ta
        if i == 1:
            assert [e.expert for e in ev] == [int(t) for t in sec["step1_order"].split()]
            assert [e.wave for e in ev] == [int(t) for t in sec["step1_waves"].split()]
        p.check_invariants()
    assert p.hits == num(sec["hits"]) and p.misses == num(sec["misses"])
    q = PagerLayer(C=2, E=6, policy=LRU, wave_order=ASCENDING)
    for i, R in enumerate(steps):
        ev = q.step(R)
        if i == 1:
            m, sl, ta = _parse_step(sec["ascending_step1"])
            assert [(e.expert, e.slot, e.evicted) for e in ev if e.kind == MISS] == m
            assert q.slots() == sl and q.tau == ta
    assert q.hits == num(sec["ascending_hits"]) and q.misses == num(sec["ascending_misses"])


@pytest.mark.parametrize("policy", [LRU, LFU])
def test_g25_hits_first_closed_form_random_streams(policy):
    """Under HITS_FIRST the faults of a step are exactly R minus the residents at step start (set arithmetic,
    not the oracle's loop); ASCENDING can only fault more on the same state; |R| <= C gives the same trace."""
    rng = random.Random(11)
    for trial in range(40):
        E = rng.randint(3, 40)
        C = rng.randint(1, E)
        k = rng.randint(1, min(E, 12))
        hf = PagerLayer(C=C, E=E, policy=policy, wave_order=HITS_FIRST)
        for t in range(50):
            R = set(rng.sample(range(E), rng.randint(1, k)))
            resident = set(hf.pi)
            asc = PagerLayer(C=C, E=E, policy=policy)          # same state, ascending order, one step
            asc.pi, asc.pi_inv, asc.tau, asc.f, asc.c, asc.steps = dict(hf.pi), list(hf.pi_inv), list(hf.tau), list(hf.f), hf.c, hf.steps
            ev = hf.step(R)
            ev_a = asc.step(R)
            assert sorted(e.expert for e in ev) == sorted(R)
            assert {e.expert for e in ev if e.kind == MISS} == R - resident
            assert {e.expert for e in ev if e.kind == HIT} == R & resident
            assert sum(e.kind == MISS for e in ev_a) >= len(R - resident)
            if len(R) <= C:
                assert [e.key() for e in ev] == [e.key() for e in ev_a]
            else:
                n_res = len(R & resident)
                assert [e.expert for e in ev] == sorted(R & resident) + sorted(R - resident)
                assert all(e.wave == 0 for e in ev[:n_res])
            for wv in set(e.wave for e in ev):
                sl = [e.slot for e in ev if e.wave == wv]
                assert len(set(sl)) == len(sl) <= C
                evicted = {e.evicted for e in ev if e.wave == wv and e.evicted >= 0}
                assert not evicted & {e.expert for e in ev if e.wave == wv}
            hf.check_invariants()
        assert hf.hits + hf.misses == hf.references


def test_p3_fig4_printed_fault_counts():
    g = {k: num(v) for k, v in read_golden("fig4_fault_counts.txt").items()}
    for cap in (8, 4, 2):
        faults = hits = 0
        for _ in range(g["n_layers"]):
            p = PagerLayer(C=cap, E=g["n_experts"], policy=LRU)
            for _ in range(g["n_steps"]):
                p.step(range(g["n_experts"]))
            faults += p.misses
            hits += p.hits
        assert (faults, hits) == (g[f"cap{cap}_faults"], g[f"cap{cap}_hits"])


def test_p7_mattson_hand_case():
    sec = TR["mattson"]
    stream = sec["stream"].split()
    want = [mvwsa.INF if t == "inf" else int(t) for t in sec["distances"].split()]
    assert mvwsa.stack_distances(stream) == want
    mc = mvwsa.miss_curve_from_hist(mvwsa.histogram(want, 4), 4)
    assert [mc[c] for c in (1, 2, 3, 4)] == [num(sec[f"m{c}"]) for c in (1, 2, 3, 4)]


def test_p7_k1_is_textbook_lru_and_matches_stack_distances():
    rng = random.Random(11)
    for trial in range(20):
        E = rng.randint(2, 12)
        stream = [rng.randrange(E) for _ in range(200)]
        dist = mvwsa.stack_distances(stream)
        for C in range(1, E + 1):
            # Algorithm 1 at k = 1
            p = PagerLayer(C=C, E=E, policy=LRU)
            for e in stream:
                p.step([e])
            # textbook LRU written independently: ordered list, most recent last
            cache, miss = [], 0
            for e in stream:
                if e in cache:
                    cache.remove(e)
                else:
                    miss += 1
                    if len(cache) == C:
                        cache.pop(0)
                cache.append(e)
            assert p.misses == miss == sum(d > C for d in dist)


@pytest.mark.parametrize("policy", [LRU, LFU])
def test_p9_invariants_random_streams(policy):
    rng = random.Random(5)
    for trial in range(30):
        E = rng.randint(2, 40)
        C = rng.randint(1, E)
        k = rng.randint(1, min(E, 9))
        p = PagerLayer(C=C, E=E, policy=policy)
        total_refs, distinct = 0, set()
        for t in range(60):
            R = set(rng.sample(range(E), k))
            resident_before = set(p.pi)
            ev = p.step(R)
            total_refs += len(R)
            distinct |= R
            assert [e.expert for e in ev] == sorted(R)
            # every expert of the LAST wave is resident at its FFN time; slots distinct within a wave
            for wv in set(e.wave for e in ev):
                sl = [e.slot for e in ev if e.wave == wv]
                assert len(set(sl)) == len(sl) and len(sl) <= C
                evicted = {e.evicted for e in ev if e.wave == wv and e.evicted >= 0}
                assert not evicted & {e.expert for e in ev if e.wave == wv}
            if len(R) <= C:
                assert all((e.kind == HIT) == (e.expert in resident_before) for e in ev)
                assert R <= set(p.pi)
            p.check_invariants()
        assert p.hits + p.misses == total_refs == p.references
        if C >= E:
            assert p.misses == len(distinct) and p.evictions == 0


def test_resize_shrink_grow_cycle():
    p = PagerLayer(C=4, E=8, policy=LRU)
    for R in ([0, 1], [2, 3], [0, 2]):
        p.step(R)
    # slots [0,1,2,3], tau [3,1,3,2]; shrink to 2 keeps the two most recent: slots 0 (e0) and 2 (e2)
    ev = p.resize(2)
    assert [(e.kind, e.expert, e.slot) for e in ev] == [(RESIZE_DROP, 1, 1), (RESIZE_DROP, 3, 3), (RESIZE_MOVE, 2, 1)]
    assert p.slots() == [0, 2] and p.tau == [3, 3] and p.C == 2
    p.check_invariants()
    ev = p.resize(5)
    assert ev == [] and p.slots() == [0, 2, None, None, None] and p.tau == [3, 3, 0, 0, 0]
    ev = p.step([0, 5])
    assert [(e.expert, e.slot, e.kind) for e in ev] == [(0, 0, HIT), (5, 2, MISS)]
    p.check_invariants()


def test_empty_step_is_noop():
    p = PagerLayer(C=2, E=4)
    assert p.step([]) == [] and p.c == 0 and p.steps == 0


def _parse_resize(spec):
    """'drop:2@1 move:3@1<2' -> [(expert, slot, evicted_or_source, kind)]"""
    out = []
    for tok in spec.split():
        kind, rest = tok.split(":")
        e, rest = rest.split("@")
        if kind == "drop":
            out.append((int(e), int(rest), -1, RESIZE_DROP))
        else:
            dst, src = rest.split("<")
            out.append((int(e), int(dst), int(src), RESIZE_MOVE))
    return out


def _lfu_state(steps):
    p = PagerLayer(C=3, E=8, policy=LFU)
    for R in steps:
        p.step(R)
    return p


def test_lfu_resize_hand_trace():
    """O4 resize rule under LFU, keep order (f desc, tau desc, slot asc): hand-stepped (golden [lfu_resize])."""
    import copy
    g = read_golden("hand_paging_trace.txt")["lfu_resize"]
    ints = lambda v: [int(t) for t in v.split()]
    base = _lfu_state([[1, 2, 3], [3], [3], [1]])
    assert base.slots() == ints(g["state_slots"]) and base.tau == ints(g["state_tau"])
    assert (base.f[1], base.f[2], base.f[3]) == (2, 1, 3)
    p = copy.deepcopy(base)
    ev = [(e.expert, e.slot, e.evicted, e.kind) for e in p.resize(2)]
    assert ev == _parse_resize(g["shrink2_events"]) and p.slots() == ints(g["shrink2_slots"]) and p.tau == ints(g["shrink2_tau"])
    p.check_invariants()
    p = copy.deepcopy(base)
    ev = [(e.expert, e.slot, e.evicted, e.kind) for e in p.resize(1)]
    assert ev == _parse_resize(g["shrink1_lfu_events"]) and p.slots() == ints(g["shrink1_lfu_slots"]) and p.tau == ints(g["shrink1_lfu_tau"])
    # the same state under LRU keeps a different survivor (the most recent, not the most frequent)
    q = copy.deepcopy(base)
    q.policy = LRU
    ev = [(e.expert, e.slot, e.evicted, e.kind) for e in q.resize(1)]
    assert ev == _parse_resize(g["shrink1_lru_events"]) and q.slots() == ints(g["shrink1_lru_slots"])
    # f ties fall back to tau descending
    t = _lfu_state([[1, 2], [1], [1], [3]])
    assert t.tau == ints(g["tie_state_tau"])
    ev = [(e.expert, e.slot, e.evicted, e.kind) for e in t.resize(2)]
    assert ev == _parse_resize(g["tie_shrink2_events"]) and t.slots() == ints(g["tie_shrink2_slots"]) and t.tau == ints(g["tie_shrink2_tau"])
    t.check_invariants()


def test_decay_and_miss_curve_two_period_hand_case():
    """PAPER.md:152 'decayed' histograms: bins of period 1 times lambda, plus period 2 (golden [decay])."""
    from oracle import mvwsa
    g = read_golden("hand_paging_trace.txt")["decay"]
    d_all = mvwsa.stack_distances(list("abab" "bc"))          # the LRU stack carries over between the periods
    h1 = mvwsa.histogram(d_all[:3], 2)
    h = mvwsa.decay(h1, 0.5)
    h2 = mvwsa.histogram(d_all[3:], 2)
    tot = [a + b for a, b in zip(h, h2)]
    assert tot[1:] == [float(v) for v in g["bins_after"].split()]
    assert mvwsa.miss_curve_from_hist(tot, 2) == [float(g["m0"]), float(g["m1"]), float(g["m2"])]


def test_static_offload_byte_model_closed_forms():
    """f2: the static layer-offload arm's traffic.  Closed forms + the config 2 numbers by hand:
    E * M_e = 128 * 9 MiB = 1152 MiB per layer; 8 GiB / 1152 MiB = 7 -> 5 resident + 2 bounce -> 43 layers streamed
    = 43 * 1152 MiB = 48.375 GiB per token (vs 3.375 GiB * (1 - carry-over) for the paged pool, sec4_traffic.txt)."""
    from oracle.paging import static_offload_bytes_per_forward as f
    MIB = 1 << 20
    L, E, Me = 48, 128, 9 * MIB
    assert f(L, E, Me, 8 << 30) == 43 * 1152 * MIB == int(48.375 * (1 << 30))
    assert f(L, E, Me, 2 * E * Me) == L * E * Me                     # two bounce buffers only: everything streams
    assert f(L, E, Me, (L + 2) * E * Me) == 0                        # everything fits
    assert f(L, E, Me, (L + 50) * E * Me) == 0
    assert f(L, E, Me, 3 * E * Me + 5) == (L - 1) * E * Me
    assert all(f(L, E, Me, (n + 2) * E * Me) - f(L, E, Me, (n + 3) * E * Me) == E * Me for n in range(L))   # one layer per E*M_e of budget
