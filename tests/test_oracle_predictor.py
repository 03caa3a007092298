"""Pins for the f3 oracle (oracle/predictor.py, PagerLayer.prefetch): hand-worked cases of tests/golden/hand_predictor.txt
(App. E) and invariants."""
import random
from fractions import Fraction

from golden_util import read_golden
from oracle.paging import LRU, PREFETCH, PagerLayer
from oracle.predictor import CoActivationPredictor

G = read_golden("hand_predictor.txt")


def test_two_layer_hand_case():
    g = G["two_layers"]
    p = CoActivationPredictor(2, 3, gamma=0.5, window=1)
    for R0, R1 in (([0], [1, 2]), ([0, 1], [2])):
        p.begin_pass(); p.observe(0, R0); p.observe(1, R1)
    assert p.A[(1, 1)][0] == [0, 1, 2] and p.A[(1, 1)][1] == [0, 0, 1] and p.row[(1, 1)] == [3, 1, 0]
    p.begin_pass(); p.observe(0, [0])
    s = p.scores(1)
    assert s[0] == 0.0
    assert s[1] == float(Fraction(int(g["s1_num"]), int(g["s1_den"]))) and s[2] == float(Fraction(int(g["s2_num"]), int(g["s2_den"])))
    assert p.predict(1, 3) == [int(t) for t in g["ranking"].split()]
    assert p.predict(1, 3, resident=[2]) == [1] and p.predict(1, 1) == [2]
    p.begin_pass(); p.observe(0, [0, 1])
    assert abs(p.scores(1)[2] - int(g["s2_both_num"]) / int(g["s2_both_den"])) < 1e-15


def test_distance_decay_three_layers():
    p = CoActivationPredictor(3, 3, gamma=0.5, window=2)
    p.begin_pass(); p.observe(0, [0]); p.observe(1, [1]); p.observe(2, [2])
    p.begin_pass(); p.observe(0, [0]); p.observe(1, [0])
    assert p.scores(2) == [0.0, 0.0, float(G["three_layers"]["s2"])]
    q = CoActivationPredictor(3, 3, gamma=0.5, window=1)          # with window 1 the distance-2 source is not seen
    q.begin_pass(); q.observe(0, [0]); q.observe(1, [1]); q.observe(2, [2])
    q.begin_pass(); q.observe(0, [0]); q.observe(1, [0])
    assert q.scores(2) == [0.0, 0.0, 0.0] and q.predict(2, 2) == []


def test_prediction_sees_earlier_passes_only_and_conditionals_sum_to_one():
    rng = random.Random(3)
    L, E, k = 4, 12, 3
    p = CoActivationPredictor(L, E, gamma=0.7, window=2)
    for _ in range(40):
        p.begin_pass()
        for l in range(L):
            before = p.scores(l) if l else None
            R = rng.sample(range(E), k)
            if l:
                assert p.scores(l) == before                     # nothing of this pass reaches layer l's tables before it routes
            p.observe(l, R)
    for (l2, dist), A in p.A.items():
        for e in range(E):
            assert sum(A[e]) == p.row[(l2, dist)][e]               # row = source marginal: P(.|e) sums to 1


def test_pager_prefetch_hand_case():
    g = G["prefetch"]
    p = PagerLayer(C=2, E=4, policy=LRU)
    p.step([0, 1])
    ev = p.prefetch([2, 1])
    assert [(e.expert, e.slot, e.evicted, e.kind) for e in ev] == [(2, 0, 0, PREFETCH)]
    assert p.slots() == [int(t) for t in g["slots1"].split()] and p.tau == [int(t) for t in g["tau1"].split()] and p.c == 1
    p.step([1, 2])
    assert p.hits == int(g["hits2"])
    ev = p.prefetch([0, 3])
    assert [(e.expert, e.slot, e.evicted) for e in ev] == [(0, 0, 2), (3, 1, 1)]
    m0 = p.misses
    p.step([1, 2])
    assert p.misses - m0 == int(g["misses3"]) and p.prefetches == 3
    p.check_invariants()
