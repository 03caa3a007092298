"""Pins for oracle O5 (MV-WSA): SURVEY.md §8(c) P5, P6, P10."""
import math
import random

import pytest

import synth_inputs as si
from golden_util import num, read_golden
from oracle import mvwsa
from oracle.paging import LRU, PagerLayer

GIB = 1 << 30
MIB = 1 << 20


def test_p5_size_accounting_matches_paper_traffic():
    g = {k: num(v) for k, v in read_golden("sec4_traffic.txt").items()}
    q = si.QWEN3
    assert q.expert_bytes == g["expert_mib"] * MIB
    assert (q.n_layers, q.top_k) == (g["n_layers"], g["top_k"])
    per_token = q.n_layers * q.top_k * q.expert_bytes
    assert per_token == int(3.375 * GIB)
    mid = 0.5 * (g["carry_over_lo"] + g["carry_over_hi"])
    assert per_token * (1 - mid) / GIB == pytest.approx(g["mandatory_gib_per_token"], abs=g["mandatory_tol_gib"])
    lo = g["h2d_gbs"] * 1e9 / (per_token * (1 - g["carry_over_lo"]))
    hi = g["h2d_gbs"] * 1e9 / (per_token * (1 - g["carry_over_hi"]))
    assert 12 < lo < hi < 16.5            # the paper's "roughly 13-16 tok/s"


def test_p6_table4_live_law_reproduces_35_and_1p53():
    g = {k: num(v) for k, v in read_golden("table4_dual_resize.txt").items()}
    a = g["a_mib"] * MIB
    assert a == si.QWEN3.slot_unit_bytes
    b = MIB                                           # block size is free here: only bytes matter
    kv_before = round(g["kv_before_gib"] * GIB / b)
    B = g["cap_before"] * a + kv_before * b
    p = g["kv_peak_frac"] * kv_before
    C, kappa, moved = mvwsa.live_law(B=B, a=a, b=b, kappa_floor=0, p=p, h=g["headroom"],
                                     C_min=8, C_max=128, C_cur=g["cap_before"], delta=1)
    assert moved and C == g["cap_after"]
    assert kappa * b / GIB == pytest.approx(g["kv_after_gib"], abs=g["kv_after_tol_gib"])
    assert C * a + kappa * b <= B                     # never overcommits
    # byte conservation: 3 slots' worth moved from KV to experts
    assert (kv_before - kappa) * b == pytest.approx(3 * a, abs=b)


def test_live_law_floor_clip_deadzone():
    a, b, B = 432 * MIB, 3 * MIB // 2, 12 * GIB
    floor_ = mvwsa.kappa_min(1, 16384 + 512, 16)
    assert floor_ == 1056                              # DESIGN.md G15
    assert (B - floor_ * b) // a == 24
    C, kappa, moved = mvwsa.live_law(B=B, a=a, b=b, kappa_floor=floor_, p=10, h=0.2, C_min=8, C_max=128, C_cur=14, delta=1)
    assert (C, moved) == (24, True) and kappa >= floor_ and C * a + kappa * b <= B
    C, kappa, moved = mvwsa.live_law(B=B, a=a, b=b, kappa_floor=floor_, p=10, h=0.2, C_min=8, C_max=20, C_cur=14, delta=1)
    assert C == 20 and kappa == (B - 20 * a) // b
    C, _, moved = mvwsa.live_law(B=B, a=a, b=b, kappa_floor=floor_, p=10, h=0.2, C_min=8, C_max=128, C_cur=24, delta=1)
    assert (C, moved) == (24, False)
    C, _, moved = mvwsa.live_law(B=B, a=a, b=b, kappa_floor=floor_, p=10, h=0.2, C_min=8, C_max=128, C_cur=22, delta=3)
    assert (C, moved) == (22, False)
    rng = random.Random(1)
    for _ in range(200):
        p = rng.randint(0, 9000)
        C, kappa, _ = mvwsa.live_law(B=B, a=a, b=b, kappa_floor=floor_, p=p, h=0.2, C_min=1, C_max=128, C_cur=14, delta=1)
        assert C * a + kappa * b <= B


def _convex_curve(n, scale, rate):
    return [scale * math.exp(-rate * c) for c in range(n + 1)]


def test_p10_configurator_bruteforce_equals_greedy_on_convex_curves():
    rng = random.Random(2)
    a, b = 432 * MIB, 3 * MIB // 2
    for _ in range(100):
        B = rng.randint(4, 40) * GIB
        m_exp = _convex_curve(128, rng.uniform(1e3, 1e5), rng.uniform(0.01, 0.3))
        s, r = rng.uniform(1e3, 1e6), rng.uniform(1e-4, 1e-2)
        m_kv = lambda kap, s=s, r=r: s * math.exp(-r * kap)
        kw = dict(B=B, a=a, b=b, kappa_floor=rng.randint(0, 1500), c_exp=rng.uniform(1e-4, 1e-3),
                  c_kv=rng.uniform(1e-5, 1e-3), m_exp=m_exp, m_kv=m_kv, C_min=1, C_max=128)
        assert mvwsa.configurator(**kw) == mvwsa.greedy_marginal_walk(**kw)
        res = mvwsa.configurator(**kw)
        if res:
            C, Bkv = res
            assert Bkv == B - C * a and Bkv >= kw["kappa_floor"] * b     # Eq. 5 + floor (Eq. 4)


def test_p10_configurator_limits():
    a, b, B = 432 * MIB, 3 * MIB // 2, 12 * GIB
    m_exp = _convex_curve(128, 1e4, 0.1)
    kw = dict(B=B, a=a, b=b, kappa_floor=1056, c_exp=1e-3, c_kv=1e-4, C_min=8, C_max=128)
    # m_kv == 0: all the bytes go to experts, up to the floor: min(E, C_max, C_feas) = 24  (Eq. 5)
    assert mvwsa.configurator(m_exp=m_exp, m_kv=lambda k: 0.0, **kw)[0] == 24
    # m_exp constant: nothing to gain on the expert side -> C_min
    assert mvwsa.configurator(m_exp=[5.0] * 129, m_kv=lambda k: 1e6 / (1 + k), **kw)[0] == 8
    # never beyond the floor whatever the curves
    assert mvwsa.configurator(m_exp=m_exp, m_kv=lambda k: 0.0, **{**kw, "C_max": 24})[0] <= 24
    assert mvwsa.configurator(m_exp=m_exp, m_kv=lambda k: 0.0, **{**kw, "kappa_floor": 10 ** 6}) is None


def test_miss_curve_limits_and_estimator_gap():
    """P7 for k > 1: the histogram is an estimator of Algorithm 1 (parity unpinned beyond these limits):
    monotone non-increasing in C; at C >= E equals the distinct-expert count."""
    rng = random.Random(9)
    E, k = 16, 2
    steps = [rng.sample(range(E), k) for _ in range(300)]
    mc = mvwsa.miss_curve([steps], E)
    assert all(mc[c] >= mc[c + 1] for c in range(E))
    assert mc[E] == len({e for s in steps for e in s})
    assert mc[0] == sum(len(set(s)) for s in steps)
    p = PagerLayer(C=E, E=E, policy=LRU)
    for s in steps:
        p.step(s)
    assert p.misses == mc[E]


def test_kv_scheduler_model_basics():
    sch = mvwsa.KVScheduler(kappa=100, block_tokens=16)
    reqs = [mvwsa.Request(i, prompt=640, target=200) for i in range(3)]   # 40 blocks each
    sch.waiting.extend(reqs)
    adm = sch.admit()
    assert [r.rid for r, _ in adm] == [0, 1] and sch.used == 80
    for _ in range(400):
        sch.admit()
        sch.decode_tick()
        assert sch.used <= sch.kappa
        if not sch.running and not sch.waiting:
            break
    assert all(r.generated == 200 for r in reqs)
    assert sch.peak <= 100
