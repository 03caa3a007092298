"""GPU tests of the residency engine on adversarial routing (SURVEY.md §4 tier 3), resize (tier 4), errors,
and the device-side MV-WSA histograms: all bit-exact against the oracle's O4/O5 simulation."""
import random

import pytest
import torch

import synth_inputs as si
from harness import make_ctx, run_chain, run_stack, sim_trace
from oracle import mvwsa
from oracle.paging import PagerLayer

pytestmark = pytest.mark.gpu

SH = si.TINY


def streams(E, C, k):
    rng = random.Random(1234)
    yield "cyclic", [[(t * k + j) % E for j in range(k)] for t in range(3 * E)]
    yield "same", [[0] * k for _ in range(10)]
    yield "all", [list(range(E)) for _ in range(6)]
    yield "random", [rng.sample(range(E), k) for _ in range(80)]
    yield "repeats", [[rng.randrange(E) for _ in range(3 * k)] for _ in range(40)]
    yield "ragged", [rng.sample(range(E), rng.randint(1, E)) for _ in range(40)]


@pytest.mark.parametrize("C", [1, 2, 6, 15, 16])
@pytest.mark.parametrize("policy", [0, 1])
@pytest.mark.parametrize("fetch", [0, 1, 2])
def test_adversarial_routing_trace_and_state(C, policy, fetch):
    E = SH.n_experts
    for name, steps in streams(E, C, 3):
        ctx = make_ctx(SH, C, policy=policy, fetch=fetch)
        pager = PagerLayer(C=C, E=E, policy=policy)
        want = []
        for R in steps:
            ctx.debug_step_routing(1, R)
            want += [(1, e.step, e.wave, e.expert, e.slot, e.evicted, e.kind) for e in pager.step(R)]
        assert ctx.trace_read() == want, name
        pi_inv, tau, freq, clock = ctx.debug_residency(1)
        assert pi_inv.tolist() == [-1 if e is None else e for e in pager.pi_inv]
        assert tau.tolist() == pager.tau and freq.tolist() == pager.f and clock == pager.c
        assert ctx.debug_verify_pool(1) == 0, name
        s = ctx.layer_stats(1)
        assert (s.hits, s.misses, s.evictions, s.references, s.steps) == (pager.hits, pager.misses, pager.evictions, pager.references, pager.steps)
        assert s.bytes_fetched == pager.misses * SH.expert_bytes
        ctx.close()


@pytest.mark.parametrize("C", [1, 2, 6, 15])
@pytest.mark.parametrize("policy", [0, 1])
@pytest.mark.parametrize("fetch", [0, 2])
def test_hits_first_wave_order_trace_and_state(C, policy, fetch):
    """G25: wisp_set_wave_order(HITS_FIRST) against the oracle's hits-first simulation, bit-exact;
    the step's faults are exactly R minus the residents at step start."""
    E = SH.n_experts
    for name, steps in streams(E, C, 3):
        ctx = make_ctx(SH, C, policy=policy, fetch=fetch, wave_order=1)
        pager = PagerLayer(C=C, E=E, policy=policy, wave_order=1)
        want, closed_form_misses = [], 0
        for R in steps:
            closed_form_misses += len(set(R) - set(pager.pi))
            ctx.debug_step_routing(1, R)
            want += [(1, e.step, e.wave, e.expert, e.slot, e.evicted, e.kind) for e in pager.step(R)]
        assert ctx.trace_read() == want, name
        pi_inv, tau, freq, clock = ctx.debug_residency(1)
        assert pi_inv.tolist() == [-1 if e is None else e for e in pager.pi_inv]
        assert tau.tolist() == pager.tau and freq.tolist() == pager.f and clock == pager.c
        assert ctx.debug_verify_pool(1) == 0, name
        s = ctx.layer_stats(1)
        assert (s.hits, s.misses, s.evictions, s.references, s.steps) == (pager.hits, pager.misses, pager.evictions, pager.references, pager.steps)
        assert s.misses == closed_form_misses
        ctx.close()


def test_set_wave_order_errors_and_switch_back():
    ctx = make_ctx(SH, 2)
    import paper_2606_21868_b200 as wp
    with pytest.raises(wp.WispError):
        ctx.set_wave_order(7)
    pager = PagerLayer(C=2, E=SH.n_experts)
    want = []
    for order, R in ((1, [4, 5]), (1, [0, 1, 5]), (0, [0, 1, 5, 7]), (1, [2, 5, 7])):
        ctx.set_wave_order(order)
        pager.wave_order = order
        ctx.debug_step_routing(0, R)
        want += [(0, e.step, e.wave, e.expert, e.slot, e.evicted, e.kind) for e in pager.step(R)]
    assert ctx.trace_read() == want
    ctx.close()


@pytest.mark.parametrize("policy", [0, 1])
def test_resize_cycle_outputs_unchanged_and_trace(policy):
    """PAPER.md:261 (D2): shrink/grow cycle leaves outputs byte-identical; trace == simulation of the same resize."""
    a = SH.slot_unit_bytes
    hidden = si.gen_decode_hidden(SH, 30, 2)
    ref_ctx = make_ctx(SH, 16, policy=policy, max_tokens=2)
    ref = run_chain(ref_ctx, SH, hidden)
    ref_ctx.close()
    ctx = make_ctx(SH, budget=8 * a, policy=policy, max_tokens=2)
    pagers = [PagerLayer(C=8, E=SH.n_experts, policy=policy) for _ in range(SH.n_layers)]
    want, got_out = [], []
    plan = {0: None, 10: 3, 20: 7, 25: 2}
    for t0 in (0, 10, 20, 25):
        if plan[t0] is not None:
            ctx.set_split(plan[t0] * a, 0)
            for l, p in enumerate(pagers):
                want += [(l, e.step, e.wave, e.expert, e.slot, e.evicted, e.kind) for e in p.resize(plan[t0])]
            for l in range(SH.n_layers):
                assert ctx.debug_verify_pool(l) == 0
        t1 = {0: 10, 10: 20, 20: 25, 25: 30}[t0]
        res = run_chain(ctx, SH, hidden[t0:t1])
        got_out += res
        for per in res:
            for l, rec in enumerate(per):
                want += [(l, e.step, e.wave, e.expert, e.slot, e.evicted, e.kind) for e in pagers[l].step(rec["ids"].flatten().tolist())]
    assert ctx.trace_read() == want
    for pa, pb in zip(ref, got_out):
        for x, y in zip(pa, pb):
            assert torch.equal(x["out"].view(torch.uint8), y["out"].view(torch.uint8))
    st = ctx.stats()
    assert st.resize_count == 3 and st.slots_per_layer == 2
    ctx.close()


def test_failed_resize_keeps_previous_split():
    """'If a resize fails, the engine keeps the previous valid split.'"""
    import paper_2606_21868_b200 as wp
    a, b = SH.slot_unit_bytes, 1 << 16
    ctx = make_ctx(SH, budget=6 * a + 40 * b, kv_block_bytes=b, kv_floor_blocks=8, max_tokens=1)
    st0 = ctx.stats()
    assert st0.slots_per_layer == 6 + (32 * b) // a and st0.kv_blocks >= 8
    C0, k0 = st0.slots_per_layer, st0.kv_blocks
    hidden = si.gen_decode_hidden(SH, 6, 1)
    before = run_chain(ctx, SH, hidden[:3])
    ctx.kv_reserve(20)
    for eb, kb in ((7 * a, 40 * b), (0, 40 * b), (6 * a, 7 * b), (2 * a, 19 * b)):   # over budget; C<1; below floor; below reservations
        with pytest.raises(wp.WispError) as ei:
            ctx.set_split(eb, kb)
        assert ei.value.status == -5
    st = ctx.stats()
    assert (st.slots_per_layer, st.kv_blocks, st.failed_resize_count, st.resize_count) == (C0, k0, 4, 0)
    after = run_chain(ctx, SH, hidden[3:])
    ref_ctx = make_ctx(SH, 16, max_tokens=1)
    ref = run_chain(ref_ctx, SH, hidden)
    for pa, pb in zip(ref, before + after):
        for x, y in zip(pa, pb):
            assert torch.equal(x["out"].view(torch.uint8), y["out"].view(torch.uint8))
    with pytest.raises(wp.WispError):
        ctx.kv_reserve(10 ** 6)
    ctx.kv_reserve(-20)
    ctx.set_split(2 * a, 19 * b)
    assert ctx.stats().slots_per_layer == 2
    ctx.close(); ref_ctx.close()


def test_api_errors():
    import paper_2606_21868_b200 as wp
    with pytest.raises(wp.WispError) as ei:
        wp.Wisp(SH.slot_unit_bytes - 1, n_layers=2, n_experts=16, top_k=2, d_model=256, d_ff=512, max_tokens=1, dtype=0)
    assert ei.value.status == -5
    with pytest.raises(wp.WispError) as ei:
        wp.Wisp(1 << 26, n_layers=2, n_experts=16, top_k=2, d_model=250, d_ff=512, max_tokens=1, dtype=0)
    assert ei.value.status == -1
    ctx = wp.Wisp(4 * SH.slot_unit_bytes, n_layers=2, n_experts=16, top_k=2, d_model=256, d_ff=512, max_tokens=2, dtype=0)
    x = torch.zeros((1, 256), device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    with pytest.raises(wp.WispError) as ei:
        ctx.moe_forward(0, x, x.clone(), st)
    assert ei.value.status == -4                       # forward before registration
    ctx.close()
    ctx = make_ctx(SH, 4, max_tokens=2)
    with pytest.raises(wp.WispError) as ei:
        ctx.moe_forward(0, torch.zeros((3, 256), device="cuda"), torch.zeros((3, 256), device="cuda"), st)
    assert ei.value.status == -1
    with pytest.raises(wp.WispError):
        ctx.moe_forward(5, x, x.clone(), st)
    ctx.close()


def test_trace_ring_overflow_counts_drops():
    ctx = make_ctx(SH, 4, trace_capacity=10)
    for _ in range(4):
        ctx.debug_step_routing(0, [0, 1, 2])
    assert len(ctx.trace_read()) == 9 and ctx.stats().trace_dropped == 3
    ctx.close()


def test_mvwsa_device_histograms_and_proposals():
    rng = random.Random(77)
    E = SH.n_experts
    ctx = make_ctx(SH, 6, kv_block_bytes=1 << 16, budget=12 * SH.slot_unit_bytes, kv_floor_blocks=16)
    ctx.mvwsa_track(True)
    per_layer = [[], []]
    for t in range(120):
        for l in range(2):
            R = rng.sample(range(E), rng.randint(1, 4))
            per_layer[l].append(R)
            ctx.debug_step_routing(l, R)
    want = mvwsa.miss_curve(per_layer, E)
    got = ctx.mvwsa_miss_curve(E + 1)
    assert got == want
    # live law (Eq. 6-8) vs the oracle, on the context's own budget
    st = ctx.stats()
    B, a, b = st.budget_bytes, SH.slot_unit_bytes, 1 << 16
    for p in (0, 20, 100, 400):
        for cmax in (16, 9):
            eb, kb, moved = ctx.mvwsa_propose(mode=0, c_min=2, c_max=cmax, dead_zone=1, headroom=0.2, kv_peak_blocks=p)
            C, kap, mv = mvwsa.live_law(B=B, a=a, b=b, kappa_floor=16, p=p, h=0.2, C_min=2, C_max=cmax, C_cur=st.slots_per_layer, delta=1)
            assert (eb, kb, moved) == (C * a, kap * b, mv)
            assert eb + kb <= B
    # configurator (Eq. 2-5) vs the oracle's exhaustive argmin on the measured curve
    m_kv = [1000.0 / (1 + 0.05 * i) for i in range(200)]
    eb, kb, _ = ctx.mvwsa_propose(mode=1, c_min=2, c_max=16, c_exp=3e-3, c_kv=1e-3, m_kv=m_kv)
    Cw, Bkv = mvwsa.configurator(B=B, a=a, b=b, kappa_floor=16, c_exp=3e-3, c_kv=1e-3, m_exp=want,
                                 m_kv=lambda kap: m_kv[min(kap, len(m_kv) - 1)], C_min=2, C_max=16)
    assert eb == Cw * a and kb == ((B - Cw * a) // b) * b
    ctx.set_split(eb, kb)
    assert ctx.stats().slots_per_layer == Cw
    ctx.close()


@pytest.mark.parametrize("T,slots,n,window,policy", [(1, 5, 2, 1, 0), (4, 6, 3, 2, 0), (2, 4, 2, 2, 1), (1, 16, 2, 1, 0)])
def test_speculative_prefetch_trace_and_outputs(T, slots, n, window, policy):
    """f3 (App. E 402-414): with the online co-activation predictor prefetching n experts per layer, the
    trace -- demand events AND prefetch events (kind 4) -- equals the oracle pager driven by the oracle predictor on the GPU's
    ids, and outputs stay byte-identical to the run without prefetch."""
    import paper_2606_21868_b200 as wp
    from oracle.paging import PagerLayer
    from oracle.predictor import CoActivationPredictor
    shape = si.MoEShape("tiny4", 4, 16, 2, 256, 512, "f32", 1.1)
    hidden = si.gen_decode_hidden(shape, 24, T, rho=0.5, noise=2.0)      # lively routing: the working set moves every step
    ctx = make_ctx(shape, slots, max_tokens=T, fetch=wp.WISP_FETCH_ZEROCOPY, policy=policy)
    ref = run_chain(ctx, shape, hidden)
    ctx.close()
    ctx = make_ctx(shape, slots, max_tokens=T, fetch=wp.WISP_FETCH_ZEROCOPY, policy=policy)
    ctx.set_prefetch(n, 0.5, window)
    res = run_chain(ctx, shape, hidden)
    for pa, pb in zip(ref, res):
        for a, b in zip(pa, pb):
            assert torch.equal(a["out"].view(torch.uint8), b["out"].view(torch.uint8)) and torch.equal(a["ids"], b["ids"])
    pagers = [PagerLayer(C=slots, E=shape.n_experts, policy=policy) for _ in range(shape.n_layers)]
    pred = CoActivationPredictor(shape.n_layers, shape.n_experts, gamma=0.5, window=window)
    want = []
    for per in res:
        pred.begin_pass()
        for l, rec in enumerate(per):
            ids = rec["ids"].flatten().tolist()
            want += [(l, e.step, e.wave, e.expert, e.slot, e.evicted, e.kind) for e in pagers[l].step(ids)]
            pred.observe(l, ids)
            if l + 1 < shape.n_layers:
                picks = pred.predict(l + 1, min(n, slots), resident=pagers[l + 1].pi.keys())
                want += [(l + 1, e.step, e.wave, e.expert, e.slot, e.evicted, e.kind) for e in pagers[l + 1].prefetch(picks)]
    got = ctx.trace_read()
    assert got == want
    st = ctx.stats()
    assert st.prefetches == sum(p.prefetches for p in pagers) and st.total.misses == sum(p.misses for p in pagers)
    assert st.prefetches > 0 or slots >= shape.n_experts
    for l in range(shape.n_layers):
        assert ctx.debug_verify_pool(l) == 0
    # the stack helper takes the same path
    ctx.debug_reset_pool()
    ctx.trace_read()
    fin = run_stack(ctx, shape, hidden)
    for t in range(hidden.shape[0]):
        last = res[t][-1]
        assert torch.equal(fin[t].view(torch.uint8), (last["x"].float() + last["out"].float()).to(shape.torch_dtype).view(torch.uint8))
    assert ctx.trace_read() == want
    ctx.close()
