"""GPU parity tests proper (-m gpu): the CUDA path through the C ABI vs the oracle.
(a) trace bit-exact vs the O4 simulation on the GPU's routing; (b) outputs byte-identical across budgets,
policies and fetch paths; (c) ids equal the oracle's where the k-th/(k+1)-th logit gap > 1e-4;
(d) max|gpu - cpu| / max|cpu| <= 1e-5 (fp32), 2e-2 (bf16)."""
import pytest
import torch

import synth_inputs as si
from harness import make_ctx, model, run_chain, run_stack, sim_trace
from oracle import moe_forward as mf

pytestmark = pytest.mark.gpu

TOL = {"f32": 1e-5, "bf16": 2e-2}
MED = si.MoEShape("medium-bf16", 2, 32, 4, 512, 768, "bf16", 1.1)


def check_vs_oracle(shape, res, tol):
    """Teacher-forced per layer (O3): recompute layer l from the exact x bits the GPU consumed."""
    experts, routers = model(shape)
    worst = 0.0
    for per in res:
        for l, rec in enumerate(per):
            out, ids, w, z = mf.moe_layer(rec["x"], experts[l], routers[l][0], routers[l][1], shape.top_k, shape.d_ff)
            zs = torch.sort(z, dim=1, descending=True).values
            clear = (zs[:, shape.top_k - 1] - zs[:, shape.top_k]) > 1e-4 if shape.top_k < shape.n_experts else torch.ones(z.shape[0], dtype=torch.bool)
            assert torch.equal(rec["ids"][clear], ids[clear]), "parity (c): top-k ids"          # (c)
            if not bool(clear.all()):   # near-tie: either id set is correct; force the GPU's routing
                out, _, w, _ = mf.moe_layer(rec["x"], experts[l], routers[l][0], routers[l][1], shape.top_k, shape.d_ff, ids=rec["ids"])
            assert torch.allclose(rec["w"].double(), w, atol=1e-5)
            err = (rec["out"].double() - out).abs().max().item() / out.abs().max().item()
            worst = max(worst, err)
            assert err <= tol, f"parity (d): layer {l} rel err {err}"                             # (d)
    return worst


def outs_bytes(res):
    return [[rec["out"].contiguous().view(torch.uint8) for rec in per] for per in res]


def assert_same_bytes(a, b):
    for pa, pb in zip(outs_bytes(a), outs_bytes(b)):
        for x, y in zip(pa, pb):
            assert torch.equal(x, y), "parity (b): outputs differ across budgets"


def test_config1_tiny_decode_all_four_parities():
    shape = si.TINY
    hidden = si.gen_decode_hidden(shape, 128, 1)
    ref = None
    for slots, policy, fetch in ((16, 0, 1), (6, 0, 1), (6, 0, 0), (6, 0, 2), (6, 1, 1), (2, 0, 1), (2, 0, 2), (1, 1, 2)):
        ctx = make_ctx(shape, slots, policy=policy, fetch=fetch)
        res = run_chain(ctx, shape, hidden)
        routed = [[rec["ids"].flatten().tolist() for rec in per] for per in res]
        want, pagers = sim_trace(shape, slots, policy, routed)
        got = ctx.trace_read()
        assert got == want, "parity (a): trace"                                                   # (a)
        st = ctx.stats()
        assert st.total.hits == sum(p.hits for p in pagers) and st.total.misses == sum(p.misses for p in pagers)
        assert st.total.evictions == sum(p.evictions for p in pagers)
        assert st.total.hits + st.total.misses == st.total.references
        for l in range(shape.n_layers):
            assert ctx.debug_verify_pool(l) == 0                                                  # slot bytes == master bytes
        if ref is None:
            ref = res
            check_vs_oracle(shape, res, TOL["f32"])
        else:
            assert_same_bytes(ref, res)                                                           # (b)
        ctx.close()


def test_config1_free_running_oracle_and_stack_helper():
    shape = si.TINY
    hidden = si.gen_decode_hidden(shape, 16, 1)
    experts, routers = model(shape)
    ctx = make_ctx(shape, 6)
    res = run_chain(ctx, shape, hidden)
    ctx2 = make_ctx(shape, 6)
    fin = run_stack(ctx2, shape, hidden)
    for t in range(hidden.shape[0]):
        xL, per = mf.stack_forward(hidden[t], experts, routers, shape.top_k, shape.d_ff, shape.torch_dtype)
        last = res[t][-1]
        gpu_xL = (last["x"].float() + last["out"].float()).to(shape.torch_dtype)
        assert torch.allclose(gpu_xL.double(), xL.double(), rtol=0, atol=1e-5 * xL.abs().max().item() * 4)
        assert torch.equal(fin[t].view(torch.uint8), gpu_xL.view(torch.uint8)), "stack helper != per-layer chain"
    assert ctx.trace_read() == ctx2.trace_read()
    ctx.close(); ctx2.close()


@pytest.mark.parametrize("T", [4, 8])
def test_batch_decode_overflow_waves(T):
    """Batch > 1 incl. overflow (|R| > C, C < k): waves, staging, ordered combine (a5)."""
    shape = si.TINY
    hidden = si.gen_decode_hidden(shape, 12, T)
    ref = None
    for slots, fetch in ((16, 1), (5, 1), (5, 2), (1, 1), (1, 2), (3, 0)):
        ctx = make_ctx(shape, slots, max_tokens=T, fetch=fetch)
        res = run_chain(ctx, shape, hidden)
        routed = [[rec["ids"].flatten().tolist() for rec in per] for per in res]
        want, _ = sim_trace(shape, slots, 0, routed)
        assert ctx.trace_read() == want
        for l in range(shape.n_layers):
            assert ctx.debug_verify_pool(l) == 0
        if ref is None:
            ref = res
            check_vs_oracle(shape, res, TOL["f32"])
        else:
            assert_same_bytes(ref, res)
        ctx.close()


@pytest.mark.parametrize("policy", [0, 1])
@pytest.mark.parametrize("T", [4, 8])
def test_hits_first_waves_outputs_unchanged(T, policy):
    """G25: the wave order never changes outputs, the trace equals the hits-first simulation, and an
    overflowing workload faults no more than under ascending waves.  Multi-kernel path and persistent kernel."""
    shape = si.TINY
    hidden = si.gen_decode_hidden(shape, 12, T)
    ctx = make_ctx(shape, 16, max_tokens=T)
    ref = run_chain(ctx, shape, hidden)
    ctx.close()
    ctx = make_ctx(shape, 16, max_tokens=T, fetch=2)
    ref_stack = run_stack(ctx, shape, hidden)
    ctx.close()
    routed = [[rec["ids"].flatten().tolist() for rec in per] for per in ref]
    for slots, fetch in ((5, 1), (5, 2), (1, 2), (3, 0)):
        want, pagers = sim_trace(shape, slots, policy, routed, wave_order=1)
        if policy == 0:     # per step from the same state this is a theorem; over this seeded LRU trajectory it is checked as measured
            _, asc = sim_trace(shape, slots, policy, routed)
            assert sum(p.misses for p in pagers) <= sum(p.misses for p in asc)
        ctx = make_ctx(shape, slots, max_tokens=T, fetch=fetch, wave_order=1, policy=policy)
        assert_same_bytes(ref, run_chain(ctx, shape, hidden))
        assert ctx.trace_read() == want
        for l in range(shape.n_layers):
            assert ctx.debug_verify_pool(l) == 0
        ctx.close()
        ctx = make_ctx(shape, slots, max_tokens=T, fetch=fetch, wave_order=1, policy=policy)
        got = run_stack(ctx, shape, hidden)
        assert all(torch.equal(a.view(torch.uint8), b.view(torch.uint8)) for a, b in zip(ref_stack, got))
        assert ctx.trace_read() == want
        ctx.close()


def test_hits_first_prefill_outputs_unchanged():
    shape, T = MED, 96
    hidden = si.gen_prefill_hidden(shape, T).view(1, T, shape.d_model)
    ctx = make_ctx(shape, shape.n_experts, max_tokens=T)
    ref = run_chain(ctx, shape, hidden)
    ctx.close()
    routed = [[rec["ids"].flatten().tolist() for rec in per] for per in ref]
    for slots, fetch in ((5, 1), (3, 2)):
        # two passes over the same batch: the second starts with residents, where the two orders differ
        ctx = make_ctx(shape, slots, fetch=fetch, max_tokens=T, wave_order=1)
        assert_same_bytes(ref, run_chain(ctx, shape, hidden))
        assert_same_bytes(ref, run_chain(ctx, shape, hidden))
        want, pagers = sim_trace(shape, slots, 0, routed + routed, wave_order=1)
        _, asc = sim_trace(shape, slots, 0, routed + routed)
        assert ctx.trace_read() == want
        assert sum(p.misses for p in pagers) < sum(p.misses for p in asc)
        ctx.close()


@pytest.mark.parametrize("shape,T", [(si.TINY, 40), (MED, 96)])
def test_prefill_grouped_path(shape, T):
    hidden = si.gen_prefill_hidden(shape, T).view(1, T, shape.d_model)
    ref = None
    for slots, fetch in ((shape.n_experts, 1), (5, 1), (5, 0), (3, 1), (3, 2)):
        ctx = make_ctx(shape, slots, fetch=fetch, max_tokens=T)
        res = run_chain(ctx, shape, hidden)
        routed = [[rec["ids"].flatten().tolist() for rec in per] for per in res]
        want, _ = sim_trace(shape, slots, 0, routed)
        assert ctx.trace_read() == want
        if ref is None:
            ref = res
            check_vs_oracle(shape, res, TOL[shape.dtype])
        else:
            assert_same_bytes(ref, res)
        ctx.close()


def test_bf16_decode_medium_shape():
    shape = MED
    hidden = si.gen_decode_hidden(shape, 24, 2)
    ref = None
    for slots, policy, fetch in ((32, 0, 1), (9, 0, 1), (9, 1, 2), (3, 0, 2), (3, 0, 0)):
        ctx = make_ctx(shape, slots, policy=policy, fetch=fetch)
        res = run_chain(ctx, shape, hidden)
        routed = [[rec["ids"].flatten().tolist() for rec in per] for per in res]
        want, _ = sim_trace(shape, slots, policy, routed)
        assert ctx.trace_read() == want
        for l in range(shape.n_layers):
            assert ctx.debug_verify_pool(l) == 0
        if ref is None:
            ref = res
            worst = check_vs_oracle(shape, res, TOL["bf16"])
            assert worst < 1e-2
        else:
            assert_same_bytes(ref, res)
        ctx.close()


def test_degenerate_inputs():
    shape = si.TINY
    ctx = make_ctx(shape, 6)
    st = torch.cuda.current_stream().cuda_stream
    x = torch.zeros((1, shape.d_model), device="cuda")
    out = torch.full_like(x, 7.0)
    ctx.moe_forward(0, x, out, st)
    torch.cuda.synchronize()
    assert torch.equal(out.cpu().view(torch.int32), torch.zeros((1, shape.d_model), dtype=torch.int32)), "x = 0 -> +0"
    before = ctx.layer_stats(0).steps
    ctx.moe_forward(0, x[:0], out[:0], st)           # n_tokens = 0: no-op, no tick (G23)
    assert ctx.layer_stats(0).steps == before
    ctx.close()


@pytest.mark.parametrize("T", [1, 4])
def test_static_layer_offload_arm(T):
    """f2: the static layer-offload comparison arm streams whole expert layers and runs the SAME kernels:
    outputs byte-identical to the paged pool, streamed bytes equal the oracle's byte model."""
    import paper_2606_21868_b200 as wp
    from oracle.paging import static_offload_bytes_per_forward
    shape = si.TINY
    hidden = si.gen_decode_hidden(shape, 6, T)
    ctx = make_ctx(shape, 16, max_tokens=T)
    ref = run_chain(ctx, shape, hidden)
    ref_stack = run_stack(ctx, shape, hidden)
    ctx.close()
    layer_bytes = shape.n_experts * shape.expert_bytes
    for n_layers_budget in (2, 3, 4):                       # 0, 1, 2 resident layers of 2
        budget = n_layers_budget * layer_bytes
        ctx = make_ctx(shape, budget=budget, fetch=wp.WISP_FETCH_STATIC, max_tokens=T, trace=False)
        assert_same_bytes(ref, run_chain(ctx, shape, hidden))
        per_fwd = static_offload_bytes_per_forward(shape.n_layers, shape.n_experts, shape.expert_bytes, budget)
        assert ctx.stats().total.bytes_fetched == per_fwd * hidden.shape[0]
        got = run_stack(ctx, shape, hidden)
        assert all(torch.equal(a.view(torch.uint8), b.view(torch.uint8)) for a, b in zip(ref_stack, got))
        st = ctx.stats()
        assert st.total.bytes_fetched == 2 * per_fwd * hidden.shape[0] and st.total.misses == 0
        with pytest.raises(wp.WispError):
            ctx.set_split(layer_bytes, 0)
        ctx.close()
    with pytest.raises(wp.WispError):                       # less than the two bounce buffers
        make_ctx(shape, budget=layer_bytes, fetch=wp.WISP_FETCH_STATIC, max_tokens=T, trace=False)


def test_wide_topk_fused_route_without_a_spare_warp():
    """T * k = 256 > 224: the fused kernel's route step cannot give warp 7 to the x reload (all eight warps select, then warp 7
    loads): same four parities, fused vs split vs oracle."""
    shape = si.MoEShape("wide-k", 2, 64, 32, 256, 256, "f32", 1.1)
    hidden = si.gen_decode_hidden(shape, 6, 8)
    ref = None
    for slots, fetch in ((64, 2), (64, 1), (40, 2)):
        ctx = make_ctx(shape, slots, max_tokens=8, fetch=fetch)
        res = run_chain(ctx, shape, hidden)
        routed = [[rec["ids"].flatten().tolist() for rec in per] for per in res]
        want, _ = sim_trace(shape, slots, 0, routed)
        assert ctx.trace_read() == want
        if ref is None:
            ref = res
            check_vs_oracle(shape, res, TOL["f32"])
        else:
            assert_same_bytes(ref, res)
        ctx2 = make_ctx(shape, slots, max_tokens=8, fetch=fetch)
        fin = run_stack(ctx2, shape, hidden)                                       # all layers in one launch: the reload path
        for t in range(hidden.shape[0]):
            last = res[t][-1]
            want_x = (last["x"].float() + last["out"].float()).to(shape.torch_dtype)
            assert torch.equal(fin[t].view(torch.uint8), want_x.view(torch.uint8))
        ctx.close(); ctx2.close()


@pytest.mark.parametrize("T", [3, 5, 6, 7])
def test_odd_batch_sizes_fused_vs_split(T):
    """Token counts that are not a multiple of the combine batch (4): the fused kernel combines 4 + 1, 4 + 2, 4 + 3 or 3 tokens per
    column block; the x-ready and accumulator counts must still add up.  bf16 (MMA path) and fp32, fused vs split vs oracle."""
    for shape in (MED, si.TINY):
        hidden = si.gen_decode_hidden(shape, 6, T)
        E = shape.n_experts
        ref = None
        for slots, fetch in ((E, 2), (E, 1), (max(shape.top_k, E // 3), 2)):
            ctx = make_ctx(shape, slots, max_tokens=T, fetch=fetch)
            res = run_chain(ctx, shape, hidden)
            routed = [[rec["ids"].flatten().tolist() for rec in per] for per in res]
            want, _ = sim_trace(shape, slots, 0, routed)
            assert ctx.trace_read() == want
            if ref is None:
                ref = res
                check_vs_oracle(shape, res, TOL[shape.dtype])
            else:
                assert_same_bytes(ref, res)
            ctx2 = make_ctx(shape, slots, max_tokens=T, fetch=fetch)
            fin = run_stack(ctx2, shape, hidden)                                   # all layers in one launch: reload + polls
            for t in range(hidden.shape[0]):
                last = res[t][-1]
                want_x = (last["x"].float() + last["out"].float()).to(shape.torch_dtype)
                assert torch.equal(fin[t].view(torch.uint8), want_x.view(torch.uint8))
            ctx.close(); ctx2.close()
