"""GPU parity at BASELINE.json's FULL layer shapes, in the launch configuration bench.py times (fused fetch, persistent
decode kernel through wisp_stack_forward; tcgen05 grouped GEMM for prefill).  The layer count is reduced (the shapes
of one layer are the config's), and the oracle is evaluated on every decode token / on sampled prefill tokens."""
import pytest
import torch

import synth_inputs as si
from harness import make_ctx, model, run_chain, run_stack, sim_trace
from oracle import moe_forward as mf
from test_gpu_parity import TOL, assert_same_bytes, check_vs_oracle

pytestmark = pytest.mark.gpu

QWEN2L = si.QWEN3.with_layers(2)
MIXTRAL1L = si.MIXTRAL.with_layers(1)


def gen_dev_model(shape):
    """harness.model() with the weights drawn on the GPU (the CPU generator is too slow at these sizes)."""
    import harness
    if shape not in harness._MODEL_CACHE:
        harness._MODEL_CACHE[shape] = si.gen_model(shape, device="cuda")
    return harness._MODEL_CACHE[shape]


def test_qwen3_shape_decode_bench_config():
    shape = QWEN2L
    gen_dev_model(shape)
    hidden = si.gen_decode_hidden(shape, 12, 1)
    ref = None
    ref_stack = None
    for slots, fetch in ((18, 2), (128, 2), (9, 1)):           # 8 GiB-equivalent pool, all-resident, 4 GiB-equivalent
        ctx = make_ctx(shape, slots, fetch=fetch, max_tokens=1)
        res = run_chain(ctx, shape, hidden)
        routed = [[rec["ids"].flatten().tolist() for rec in per] for per in res]
        want, _ = sim_trace(shape, slots, 0, routed)
        assert ctx.trace_read() == want                          # (a)
        for l in range(shape.n_layers):
            assert ctx.debug_verify_pool(l) == 0
        if ref is None:
            ref = res
            worst = check_vs_oracle(shape, res, TOL["bf16"])   # (c), (d), teacher-forced
            assert worst < 1e-2
        else:
            assert_same_bytes(ref, res)                          # (b)
        ctx.close()
        # the call bench.py times: one persistent launch per token
        ctx = make_ctx(shape, slots, fetch=fetch, max_tokens=1, trace=False)
        outs = run_stack(ctx, shape, hidden)
        if ref_stack is None:
            ref_stack = outs
            last = [per[-1] for per in ref]
            for t, y in enumerate(outs):                         # stack helper == per-layer chain, bit for bit
                xn = (last[t]["x"].float() + last[t]["out"].float()).to(shape.torch_dtype)
                assert torch.equal(y.view(torch.uint8), xn.view(torch.uint8))
        else:
            for y0, y1 in zip(ref_stack, outs):
                assert torch.equal(y0.view(torch.uint8), y1.view(torch.uint8))
        ctx.close()


def test_qwen3_shape_batch4_decode():
    shape = QWEN2L
    gen_dev_model(shape)
    hidden = si.gen_decode_hidden(shape, 6, 4)
    ref = None
    for slots, fetch in ((128, 2), (9, 2), (37, 1)):             # C = 9 < |R|: overflow waves in decode
        ctx = make_ctx(shape, slots, fetch=fetch, max_tokens=4)
        res = run_chain(ctx, shape, hidden)
        routed = [[rec["ids"].flatten().tolist() for rec in per] for per in res]
        want, _ = sim_trace(shape, slots, 0, routed)
        assert ctx.trace_read() == want
        if ref is None:
            ref = res
            assert check_vs_oracle(shape, res, TOL["bf16"]) < 1e-2
        else:
            assert_same_bytes(ref, res)
        ctx.close()
    # G25: hits-first waves at the same shape (C = 9 < |R|), multi-kernel path and persistent kernel
    want, pagers = sim_trace(shape, 9, 0, routed, wave_order=1)
    _, asc = sim_trace(shape, 9, 0, routed)
    assert sum(p.misses for p in pagers) < sum(p.misses for p in asc)
    ctx = make_ctx(shape, 9, fetch=2, max_tokens=4, wave_order=1)
    assert_same_bytes(ref, run_chain(ctx, shape, hidden))
    assert ctx.trace_read() == want
    ctx.close()
    ctx = make_ctx(shape, 128, fetch=2, max_tokens=4, trace=False)
    ref_stack = run_stack(ctx, shape, hidden)
    ctx.close()
    ctx = make_ctx(shape, 9, fetch=2, max_tokens=4, wave_order=1)
    got = run_stack(ctx, shape, hidden)
    assert all(torch.equal(a.view(torch.uint8), b.view(torch.uint8)) for a, b in zip(ref_stack, got))
    assert ctx.trace_read() == want
    for l in range(shape.n_layers):
        assert ctx.debug_verify_pool(l) == 0
    ctx.close()


def test_qwen3_shape_prefill_sampled_tokens():
    shape = si.QWEN3.with_layers(1)
    experts, routers = gen_dev_model(shape)
    T = 2048
    x = si.gen_prefill_hidden(shape, T).to(shape.torch_dtype)
    outs = []
    for slots in (128, 37):                                       # all-resident and 16 GiB-equivalent (overflow waves)
        ctx = make_ctx(shape, slots, fetch=1, max_tokens=T, trace=False)
        xd = x.cuda()
        out = torch.empty_like(xd)
        ctx.moe_forward(0, xd, out, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        ids, w = ctx.last_topk(0)
        outs.append(out.cpu())
        assert ctx.debug_verify_pool(0) == 0
        ctx.close()
    assert torch.equal(outs[0].view(torch.uint8), outs[1].view(torch.uint8))   # (b) across budgets
    sample = torch.arange(0, T, 128).tolist() + [1, T - 1]
    xs = x[sample]
    ref, rids, rw, z = mf.moe_layer(xs, experts[0], routers[0][0], routers[0][1], shape.top_k, shape.d_ff)
    gids = torch.from_numpy(ids).long()[sample]
    zs = torch.sort(z, dim=1, descending=True).values
    clear = (zs[:, shape.top_k - 1] - zs[:, shape.top_k]) > 1e-4
    assert torch.equal(gids[clear], rids[clear])                  # (c)
    if not bool(clear.all()):
        ref, _, _, _ = mf.moe_layer(xs, experts[0], routers[0][0], routers[0][1], shape.top_k, shape.d_ff, ids=gids)
    err = (outs[0][sample].double() - ref).abs().max().item() / ref.abs().max().item()
    assert err <= TOL["bf16"], err                                # (d)


def test_mixtral_shape_decode():
    shape = MIXTRAL1L
    gen_dev_model(shape)
    hidden = si.gen_decode_hidden(shape, 4, 1)
    ref = None
    for slots, fetch in ((2, 2), (8, 2)):                         # 24 GiB -> C = 2 = k, and all-resident
        ctx = make_ctx(shape, slots, fetch=fetch, max_tokens=1)
        res = run_chain(ctx, shape, hidden)
        routed = [[rec["ids"].flatten().tolist() for rec in per] for per in res]
        want, _ = sim_trace(shape, slots, 0, routed)
        assert ctx.trace_read() == want
        if ref is None:
            ref = res
            assert check_vs_oracle(shape, res, TOL["bf16"]) < 1e-2
        else:
            assert_same_bytes(ref, res)
        ctx.close()
    import harness
    harness._MODEL_CACHE.pop(shape, None)                         # 2.6 GiB of host weights
