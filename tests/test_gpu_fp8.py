"""f4: fp8 block-quantised experts through the C ABI vs the oracle's dequantised definition.
Same four parities as the bf16 path: (a) trace, (b) byte identity across budgets / fetch paths, (c) ids, (d) outputs."""
from dataclasses import replace

import pytest
import torch

import synth_inputs as si
from harness import make_ctx, run_chain, run_stack, sim_trace
from test_gpu_parity import assert_same_bytes, check_vs_oracle

pytestmark = pytest.mark.gpu

TOL_F8 = 2e-2                      # bf16 hidden states and outputs: the bf16 path's bound
MED_F8 = si.MoEShape("medium-fp8", 2, 16, 4, 1024, 512, "fp8", 1.1)
BIG_D_F8 = si.MoEShape("two-slab-fp8", 1, 8, 2, 4096, 256, "fp8", 1.1)       # d = 4096: two slabs per 8-row group


@pytest.mark.parametrize("T", [1, 2, 3, 4, 5, 8])
def test_fp8_decode_parities(T):
    shape = MED_F8
    hidden = si.gen_decode_hidden(shape, 10, T)
    ref = None
    for slots, policy, fetch in ((16, 0, 2), (16, 0, 1), (6, 0, 2), (6, 1, 1), (6, 0, 0), (3, 0, 2), (3, 0, 1)):
        ctx = make_ctx(shape, slots, policy=policy, fetch=fetch, max_tokens=T)
        res = run_chain(ctx, shape, hidden)
        routed = [[rec["ids"].flatten().tolist() for rec in per] for per in res]
        want, _ = sim_trace(shape, slots, policy, routed)
        assert ctx.trace_read() == want, "parity (a)"
        for l in range(shape.n_layers):
            assert ctx.debug_verify_pool(l) == 0          # slot bytes == master bytes, scales included
        if ref is None:
            ref = res
            check_vs_oracle(shape, res, TOL_F8)
        else:
            assert_same_bytes(ref, res)
        ctx.close()


def test_fp8_two_slabs_and_stack_helper():
    shape = BIG_D_F8
    hidden = si.gen_decode_hidden(shape, 6, 2)
    ctx = make_ctx(shape, 8, fetch=2, max_tokens=2)
    res = run_chain(ctx, shape, hidden)
    check_vs_oracle(shape, res, TOL_F8)
    ctx2 = make_ctx(shape, 3, fetch=2, max_tokens=2)
    fin = run_stack(ctx2, shape, hidden)
    for t in range(hidden.shape[0]):
        last = res[t][-1]
        want = (last["x"].float() + last["out"].float()).to(torch.bfloat16)
        assert torch.equal(fin[t].view(torch.uint8), want.view(torch.uint8))
    ctx.close(); ctx2.close()


def test_fp8_large_magnitude_hidden_states():
    """Hidden states outside f16's range (|x| up to ~1e5; the router's fixed-point logits bound larger inputs) and far
    below it: the per-token power-of-two scaling keeps the products exact."""
    shape = MED_F8
    hidden = si.gen_decode_hidden(shape, 4, 4) * torch.tensor([3e5, 1e-9, 1.0, 3e4]).view(1, 4, 1)
    ctx = make_ctx(shape, 16, fetch=2, max_tokens=4)
    res = run_chain(ctx, shape, hidden)
    check_vs_oracle(shape, [[per[0]] for per in res], TOL_F8)          # layer 0 sees the scaled inputs themselves
    ctx.close()


def test_fp8_prefill_path():
    shape = MED_F8
    T = 96
    x = si.gen_prefill_hidden(shape, T).view(1, T, shape.d_model)
    ref = None
    for slots, fetch in ((16, 1), (5, 1), (5, 0)):
        ctx = make_ctx(shape, slots, fetch=fetch, max_tokens=T)
        res = run_chain(ctx, shape, x)
        routed = [[rec["ids"].flatten().tolist() for rec in per] for per in res]
        want, _ = sim_trace(shape, slots, 0, routed)
        assert ctx.trace_read() == want
        if ref is None:
            ref = res
            check_vs_oracle(shape, res, TOL_F8)
        else:
            assert_same_bytes(ref, res)
        ctx.close()


def test_fp8_qwen3_layer_shape():
    """The headline shape's quantised variant, 2 layers x 128 experts: budgets 18 slots (configs[1]'s C) and all-resident."""
    shape = si.QWEN3_FP8.with_layers(2)
    hidden = si.gen_decode_hidden(shape, 6, 1)
    ctx = make_ctx(shape, 128, fetch=2, max_tokens=1)
    ref = run_chain(ctx, shape, hidden)
    check_vs_oracle(shape, ref, TOL_F8)
    ctx.close()
    ctx = make_ctx(shape, 18, fetch=2, max_tokens=1)
    res = run_chain(ctx, shape, hidden)
    assert_same_bytes(ref, res)
    for l in range(shape.n_layers):
        assert ctx.debug_verify_pool(l) == 0
    ctx.close()
