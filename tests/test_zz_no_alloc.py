"""wisp_route_noalloc (the allocation-free router entry point, include/wisp.h) against the existing context path
(wisp_moe_forward -> wisp_last_logits / wisp_last_topk), on two calls in a row.  Collected last on purpose (file name)."""
import pytest
import torch

import synth_inputs as si
from harness import make_ctx, model

pytestmark = pytest.mark.gpu

MED = si.MoEShape("medium-bf16", 2, 32, 4, 512, 768, "bf16", 1.1)


@pytest.mark.parametrize("shape,T", [(si.TINY, 4), (MED, 8)])
def test_route_noalloc_matches_context_path_twice(shape, T):
    import paper_2606_21868_b200 as wp
    dtype = wp.WISP_F32 if shape.dtype == "f32" else wp.WISP_BF16
    E, k, d = shape.n_experts, shape.top_k, shape.d_model
    _, routers = model(shape)
    w_r, bias = routers[0][0].cuda(), routers[0][1].cuda()
    ctx = make_ctx(shape, E, fetch=1, max_tokens=T, trace=False)
    hidden = si.gen_decode_hidden(shape, 3, T)
    st = torch.cuda.current_stream().cuda_stream
    z = torch.empty((T, E), dtype=torch.float32, device="cuda")
    ids = torch.empty((T, k), dtype=torch.int32, device="cuda")
    w = torch.empty((T, k), dtype=torch.float32, device="cuda")
    # calls 1 and 2: full batch, different inputs; call 3: fewer tokens (stale sums of call 2 lie behind the words it clears)
    for step, n in ((0, T), (1, T), (2, max(1, T // 2))):
        x = hidden[step, :n].to(shape.torch_dtype).cuda().contiguous()
        out = torch.empty_like(x)
        ctx.moe_forward(0, x, out, st)
        z_ref = torch.from_numpy(ctx.last_logits(n))
        ids_ref, w_ref = ctx.last_topk(0)
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        wp.route_noalloc(x, w_r, bias, k, dtype, z[:n], ids[:n], w[:n], st)
        torch.cuda.synchronize()
        if step > 0:
            assert torch.cuda.mem_get_info()[0] == free0, "the entry point allocated device memory"
        assert torch.equal(ids[:n].cpu().long(), torch.from_numpy(ids_ref[:n]).long())
        # the test suite's tolerance for routing weights (test_gpu_parity.check_vs_oracle) -- the two paths run the same arithmetic,
        # so the bits agree as well
        assert torch.allclose(z[:n].cpu(), z_ref, rtol=0, atol=1e-5)
        assert torch.allclose(w[:n].cpu(), torch.from_numpy(w_ref[:n]), rtol=0, atol=1e-5)
        assert torch.equal(z[:n].cpu(), z_ref) and torch.equal(w[:n].cpu(), torch.from_numpy(w_ref[:n]))
    ctx.close()


def test_route_noalloc_no_bias_and_no_logits_output():
    import paper_2606_21868_b200 as wp
    shape = si.TINY
    _, routers = model(shape)
    w_r = routers[0][0].cuda()
    x = si.gen_decode_hidden(shape, 1, 2)[0].cuda().contiguous()
    st = torch.cuda.current_stream().cuda_stream
    ids = torch.empty((2, shape.top_k), dtype=torch.int32, device="cuda")
    w = torch.empty((2, shape.top_k), dtype=torch.float32, device="cuda")
    wp.route_noalloc(x, w_r, None, shape.top_k, wp.WISP_F32, None, ids, w, st)
    torch.cuda.synchronize()
    zs = x.double().cpu() @ routers[0][0].double().T                   # plain definition, bias = 0
    want = torch.sort(zs, dim=1, descending=True, stable=True).indices[:, :shape.top_k]
    gap = torch.sort(zs, dim=1, descending=True).values
    clear = (gap[:, shape.top_k - 1] - gap[:, shape.top_k]) > 1e-4
    assert torch.equal(ids.cpu().long()[clear], want[clear])
    assert torch.allclose(w.sum(dim=1).cpu(), torch.ones(2), atol=1e-5)


def test_route_noalloc_rejects_sizes_beyond_the_static_scratch():
    import paper_2606_21868_b200 as wp
    E, d, k = 1024, 256, 2
    x = torch.zeros((9, d), dtype=torch.float32, device="cuda")         # 9 * 1024 > 8192 accumulators
    w_r = torch.zeros((E, d), dtype=torch.float32, device="cuda")
    ids = torch.empty((9, k), dtype=torch.int32, device="cuda")
    w = torch.empty((9, k), dtype=torch.float32, device="cuda")
    with pytest.raises(wp.WispError) as ei:
        wp.route_noalloc(x, w_r, None, k, wp.WISP_F32, None, ids, w, torch.cuda.current_stream().cuda_stream)
    assert ei.value.status == -1
    wp.route_noalloc(x[:8], w_r, None, k, wp.WISP_F32, None, ids[:8], w[:8], torch.cuda.current_stream().cuda_stream)   # exactly the maximum
    torch.cuda.synchronize()
    assert torch.equal(ids[:8].cpu(), torch.tensor([[0, 1]] * 8, dtype=torch.int32))       # all-equal logits: ids ascending
