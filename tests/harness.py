"""Shared GPU-test harness: builds a Wisp context from synthetic inputs and drives the residual chain
(O3 semantics) through the C ABI.  Holds no method arithmetic: residual adds go through
wisp_residual_add, everything else through wisp_moe_forward / wisp_stack_forward."""
from __future__ import annotations

import torch

import synth_inputs as si

_MODEL_CACHE = {}


def model(shape):
    if shape not in _MODEL_CACHE:
        _MODEL_CACHE[shape] = si.gen_model(shape)
    return _MODEL_CACHE[shape]


def make_ctx(shape, slots=None, *, budget=None, policy=0, fetch=1, max_tokens=8, kv_block_bytes=0, kv_floor_blocks=0,
             trace=True, trace_capacity=0, wave_order=0):
    import paper_2606_21868_b200 as wp
    if budget is None:
        budget = slots * shape.slot_unit_bytes + kv_floor_blocks * kv_block_bytes
    ctx = wp.Wisp(budget, n_layers=shape.n_layers, n_experts=shape.n_experts, top_k=shape.top_k, d_model=shape.d_model,
                  d_ff=shape.d_ff, max_tokens=max_tokens,
                  dtype={"f32": wp.WISP_F32, "bf16": wp.WISP_BF16, "fp8": wp.WISP_FP8_E4M3}[shape.dtype],
                  policy=policy, fetch=fetch, kv_block_bytes=kv_block_bytes, kv_floor_blocks=kv_floor_blocks,
                  trace_capacity=trace_capacity)
    experts, routers = model(shape)
    for l in range(shape.n_layers):
        ctx.register_host_experts(l, experts[l], routers[l][0], routers[l][1])
    if trace:
        ctx.trace_enable(True)
    if wave_order:
        ctx.set_wave_order(wave_order)
    return ctx


def run_chain(ctx, shape, hidden, *, collect=True):
    """hidden [n_steps, T, d] fp32 (host).  Per step: x_0 = cast(h); per layer y = MoE(x); x <- x + y.
    Returns list over steps of list over layers of dict(x, out, ids, w) with host tensors."""
    dev = torch.device("cuda")
    st = torch.cuda.current_stream().cuda_stream
    n_steps, T, d = hidden.shape
    res = []
    for t in range(n_steps):
        x = hidden[t].to(shape.torch_dtype).to(dev)
        per = []
        for l in range(shape.n_layers):
            out = torch.empty_like(x)
            ctx.moe_forward(l, x, out, st)
            xn = torch.empty_like(x)
            ctx.residual_add(x, out, xn, st)
            if collect:
                ids, w = ctx.last_topk(l)
                per.append(dict(x=x.cpu(), out=out.cpu(), ids=torch.from_numpy(ids).long(), w=torch.from_numpy(w)))
            x = xn
        torch.cuda.synchronize()
        res.append(per if collect else x.cpu())
    return res


def run_stack(ctx, shape, hidden):
    """Same chain through wisp_stack_forward; returns final hidden per step (host)."""
    dev = torch.device("cuda")
    s = torch.cuda.Stream()
    outs = []
    with torch.cuda.stream(s):
        for t in range(hidden.shape[0]):
            x = hidden[t].to(shape.torch_dtype).to(dev)
            y = torch.empty_like(x)
            ctx.stack_forward(x, y, s.cuda_stream)
            s.synchronize()
            outs.append(y.cpu())
    return outs


def sim_trace(shape, slots, policy, routed_per_step_layer, resize_at=None, wave_order=0):
    """Oracle O4 simulation fed the GPU's routing.  routed_per_step_layer[t][l] = iterable of ids.
    Returns events as tuples matching Wisp.trace_read()."""
    from oracle.paging import PagerLayer
    pagers = [PagerLayer(C=slots, E=shape.n_experts, policy=policy, wave_order=wave_order) for _ in range(shape.n_layers)]
    ev = []
    for t, per in enumerate(routed_per_step_layer):
        for l, ids in enumerate(per):
            for e in pagers[l].step(ids):
                ev.append((l, e.step, e.wave, e.expert, e.slot, e.evicted, e.kind))
    return ev, pagers
