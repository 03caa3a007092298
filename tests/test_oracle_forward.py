"""Pins for oracle O1-O3 (router/top-k/softmax, SwiGLU FFN, combine): SURVEY.md §8(c) P1, P2, P8."""
import itertools
import math

import pytest
import torch

import synth_inputs as si
from golden_util import num, read_golden
from oracle import moe_forward as mf

G = {k: num(v) for k, v in read_golden("hand_router_ffn.txt").items()}
F64 = torch.float64


def test_p1_hand_topk_softmax():
    ids, w = mf.topk_softmax(torch.tensor([[1.0, 3.0, 2.0, 0.0]], dtype=F64), 2)
    assert ids.tolist() == [[G["p1_id0"], G["p1_id1"]]]
    assert w[0, 0].item() == pytest.approx(G["p1_w0"], abs=1e-9)
    assert w[0, 1].item() == pytest.approx(G["p1_w1"], abs=1e-9)


def _expert_blob(g, u, d):
    return torch.cat([torch.tensor(m, dtype=F64).flatten() for m in (g, u, d)])


def test_p2_hand_ffn_and_combine():
    x = torch.tensor([[1.0, 2.0]], dtype=F64)
    A = ([[1, 0], [0, 1]], [[1, 1], [0, 1]], [[1, 0], [1, 1]])
    B = ([[-1, 0], [0, -1]], [[1, 0], [0, 1]], [[1, 0], [0, 1]])
    yA = mf.expert_ffn(x, *(torch.tensor(m, dtype=F64) for m in A))[0]
    yB = mf.expert_ffn(x, *(torch.tensor(m, dtype=F64) for m in B))[0]
    assert yA.tolist() == pytest.approx([G["p2_yA0"], G["p2_yA1"]], abs=1e-9)
    assert yB.tolist() == pytest.approx([G["p2_yB0"], G["p2_yB1"]], abs=1e-9)
    # layer: 4 experts, router rows chosen so that logits = (1, 3, 2, 0): expert 1 = A, expert 2 = B
    zero = ([[0, 0], [0, 0]],) * 3
    experts = torch.stack([_expert_blob(*zero), _expert_blob(*A), _expert_blob(*B), _expert_blob(*zero)])
    w_r = torch.zeros((4, 2), dtype=F64)
    bias = torch.tensor([1.0, 3.0, 2.0, 0.0])
    out, ids, w, _ = mf.moe_layer(x, experts, w_r, bias, k=2, d_ff=2)
    assert ids.tolist() == [[1, 2]]
    assert out[0].tolist() == pytest.approx([G["p2_out0"], G["p2_out1"]], abs=1e-9)
    # a transposed D or swapped gate/up would change these numbers: the case is asymmetric on purpose
    assert abs(G["p2_yA0"] - G["p2_yA1"]) > 1


def test_topk_brute_force_and_invariants():
    g = torch.Generator().manual_seed(7)
    for E, k in ((4, 2), (16, 2), (128, 8), (256, 8), (8, 8)):
        z = torch.randn((64, E), dtype=F64, generator=g)
        z[3, :] = z[3, 0]                 # full tie row
        z[5, 1] = z[5, 0]                 # partial tie
        ids, w = mf.topk_softmax(z, k)
        for t in range(z.shape[0]):
            brute = sorted(range(E), key=lambda e: (-z[t, e].item(), e))[:k]
            assert ids[t].tolist() == brute
            assert len(set(brute)) == k
            zs = [z[t, e].item() for e in brute]
            den = sum(math.exp(v - zs[0]) for v in zs)
            assert w[t].tolist() == pytest.approx([math.exp(v - zs[0]) / den for v in zs], abs=1e-12)
        assert torch.allclose(w.sum(1), torch.ones(64, dtype=F64), atol=1e-12)
        # renormalised full softmax == softmax over the selected logits
        full = torch.softmax(z, dim=1)
        sel = torch.gather(full, 1, ids)
        assert torch.allclose(sel / sel.sum(1, keepdim=True), w, atol=1e-12)
        # permuting experts permutes ids (no ties in the rows checked)
        perm = torch.randperm(E, generator=g)
        ids_p, _ = mf.topk_softmax(z[:, perm], k)
        for t in (0, 1, 2, 7):
            assert perm[ids_p[t]].tolist() == ids[t].tolist()


def test_ffn_special_cases():
    g = torch.Generator().manual_seed(3)
    d, dff = 8, 12
    G_, U_, D_ = (torch.randn(s, dtype=F64, generator=g) for s in ((dff, d), (dff, d), (d, dff)))
    assert torch.equal(mf.expert_ffn(torch.zeros((1, d), dtype=F64), G_, U_, D_), torch.zeros((1, d), dtype=F64))
    x = torch.randn((3, d), dtype=F64, generator=g)
    assert torch.equal(mf.expert_ffn(x, torch.zeros_like(G_), U_, D_), torch.zeros((3, d), dtype=F64))
    # element-by-element loops (the definition written out) vs the matmul form
    y = mf.expert_ffn(x, G_, U_, D_)
    for t in range(3):
        a = []
        for r in range(dff):
            gv = sum(G_[r, j].item() * x[t, j].item() for j in range(d))
            uv = sum(U_[r, j].item() * x[t, j].item() for j in range(d))
            a.append(gv / (1.0 + math.exp(-gv)) * uv)
        for c in range(d):
            assert y[t, c].item() == pytest.approx(sum(D_[c, r].item() * a[r] for r in range(dff)), rel=1e-12)


def test_k_equals_E_equal_logits_is_plain_average():
    g = torch.Generator().manual_seed(5)
    d, dff, E = 4, 6, 3
    experts = torch.randn((E, 3 * d * dff), dtype=F64, generator=g)
    x = torch.randn((2, d), dtype=F64, generator=g)
    out, ids, w, _ = mf.moe_layer(x, experts, torch.zeros((E, d), dtype=F64), None, k=E, d_ff=dff)
    assert ids.tolist() == [[0, 1, 2]] * 2
    avg = sum(mf.expert_ffn(x, *mf.split_expert_blob(experts[e], d, dff)) for e in range(E)) / E
    assert torch.allclose(out, avg, atol=1e-14)


@pytest.mark.parametrize("shape", [si.TINY])
def test_layer_vs_dense_textbook_formulation(shape):
    """Library cross-check (P2): the sparse rank-ordered combine equals the dense 'gate matrix times all
    experts' formulation computed with batched fp64 matmuls (a different, textbook code path)."""
    experts = si.gen_layer_experts(shape, 0)
    w_r, bias = si.gen_router(shape, 0)
    x = si.gen_decode_hidden(shape, 6)[:, 0, :]
    d, dff, E, k = shape.d_model, shape.d_ff, shape.n_experts, shape.top_k
    out, ids, w, z = mf.moe_layer(x, experts, w_r, bias, k, dff)
    n = d * dff
    Gm = experts[:, :n].view(E, dff, d).to(F64)
    Um = experts[:, n:2 * n].view(E, dff, d).to(F64)
    Dm = experts[:, 2 * n:].view(E, d, dff).to(F64)
    xg = torch.einsum("efd,td->tef", Gm, x.to(F64))
    xu = torch.einsum("efd,td->tef", Um, x.to(F64))
    y_all = torch.einsum("edf,tef->ted", Dm, torch.nn.functional.silu(xg) * xu)
    gate = torch.zeros((x.shape[0], E), dtype=F64)
    p = torch.softmax(z, 1)
    topv = torch.topk(z, k, dim=1).indices
    gate.scatter_(1, topv, torch.gather(p, 1, topv))
    gate = gate / gate.sum(1, keepdim=True)
    dense = torch.einsum("te,ted->td", gate, y_all)
    assert torch.allclose(out, dense, rtol=1e-10, atol=1e-14)
    assert sorted(topv[0].tolist()) == sorted(ids[0].tolist())


def test_stack_residual_chain_and_paging_independence():
    """O3 + P8: the oracle has no notion of budget; the chain feeds layer l+1 from x_l + y_l."""
    shape = si.TINY
    experts, routers = si.gen_model(shape)
    h = si.gen_decode_hidden(shape, 2)[:, 0, :]
    xL, per = mf.stack_forward(h, experts, routers, shape.top_k, shape.d_ff, shape.torch_dtype)
    assert len(per) == shape.n_layers
    x1 = (per[0]["x"].float() + per[0]["out"].to(shape.torch_dtype).float()).to(shape.torch_dtype)
    assert torch.equal(per[1]["x"], x1)
    assert torch.equal(per[0]["x"], h.to(shape.torch_dtype))


def test_p1b_router_logits_hand_case_nonzero_rows_and_bias():
    """Pins the W_r.x term of O1 (orientation, bias add) on hand arithmetic (tests/golden/hand_router_ffn.txt P1b)."""
    x = torch.tensor([[1.0, 2.0]], dtype=F64)
    w_r = torch.tensor([[1.0, -0.5], [0.5, 1.0], [-1.0, 1.0], [2.0, -1.5]], dtype=F64)
    bias = torch.tensor([1.0, 0.5, 1.0, 1.0])
    z = mf.router_logits(x, w_r, bias)
    assert z[0].tolist() == [G["p1b_z0"], G["p1b_z1"], G["p1b_z2"], G["p1b_z3"]]
    ids, w = mf.topk_softmax(z, 2)
    assert ids.tolist() == [[G["p1_id0"], G["p1_id1"]]]
    assert w[0].tolist() == pytest.approx([G["p1_w0"], G["p1_w1"]], abs=1e-9)
    # square W_r: a transposed product passes the shape check but not the numbers
    z2 = mf.router_logits(x, torch.tensor([[1.0, 2.0], [3.0, 4.0]], dtype=F64), torch.tensor([0.5, -0.5]))
    assert z2[0].tolist() == [G["p1b_sq_z0"], G["p1b_sq_z1"]]
    # two tokens: rows of x map to rows of z
    z3 = mf.router_logits(torch.tensor([[1.0, 2.0], [2.0, 4.0]], dtype=F64), w_r, bias)
    assert z3[1].tolist() == [1.0, 5.5, 3.0, -1.0]            # 2 * (W_r x) + bias, by hand


def test_p1c_bf16_inputs_are_widened_exactly_before_the_product():
    """O1: 'fp64 from the stored values'.  With the product rounded to bf16 the winner flips (golden P1c)."""
    x = torch.tensor([[1.0 + 2.0 ** -7]], dtype=torch.bfloat16)
    w_r = torch.tensor([[1.0 + 2.0 ** -7], [1.0]], dtype=torch.bfloat16)
    bias = torch.tensor([0.0, 0.00785], dtype=torch.float32)
    assert x.double().item() == 1.0078125 and w_r.double()[0, 0].item() == 1.0078125   # both are bf16 values
    z = mf.router_logits(x, w_r, bias)
    assert z[0, 0].item() == G["p1c_z0"]                        # exact: (1 + 2^-7)^2
    ids, _ = mf.topk_softmax(z, 1)
    assert ids.tolist() == [[G["p1c_top1"]]]
    # the mistake this pins: rounding the product to bf16 first gives 1.015625 < z1
    wrong = (x * w_r[0]).double().item()
    assert wrong == 1.015625 and wrong + 0.0 < z[0, 1].item() < z[0, 0].item()
