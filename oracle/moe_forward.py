"""Oracle O1-O3: all-experts-resident routed MoE forward, fp64, plain PyTorch CPU ops.

TEST INFRASTRUCTURE (see oracle/__init__.py).  The method is exact -- paging changes where weights
live, not what is computed -- so the oracle for the numerical result is the
plain definition with every expert resident.  The paper never defines the router or the FFN (they
are the engine's); BASELINE.json's configs do: top-k routing with renormalised
softmax over the top-k, SwiGLU experts (readings G7, G8).

Canonical expert blob (one expert, model dtype), row-major out x in:
    [ gate (d_ff x d) | up (d_ff x d) | down (d x d_ff) ]

FP8 block-quantised experts ("The FP8 block-quantized path pages four tensors per expert (the
weights and their block scales)"; reading G29): the blob is bytes,
    [ W13 codes (2 d_ff x d) | W2 codes (d x d_ff) | S13 fp32 (2 d_ff/128 x d/128) | S2 fp32 (d/128 x d_ff/128) ]
with W13 = [gate; up], codes in OCP e4m3 ("e4m3fn": 1 sign, 4 exponent bits of bias 7, 3 mantissa bits, no infinities, 0x7f / 0xff
NaN), and the weight a code stands for is  W[r, c] = e4m3(code[r, c]) * S[r // 128, c // 128].  The method does not change
the arithmetic ("without changing kernels, model weights, or quantization"), so the oracle is the same plain
definition on the dequantised weights (weight-only quantisation: hidden states stay in the model's bf16).
"""
from __future__ import annotations

import torch

F64 = torch.float64


def router_logits(x: torch.Tensor, w_r: torch.Tensor, bias: torch.Tensor | None) -> torch.Tensor:
    """O1: z[t, e] = bias[e] + sum_j W_r[e, j] * x[t, j], in fp64 from the stored values.

    x [T, d], w_r [E, d] (model dtype; widened exactly), bias [E] fp32 or None -> z [T, E] fp64."""
    z = x.to(F64) @ w_r.to(F64).T
    if bias is not None:
        z = z + bias.to(F64)[None, :]
    return z


def topk_softmax(z: torch.Tensor, k: int) -> tuple[torch.Tensor, torch.Tensor]:
    """O1: ids = the k indices with largest z ordered by (z descending, id ascending);
    w_i = exp(z_ids[i] - z_ids[0]) / sum_{j<k} exp(z_ids[j] - z_ids[0])
    (softmax over the k selected logits == full softmax renormalised over the top-k).

    Full sort of all E logits (stable, so equal logits keep ascending id).  z [T, E] fp64."""
    order = torch.sort(z, dim=-1, descending=True, stable=True).indices
    ids = order[:, :k].contiguous()
    zs = torch.gather(z, 1, ids)
    ex = torch.exp(zs - zs[:, :1])
    w = ex / ex.sum(dim=1, keepdim=True)
    return ids, w


def split_expert_blob(blob: torch.Tensor, d: int, d_ff: int):
    """Views (G [d_ff, d], U [d_ff, d], D [d, d_ff]) of one canonical expert blob."""
    n = d * d_ff
    return blob[:n].view(d_ff, d), blob[n:2 * n].view(d_ff, d), blob[2 * n:3 * n].view(d, d_ff)


FP8_BLOCK = 128


def e4m3_value(code: int) -> float:
    """The real number an OCP e4m3 byte stands for: (-1)^s * 2^(e-7) * (1 + m/8) for e > 0, (-1)^s * 2^-6 * (m/8) for e = 0;
    s = bit 7, e = bits 6..3, m = bits 2..0; e = 15, m = 7 is NaN (the format has no infinities; largest finite 448)."""
    s, e, m = (code >> 7) & 1, (code >> 3) & 0xF, code & 7
    if e == 15 and m == 7:
        return float("nan")
    mag = (m / 8.0) * 2.0 ** -6 if e == 0 else (1.0 + m / 8.0) * 2.0 ** (e - 7)
    return -mag if s else mag


_E4M3_TABLE = torch.tensor([e4m3_value(c) for c in range(256)], dtype=F64)


def split_expert_blob_fp8(blob: torch.Tensor, d: int, d_ff: int):
    """Dequantised (G [d_ff, d], U [d_ff, d], D [d, d_ff]) in fp64 of one fp8 expert blob (uint8, layout in the module header)."""
    n13, n2, B = 2 * d_ff * d, d * d_ff, FP8_BLOCK
    blob = blob.contiguous()
    q13 = _E4M3_TABLE[blob[:n13].long()].view(2 * d_ff, d)
    q2 = _E4M3_TABLE[blob[n13:n13 + n2].long()].view(d, d_ff)
    ns13 = (2 * d_ff // B) * (d // B)
    sc = blob[n13 + n2:].clone().view(torch.float32).to(F64)
    s13 = sc[:ns13].view(2 * d_ff // B, d // B)
    s2 = sc[ns13:].view(d // B, d_ff // B)
    w13 = q13 * s13.repeat_interleave(B, dim=0).repeat_interleave(B, dim=1)
    w2 = q2 * s2.repeat_interleave(B, dim=0).repeat_interleave(B, dim=1)
    return w13[:d_ff], w13[d_ff:], w2


def silu(v: torch.Tensor) -> torch.Tensor:
    """silu(v) = v / (1 + e^{-v})."""
    return v / (1.0 + torch.exp(-v))


def expert_ffn(x: torch.Tensor, g: torch.Tensor, u: torch.Tensor, dn: torch.Tensor) -> torch.Tensor:
    """O2: y_e(x) = D (silu(G x) * (U x)), fp64, no intermediate rounding.  x [n, d] -> [n, d]."""
    x = x.to(F64)
    a = silu(x @ g.to(F64).T) * (x @ u.to(F64).T)
    return a @ dn.to(F64).T


def moe_layer(x: torch.Tensor, experts: torch.Tensor, w_r: torch.Tensor, bias: torch.Tensor | None,
              k: int, d_ff: int, ids: torch.Tensor | None = None, w: torch.Tensor | None = None):
    """O1 + O2 for one layer: out[t] = sum_{i<k} w[t,i] * y_{ids[t,i]}(x[t]), summed in rank order, fp64.

    experts [E, 3*d*d_ff] canonical blobs (uint8 [E, M_e]: fp8 block-quantised blobs, dequantised first).  If `ids`/`w` are given the routing is forced (used when a
    near-tie makes two id sets equally correct, G7/G22).  No shared expert, no FFN bias, no
    normalisation, no capacity factor.  Returns (out [T, d] fp64, ids [T, k] int64, w [T, k] fp64, z)."""
    T, d = x.shape
    z = router_logits(x, w_r, bias)
    if ids is None:
        ids, w = topk_softmax(z, k)
    elif w is None:
        zs = torch.gather(z, 1, ids)
        ex = torch.exp(zs - zs.max(dim=1, keepdim=True).values)
        w = ex / ex.sum(dim=1, keepdim=True)
    out = torch.zeros((T, d), dtype=F64)
    for i in range(k):                       # rank order
        for e in torch.unique(ids[:, i]).tolist():
            rows = (ids[:, i] == e).nonzero().flatten()
            g, u, dn = (split_expert_blob_fp8 if experts.dtype == torch.uint8 else split_expert_blob)(experts[e], d, d_ff)
            out[rows] += w[rows, i:i + 1] * expert_ffn(x[rows], g, u, dn)
    return out, ids, w, z


def stack_forward(h: torch.Tensor, experts: list, routers: list, k: int, d_ff: int, model_dtype):
    """O3 (harness-level semantics): x_0 = h; y_l = MoE_l(x_l); x_{l+1} = x_l + y_l.

    The residual add is done in fp32 on the model-dtype values and stored in the model dtype, and the
    layer output y_l is stored in the model dtype, exactly as the GPU harness stores them; the MoE
    itself is fp64.  Returns (x_L, [per-layer dict(x, out, ids, w)])."""
    x = h.to(model_dtype)
    per_layer = []
    for (blob, (w_r, bias)) in zip(experts, routers):
        out, ids, w, z = moe_layer(x, blob, w_r, bias, k, d_ff)
        y = out.to(model_dtype)
        per_layer.append(dict(x=x, out=out, ids=ids, w=w, z=z))
        x = (x.to(torch.float32) + y.to(torch.float32)).to(model_dtype)
    return x, per_layer
