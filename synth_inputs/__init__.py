"""Seeded synthetic inputs for the WiSP hot path (BASELINE.json configs).

This module is shared by the oracle (`oracle/`), the tests and `bench.py`.  It holds NONE of the
method's arithmetic (no router, no FFN, no paging policy): only the shapes of the five
BASELINE.json configs and a counter-based random generator that fills weight / router / hidden
buffers.  Both the CPU oracle and the CUDA library *read the buffers produced here*; neither side
re-derives them, so the generator may run on either the CPU or the GPU (the bits of a given run
are whatever this module wrote into the host buffers of that run).

Recipe:
  * expert and router weights ~ N(0, 0.02^2), rounded to the model dtype (bf16: RNE of the fp32 draw);
  * router bias[perm[r-1]] = -0.5 * alpha * ln(r), r = 1..E, one seeded permutation per layer
    (alpha = 1.1; 0.8 for the Mixtral-shaped config)  -> Zipf-skewed popularity;
  * decode hidden states: AR(1) h_t = 0.9 h_{t-1} + 0.1 xi_t, xi ~ N(0,1), stationary start
    h_{-1} ~ N(0, 0.01/0.19), kept in fp32 and cast when fed; batch streams are independent;
  * prefill hidden states: i.i.d. N(0,1);
  * dtype "fp8" ("the FP8 block-quantized path pages four tensors per expert (the weights and
    their block scales)"): the same N(0, 0.02^2) draws stored the way an FP8 block-quantised checkpoint stores them -- per
    128 x 128 block of W13 = [gate; up] and of W2 = down, the block's draws are first multiplied by a seeded gain 2^u,
    u ~ U(-1, 1) (so block scales differ by up to 4x, as they do in real checkpoints), then scale = amax / 448 (fp32) and
    code = RNE_e4m3(w / scale) (torch's float8_e4m3fn cast).  That is data preparation: both sides read the resulting bytes; hidden states and the router stay bf16.
Base seed 21868; tensor-kind ids: 1 experts, 2 router W, 3 permutation, 4 hidden stream, 5 prompt
lengths, 6 prefill tokens, 7 fp8 block gains.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, replace

import torch

BASE_SEED = 21868
FP8_BLOCK = 128          # block-scale granularity of the fp8 expert weights (both dimensions)
KIND_EXPERTS, KIND_ROUTER, KIND_PERM, KIND_HIDDEN, KIND_PROMPT_LEN, KIND_PREFILL, KIND_FP8_GAIN = 1, 2, 3, 4, 5, 6, 7

_M1 = 0xBF58476D1CE4E5B9
_M2 = 0x94D049BB133111EB
_GOLD = 0x9E3779B97F4A7C15


def _s64(v: int) -> int:
    """Python int -> the signed 64-bit value with the same bits (torch int64 arithmetic wraps)."""
    v &= (1 << 64) - 1
    return v - (1 << 64) if v >= (1 << 63) else v


def _lsr(z: torch.Tensor, s: int) -> torch.Tensor:
    return (z >> s) & ((1 << (64 - s)) - 1)


def _mix64(z: torch.Tensor) -> torch.Tensor:
    """SplitMix64 finaliser on an int64 tensor (wrapping arithmetic)."""
    z = (z ^ _lsr(z, 30)) * _s64(_M1)
    z = (z ^ _lsr(z, 27)) * _s64(_M2)
    return z ^ _lsr(z, 31)


def _mix64_int(v: int) -> int:
    m = (1 << 64) - 1
    v &= m
    v = ((v ^ (v >> 30)) * _M1) & m
    v = ((v ^ (v >> 27)) * _M2) & m
    return v ^ (v >> 31)


def stream_key(seed: int, kind: int, *idx: int) -> int:
    """Fold (seed, tensor-kind, indices...) into one 64-bit stream key."""
    h = _mix64_int(seed * _GOLD + kind)
    for i in idx:
        h = _mix64_int(h ^ ((i + 1) * _GOLD))
    return h


def _hash_counter(key: int, n: int, device, offset: int = 0) -> torch.Tensor:
    ctr = torch.arange(offset, offset + n, dtype=torch.int64, device=device)
    return _mix64(ctr * _s64(_GOLD) + _s64(key))


def normal(key: int, n: int, device="cpu", offset: int = 0) -> torch.Tensor:
    """n standard normals (fp32) from the counter stream `key`, elements offset..offset+n-1.

    One Box-Muller draw per 64-bit hash: u1 from the high 32 bits, u2 from the low 32 bits."""
    h = _hash_counter(key, n, device, offset)
    hi = _lsr(h, 32).to(torch.float32)
    lo = (h & 0xFFFFFFFF).to(torch.float32)
    u1 = (hi + 0.5) * (1.0 / 4294967296.0)
    u2 = (lo + 0.5) * (1.0 / 4294967296.0)
    u1 = u1.clamp_(min=1e-10, max=1.0 - 2.0 ** -24)
    r = torch.sqrt(-2.0 * torch.log(u1))
    return r * torch.cos((2.0 * math.pi) * u2)


def uniform_int(key: int, n: int, lo: int, hi: int) -> list[int]:
    """n integers uniform over lo..hi inclusive (host side, pure Python)."""
    span = hi - lo + 1
    return [lo + _mix64_int(key + (i + 1) * _GOLD) % span for i in range(n)]


def permutation(key: int, n: int) -> list[int]:
    """Seeded permutation of range(n): argsort of per-index hashes (ties impossible in practice)."""
    return sorted(range(n), key=lambda i: (_mix64_int(key + (i + 1) * _GOLD), i))


@dataclass(frozen=True)
class MoEShape:
    """Layer shapes (uniform across layers) plus the config's workload constants."""
    name: str
    n_layers: int
    n_experts: int
    top_k: int
    d_model: int
    d_ff: int
    dtype: str            # "f32" | "bf16" | "fp8" (e4m3 expert weights with 128 x 128 fp32 block scales; hidden states / router bf16)
    zipf_alpha: float
    seed: int = BASE_SEED

    @property
    def torch_dtype(self):
        return torch.float32 if self.dtype == "f32" else torch.bfloat16

    @property
    def elem_bytes(self) -> int:            # bytes per hidden-state / router element
        return 4 if self.dtype == "f32" else 2

    @property
    def expert_elems(self) -> int:
        return 3 * self.d_model * self.d_ff

    @property
    def scale_elems(self) -> int:           # fp8: fp32 block scales of W13 and W2 (one per 128 x 128 block)
        return self.expert_elems // (FP8_BLOCK * FP8_BLOCK) if self.dtype == "fp8" else 0

    @property
    def expert_bytes(self) -> int:          # M_e
        if self.dtype == "fp8":
            return self.expert_elems + 4 * self.scale_elems
        return self.expert_elems * self.elem_bytes

    @property
    def blob_dtype(self):                   # element type of the tensor that holds the canonical expert blobs
        return torch.uint8 if self.dtype == "fp8" else self.torch_dtype

    @property
    def blob_len(self) -> int:              # elements of blob_dtype per expert
        return self.expert_bytes if self.dtype == "fp8" else self.expert_elems

    @property
    def slot_unit_bytes(self) -> int:       # a = L * M_e
        return self.n_layers * self.expert_bytes

    def with_layers(self, n_layers: int) -> "MoEShape":
        return replace(self, n_layers=n_layers)


# BASELINE.json configs[0..3] (config 5 reuses QWEN3).
TINY = MoEShape("tiny", 2, 16, 2, 256, 512, "f32", 1.1)
QWEN3 = MoEShape("qwen3-30b-a3b-shaped", 48, 128, 8, 2048, 768, "bf16", 1.1)
MIXTRAL = MoEShape("mixtral-8x7b-shaped", 32, 8, 2, 4096, 14336, "bf16", 0.8)
QWEN3_FP8 = replace(QWEN3, name="qwen3-30b-a3b-shaped-fp8", dtype="fp8")       # f4: the quantised variant of the headline shape
SHAPES = {s.name: s for s in (TINY, QWEN3, MIXTRAL, QWEN3_FP8)}


def slots_for_budget(shape: MoEShape, expert_bytes: int) -> int:
    """C = floor(B_exp / a) clipped to [0, E]."""
    return max(0, min(shape.n_experts, expert_bytes // shape.slot_unit_bytes))


def normal_multi(keys: list[int], n: int, device="cpu") -> torch.Tensor:
    """[len(keys), n] standard normals: row r is exactly normal(keys[r], n) (same counter streams)."""
    ctr = torch.arange(0, n, dtype=torch.int64, device=device) * _s64(_GOLD)
    kt = torch.tensor([_s64(k) for k in keys], dtype=torch.int64, device=device)
    h = _mix64(ctr[None, :] + kt[:, None])
    hi = _lsr(h, 32).to(torch.float32)
    lo = (h & 0xFFFFFFFF).to(torch.float32)
    del h
    u1 = ((hi + 0.5) * (1.0 / 4294967296.0)).clamp_(min=1e-10, max=1.0 - 2.0 ** -24)
    u2 = (lo + 0.5) * (1.0 / 4294967296.0)
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2)


def _block_quantise_fp8(w: torch.Tensor, rows: int, cols: int, keys: list[int]):
    """[n, rows, cols] fp32 -> (codes uint8 [n, rows, cols], scales fp32 [n, rows/128, cols/128]); data preparation only.
    keys[i]: counter stream of item i's block gains."""
    n, B = w.shape[0], FP8_BLOCK
    nb = (rows // B) * (cols // B)
    u = torch.stack([(_lsr(_hash_counter(k, nb, w.device), 40).to(torch.float32) + 0.5) * (2.0 ** -24) for k in keys])   # U(0,1)
    gain = torch.exp2(2.0 * u - 1.0).view(n, rows // B, 1, cols // B, 1)
    blk = w.view(n, rows // B, B, cols // B, B) * gain
    scale = blk.abs().amax(dim=(2, 4)) / 448.0
    scale = torch.where(scale > 0, scale, torch.ones_like(scale))
    q = (blk / scale[:, :, None, :, None]).to(torch.float8_e4m3fn)
    return q.view(torch.uint8).reshape(n, rows, cols), scale


def gen_layer_experts(shape: MoEShape, layer: int, device="cpu", out: torch.Tensor | None = None,
                      chunk_experts: int | None = None) -> torch.Tensor:
    """Expert blobs of one layer, canonical layout [E, gate(d_ff x d) | up(d_ff x d) | down(d x d_ff)],
    row-major out x in, in the model dtype.  `out` may be a preallocated (pinned) host tensor.

    dtype "fp8": uint8 blobs [E, expert_bytes] = [ W13 codes (2 d_ff x d) | W2 codes (d x d_ff) | S13 fp32 (2 d_ff/128 x d/128) |
    S2 fp32 (d/128 x d_ff/128) ], the four tensors of PAPER.md:369."""
    E, n = shape.n_experts, shape.expert_elems
    if shape.dtype == "fp8":
        d, f = shape.d_model, shape.d_ff
        if out is None:
            out = torch.empty((E, shape.expert_bytes), dtype=torch.uint8)
        if chunk_experts is None:
            chunk_experts = max(1, min(E, (1 << 26) // n)) if str(device) != "cpu" else 1
        for e0 in range(0, E, chunk_experts):
            e1 = min(E, e0 + chunk_experts)
            keys = [stream_key(shape.seed, KIND_EXPERTS, layer, e) for e in range(e0, e1)]
            v = normal_multi(keys, n, device).mul_(0.02)
            q13, s13 = _block_quantise_fp8(v[:, :2 * d * f].reshape(e1 - e0, 2 * f, d), 2 * f, d,
                                           [stream_key(shape.seed, KIND_FP8_GAIN, layer, e, 0) for e in range(e0, e1)])
            q2, s2 = _block_quantise_fp8(v[:, 2 * d * f:].reshape(e1 - e0, d, f), d, f,
                                         [stream_key(shape.seed, KIND_FP8_GAIN, layer, e, 1) for e in range(e0, e1)])
            sc = torch.cat([s13.reshape(e1 - e0, -1), s2.reshape(e1 - e0, -1)], dim=1).contiguous()
            blob = torch.cat([q13.reshape(e1 - e0, -1), q2.reshape(e1 - e0, -1), sc.view(torch.uint8).reshape(e1 - e0, -1)], dim=1)
            out[e0:e1].copy_(blob)
        return out
    if out is None:
        out = torch.empty((E, n), dtype=shape.torch_dtype)
    if chunk_experts is None:
        chunk_experts = max(1, min(E, (1 << 27) // n)) if str(device) != "cpu" else 1
    for e0 in range(0, E, chunk_experts):
        e1 = min(E, e0 + chunk_experts)
        keys = [stream_key(shape.seed, KIND_EXPERTS, layer, e) for e in range(e0, e1)]
        v = normal_multi(keys, n, device).mul_(0.02).to(shape.torch_dtype)
        out[e0:e1].copy_(v)
    return out


def gen_router(shape: MoEShape, layer: int) -> tuple[torch.Tensor, torch.Tensor]:
    """(W_r [E, d] in the model dtype, bias [E] fp32) for one layer (host tensors)."""
    E, d = shape.n_experts, shape.d_model
    w = normal(stream_key(shape.seed, KIND_ROUTER, layer), E * d).mul_(0.02).to(shape.torch_dtype).view(E, d)
    perm = permutation(stream_key(shape.seed, KIND_PERM, layer), E)
    bias = torch.empty(E, dtype=torch.float32)
    for r in range(1, E + 1):
        bias[perm[r - 1]] = -0.5 * shape.zipf_alpha * math.log(r)
    return w, bias


def gen_decode_hidden(shape: MoEShape, n_steps: int, batch: int = 1, stream_base: int = 0,
                      rho: float = 0.9, noise: float = 0.1) -> torch.Tensor:
    """AR(1) decode hidden states [n_steps, batch, d] in fp32 (cast by the caller when fed).

    h_t = rho*h_{t-1} + noise*xi_t with a stationary start; stream b uses key (.., stream_base+b)."""
    d = shape.d_model
    out = torch.empty((n_steps, batch, d), dtype=torch.float32)
    var0 = noise * noise / (1.0 - rho * rho)
    for b in range(batch):
        key = stream_key(shape.seed, KIND_HIDDEN, stream_base + b)
        xi = normal(key, (n_steps + 1) * d).view(n_steps + 1, d)
        h = xi[0] * math.sqrt(var0)
        for t in range(n_steps):
            h = rho * h + noise * xi[t + 1]
            out[t, b] = h
    return out


def gen_prefill_hidden(shape: MoEShape, n_tokens: int, request: int = 0) -> torch.Tensor:
    """Prefill hidden states [n_tokens, d] i.i.d. N(0,1), fp32."""
    key = stream_key(shape.seed, KIND_PREFILL, request)
    return normal(key, n_tokens * shape.d_model).view(n_tokens, shape.d_model)


def gen_prompt_lengths(shape: MoEShape, n_requests: int, lo: int = 1024, hi: int = 16384) -> list[int]:
    return uniform_int(stream_key(shape.seed, KIND_PROMPT_LEN), n_requests, lo, hi)


def gen_model(shape: MoEShape, device="cpu", pin: bool = False):
    """All layers: list of expert blobs [E, 3*d*d_ff], list of (W_r, bias).  Host tensors."""
    experts, routers = [], []
    for l in range(shape.n_layers):
        buf = torch.empty((shape.n_experts, shape.blob_len), dtype=shape.blob_dtype, pin_memory=pin)
        experts.append(gen_layer_experts(shape, l, device, out=buf))
        routers.append(gen_router(shape, l))
    return experts, routers
