"""Pins of the fp8 block-quantised expert path of the oracle (G29)."""
import math
import os

import torch

from oracle import moe_forward as mf

GOLD = os.path.join(os.path.dirname(__file__), "golden", "hand_fp8.txt")


def _sections():
    sec, cur = {}, None
    for raw in open(GOLD):
        line = raw.split("#")[0].strip()
        if not line:
            continue
        if line.startswith("["):
            cur = line.strip("[]")
            sec[cur] = []
        else:
            sec[cur].append(line.split())
    return sec


def test_e4m3_hand_codes():
    sec = _sections()
    for code, val in sec["codes"]:
        got = mf.e4m3_value(int(code, 16))
        assert got == float(val) and math.copysign(1.0, got) == math.copysign(1.0, float(val)), (code, got)
    for (code,) in sec["nan"]:
        assert math.isnan(mf.e4m3_value(int(code, 16)))


def test_e4m3_table_matches_library_cast():
    """Independent of the formula: torch's float8_e4m3fn widening of every finite code."""
    codes = torch.arange(256, dtype=torch.uint8)
    lib = codes.view(torch.float8_e4m3fn).to(torch.float64)
    finite = ~torch.isnan(lib)
    assert int(finite.sum()) == 254
    assert torch.equal(mf._E4M3_TABLE[finite], lib[finite])
    assert torch.isnan(mf._E4M3_TABLE[~finite]).all()


def _hand_blob():
    sec = _sections()
    d = dff = 256
    s13 = torch.tensor([[float(v) for v in row] for row in sec["s13"]], dtype=torch.float32)
    s2 = torch.tensor([[float(v) for v in row] for row in sec["s2"]], dtype=torch.float32)
    codes = torch.full((3 * d * dff,), 0x38, dtype=torch.uint8)
    blob = torch.cat([codes, s13.reshape(-1).view(torch.uint8), s2.reshape(-1).view(torch.uint8)])
    return sec, blob, d, dff


def test_block_scale_indexing_hand_case():
    sec, blob, d, dff = _hand_blob()
    G, U, D = mf.split_expert_blob_fp8(blob, d, dff)
    mats = {"G": G, "U": U, "D": D}
    for name, r, c, v in sec["dequant"]:
        assert float(mats[name][int(r), int(c)]) == float(v), (name, r, c)


def test_fp8_ffn_unit_vector_closed_form():
    _, blob, d, dff = _hand_blob()
    G, U, D = mf.split_expert_blob_fp8(blob, d, dff)
    x = torch.zeros((1, d), dtype=torch.float64)
    x[0, 0] = 1.0
    y = mf.expert_ffn(x, G, U, D)[0]
    silu = lambda v: v / (1.0 + math.exp(-v))
    y0 = 128 * (23 * silu(2.0) * 11 + 29 * silu(5.0) * 17)
    y128 = 128 * (31 * silu(2.0) * 11 + 37 * silu(5.0) * 17)
    assert abs(float(y[0]) - y0) <= 1e-12 * y0 and abs(float(y[127]) - y0) <= 1e-12 * y0
    assert abs(float(y[128]) - y128) <= 1e-12 * y128 and abs(float(y[255]) - y128) <= 1e-12 * y128


def test_codes_and_signs_enter_the_product():
    """One non-trivial code per matrix: the dequantised entry is value(code) * its block scale, sign included."""
    _, blob, d, dff = _hand_blob()
    blob = blob.clone()
    blob[0 * d + 130] = 0xC4                      # G[0, 130] = -3 * S13[0][1]
    blob[d * dff + 129 * d + 1] = 0x01            # U[129, 1] = 2^-9 * S13[3][0]
    blob[2 * d * dff + 200 * dff + 5] = 0x7E      # D[200, 5] = 448 * S2[1][0]
    G, U, D = mf.split_expert_blob_fp8(blob, d, dff)
    assert float(G[0, 130]) == -9.0 and float(U[129, 1]) == 17.0 * 2.0 ** -9 and float(D[200, 5]) == 448.0 * 31.0


def test_moe_layer_accepts_fp8_blobs():
    """Routing + combine around the dequantised experts: same result as the dense formula on the dequantised matrices."""
    import synth_inputs as si
    from dataclasses import replace
    sh = replace(si.QWEN3_FP8, n_layers=1, n_experts=4, top_k=2, d_model=256, d_ff=256)
    ex = si.gen_layer_experts(sh, 0)
    wr, bias = si.gen_router(sh, 0)
    x = si.gen_decode_hidden(sh, 1, 3)[0].to(torch.bfloat16)
    out, ids, w, _ = mf.moe_layer(x, ex, wr, bias, 2, sh.d_ff)
    for t in range(3):
        acc = torch.zeros(sh.d_model, dtype=torch.float64)
        for i in range(2):
            G, U, D = mf.split_expert_blob_fp8(ex[int(ids[t, i])], sh.d_model, sh.d_ff)
            xv = x[t].to(torch.float64)
            acc += w[t, i] * (D @ (mf.silu(G @ xv) * (U @ xv)))
        assert torch.allclose(acc, out[t], rtol=1e-12, atol=0)
    # the codes really are e4m3 and the scales really are amax / 448 of their block (recipe check, synth_inputs)
    q = ex[0, :sh.expert_elems].view(torch.float8_e4m3fn).float()
    assert float(q.abs().max()) == 448.0
