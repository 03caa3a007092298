"""CPU-side check (-m 'not gpu'): libwisp.so builds/loads and exports every symbol include/wisp.h declares;
without a CUDA device the product path fails loudly (no CPU fallback)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    txt = open(os.path.join(ROOT, "include", "wisp.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(wisp_[a-z_0-9]+)\s*\(", txt)))


def test_header_symbols_exported():
    from paper_2606_21868_b200 import build, lib, lib_path
    build.build()
    L = ctypes.CDLL(lib_path())
    syms = declared_symbols()
    assert {"wisp_create", "wisp_register_host_experts", "wisp_moe_forward", "wisp_set_split", "wisp_stats"} <= set(syms)
    for s in syms:
        assert hasattr(L, s), f"{s} declared in wisp.h but not exported"
    assert b"sm_100a" in lib().wisp_version()


def test_binding_covers_every_entry_point():
    from paper_2606_21868_b200 import binding
    assert sorted(binding._SIGS) == declared_symbols()


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import paper_2606_21868_b200 as wp
    with pytest.raises(wp.WispError) as ei:
        wp.Wisp(1 << 26, n_layers=2, n_experts=16, top_k=2, d_model=256, d_ff=512, max_tokens=1, dtype=0)
    assert ei.value.status == -3


def test_struct_sizes_match_header():
    from paper_2606_21868_b200 import binding as b
    assert ctypes.sizeof(b.WispConfig) == 72 and ctypes.sizeof(b.WispTraceEvent) == 32
    assert ctypes.sizeof(b.WispLayerStats) == 48 and ctypes.sizeof(b.WispStats) == 48 + 8 + 13 * 8
    assert ctypes.sizeof(b.WispMvwsaIn) == 64
