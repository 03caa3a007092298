"""ctypes binding of libwisp.so: the same entry points as include/wisp.h, plus `Wisp`, a small holder
class that turns torch tensors into pointers.  PyTorch is used for device memory and streams only."""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

WISP_F32, WISP_BF16, WISP_FP8_E4M3 = 0, 1, 2
WISP_LRU, WISP_LFU = 0, 1
WISP_FETCH_MEMCPY, WISP_FETCH_ZEROCOPY, WISP_FETCH_FUSED, WISP_FETCH_STATIC = 0, 1, 2, 3
WISP_WAVES_ASCENDING, WISP_WAVES_HITS_FIRST = 0, 1
KERNEL_CLASSES = ("router", "topk", "residency", "fetch", "ffn", "ffn_miss", "combine", "prefill_gate_up",
                  "prefill_down", "other")
N_KERNEL_CLASSES = len(KERNEL_CLASSES)
STATUS_NAMES = {0: "WISP_OK", -1: "WISP_EINVAL", -2: "WISP_ENOMEM", -3: "WISP_ECUDA", -4: "WISP_ESTATE", -5: "WISP_EBUDGET"}


class WispConfig(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("n_experts", C.c_int32), ("top_k", C.c_int32), ("d_model", C.c_int32),
                ("d_ff", C.c_int32), ("max_tokens", C.c_int32), ("dtype", C.c_int32), ("policy", C.c_int32),
                ("fetch", C.c_int32), ("ring_stages", C.c_int32), ("unit_rows", C.c_int32), ("reserved0", C.c_int32), ("kv_block_bytes", C.c_uint64),
                ("kv_floor_blocks", C.c_uint64), ("trace_capacity", C.c_uint64)]


class WispLayerStats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in ("steps", "references", "hits", "misses", "evictions", "bytes_fetched")]


class WispStats(C.Structure):
    _fields_ = [("total", WispLayerStats), ("n_layers", C.c_int32), ("slots_per_layer", C.c_int32)] + [
        (n, C.c_uint64) for n in ("budget_bytes", "expert_bytes", "kv_bytes", "kv_blocks", "kv_blocks_reserved",
                                  "kv_blocks_peak", "resize_count", "failed_resize_count", "trace_dropped", "fetch_ns",
                                  "kernel_launches", "prefetches", "prefetch_bytes")]


class WispTraceEvent(C.Structure):
    _fields_ = [("step", C.c_uint64), ("layer", C.c_uint32), ("wave", C.c_uint32), ("expert", C.c_int32),
                ("slot", C.c_int32), ("evicted", C.c_int32), ("kind", C.c_uint32)]


class WispMvwsaIn(C.Structure):
    _fields_ = [("mode", C.c_int32), ("c_min", C.c_int32), ("c_max", C.c_int32), ("dead_zone", C.c_int32),
                ("headroom", C.c_double), ("kv_peak_blocks", C.c_uint64), ("c_exp", C.c_double), ("c_kv", C.c_double),
                ("m_kv", C.POINTER(C.c_double)), ("m_kv_len", C.c_uint64)]


class WispError(RuntimeError):
    def __init__(self, status: int, what: str, msg: str = ""):
        self.status = status
        super().__init__(f"{what}: {STATUS_NAMES.get(status, status)} {msg}")


def lib_path() -> str:
    return os.path.join(_HERE, "libwisp.so")


_SIGS = {
    "wisp_create": (C.c_int, [C.c_uint64, C.POINTER(WispConfig), C.POINTER(C.c_void_p)]),
    "wisp_destroy": (C.c_int, [C.c_void_p]),
    "wisp_register_host_experts": (C.c_int, [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]),
    "wisp_moe_forward": (C.c_int, [C.c_void_p, C.c_int32, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]),
    "wisp_set_split": (C.c_int, [C.c_void_p, C.c_uint64, C.c_uint64]),
    "wisp_stats": (C.c_int, [C.c_void_p, C.POINTER(WispStats)]),
    "wisp_stack_forward": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]),
    "wisp_residual_add": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]),
    "wisp_layer_stats_read": (C.c_int, [C.c_void_p, C.c_int32, C.POINTER(WispLayerStats)]),
    "wisp_trace_enable": (C.c_int, [C.c_void_p, C.c_int32]),
    "wisp_set_wave_order": (C.c_int, [C.c_void_p, C.c_int32]),
    "wisp_set_policy": (C.c_int, [C.c_void_p, C.c_int32]),
    "wisp_set_prefetch": (C.c_int, [C.c_void_p, C.c_int32, C.c_double, C.c_int32]),
    "wisp_trace_read": (C.c_int, [C.c_void_p, C.POINTER(WispTraceEvent), C.c_uint64, C.POINTER(C.c_uint64)]),
    "wisp_last_topk": (C.c_int, [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.POINTER(C.c_int32)]),
    "wisp_last_logits": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int32]),
    "wisp_route_noalloc": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_void_p,
                                     C.c_void_p, C.c_void_p, C.c_void_p]),
    "wisp_debug_step_routing": (C.c_int, [C.c_void_p, C.c_int32, C.POINTER(C.c_int32), C.c_int32]),
    "wisp_debug_reset_pool": (C.c_int, [C.c_void_p]),
    "wisp_debug_ffn_launch": (C.c_int, [C.c_void_p, C.c_int32, C.c_void_p, C.c_int32, C.c_void_p]),
    "wisp_debug_residency": (C.c_int, [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "wisp_debug_verify_pool": (C.c_int, [C.c_void_p, C.c_int32, C.POINTER(C.c_int32)]),
    "wisp_timing_enable": (C.c_int, [C.c_void_p, C.c_int32]),
    "wisp_timing_read": (C.c_int, [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_uint64), C.c_int32]),
    "wisp_kv_reserve": (C.c_int, [C.c_void_p, C.c_int64]),
    "wisp_mvwsa_propose": (C.c_int, [C.c_void_p, C.POINTER(WispMvwsaIn), C.POINTER(C.c_uint64), C.POINTER(C.c_uint64),
                                     C.POINTER(C.c_int32)]),
    "wisp_mvwsa_miss_curve": (C.c_int, [C.c_void_p, C.POINTER(C.c_double), C.c_int32, C.c_double]),
    "wisp_mvwsa_track": (C.c_int, [C.c_void_p, C.c_int32]),
    "wisp_last_error": (C.c_char_p, [C.c_void_p]),
    "wisp_version": (C.c_char_p, []),
}


def lib() -> C.CDLL:
    """Load libwisp.so (built in-tree by `python -m paper_2606_21868_b200.build`).  Fails loudly if absent."""
    global _LIB
    if _LIB is None:
        p = lib_path()
        if not os.path.exists(p):
            raise ImportError(f"{p} not found: build it with `python -m paper_2606_21868_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(p)
        for name, (res, args) in _SIGS.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _LIB = L
    return _LIB


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def route_noalloc(hidden, router_w, router_bias, top_k, dtype, logits, ids, w, stream):
    """wisp_route_noalloc: device tensors in and out (hidden [T, d], router_w [E, d], router_bias [E] or None, logits [T, E] or None,
    ids [T, k] int32, w [T, k] fp32); allocates nothing.  Raises WispError on a non-zero status."""
    rc = lib().wisp_route_noalloc(_ptr(hidden), _ptr(router_w), _ptr(router_bias), hidden.shape[0], router_w.shape[0], hidden.shape[1],
                                  top_k, dtype, _ptr(logits), _ptr(ids), _ptr(w), C.c_void_p(stream))
    if rc:
        raise WispError(rc, "wisp_route_noalloc")


class Wisp:
    """Holder of one wisp_ctx.  Methods mirror the C entry points one to one."""

    def __init__(self, budget_bytes: int, *, n_layers, n_experts, top_k, d_model, d_ff, max_tokens, dtype, policy=WISP_LRU,
                 fetch=WISP_FETCH_ZEROCOPY, kv_block_bytes=0, kv_floor_blocks=0, trace_capacity=0, ring_stages=0, unit_rows=0):
        self.L = lib()
        self.cfg = WispConfig(n_layers, n_experts, top_k, d_model, d_ff, max_tokens, dtype, policy, fetch, ring_stages, unit_rows, 0,
                              kv_block_bytes, kv_floor_blocks, trace_capacity)
        self.ctx = C.c_void_p()
        rc = self.L.wisp_create(budget_bytes, C.byref(self.cfg), C.byref(self.ctx))
        if rc:
            self.ctx = None
            raise WispError(rc, "wisp_create")

    def _ck(self, rc, what):
        if rc:
            raise WispError(rc, what, (self.L.wisp_last_error(self.ctx) or b"").decode())

    def close(self):
        if self.ctx:
            self.L.wisp_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def register_host_experts(self, layer, experts, router_w, router_bias=None):
        assert experts.is_contiguous() and router_w.is_contiguous() and not experts.is_cuda
        self._ck(self.L.wisp_register_host_experts(self.ctx, layer, _ptr(experts), _ptr(router_w), _ptr(router_bias)),
                 "wisp_register_host_experts")

    def moe_forward(self, layer, hidden, out, stream):
        n = hidden.shape[0] if hidden is not None else 0
        self._ck(self.L.wisp_moe_forward(self.ctx, layer, _ptr(hidden), n, _ptr(out), C.c_void_p(stream)), "wisp_moe_forward")

    def stack_forward(self, hidden, hidden_out, stream):
        self._ck(self.L.wisp_stack_forward(self.ctx, _ptr(hidden), hidden.shape[0], _ptr(hidden_out), C.c_void_p(stream)),
                 "wisp_stack_forward")

    def residual_add(self, x, y, out, stream):
        self._ck(self.L.wisp_residual_add(self.ctx, _ptr(x), _ptr(y), _ptr(out), x.numel(), C.c_void_p(stream)), "wisp_residual_add")

    def set_split(self, expert_bytes, kv_bytes):
        self._ck(self.L.wisp_set_split(self.ctx, expert_bytes, kv_bytes), "wisp_set_split")

    def stats(self) -> WispStats:
        s = WispStats()
        self._ck(self.L.wisp_stats(self.ctx, C.byref(s)), "wisp_stats")
        return s

    def layer_stats(self, layer) -> WispLayerStats:
        s = WispLayerStats()
        self._ck(self.L.wisp_layer_stats_read(self.ctx, layer, C.byref(s)), "wisp_layer_stats_read")
        return s

    def trace_enable(self, on=True):
        self._ck(self.L.wisp_trace_enable(self.ctx, int(on)), "wisp_trace_enable")

    def set_wave_order(self, order):
        self._ck(self.L.wisp_set_wave_order(self.ctx, int(order)), "wisp_set_wave_order")

    def set_prefetch(self, n_per_layer, gamma=0.5, window=1):
        self._ck(self.L.wisp_set_prefetch(self.ctx, int(n_per_layer), float(gamma), int(window)), "wisp_set_prefetch")

    def set_policy(self, policy):
        self._ck(self.L.wisp_set_policy(self.ctx, int(policy)), "wisp_set_policy")

    def trace_read(self, cap=1 << 20):
        buf = (WispTraceEvent * cap)()
        n = C.c_uint64()
        self._ck(self.L.wisp_trace_read(self.ctx, buf, cap, C.byref(n)), "wisp_trace_read")
        return [(e.layer, e.step, e.wave, e.expert, e.slot, e.evicted, e.kind) for e in buf[:n.value]]

    def last_topk(self, layer):
        import numpy as np
        k, mt = self.cfg.top_k, self.cfg.max_tokens
        ids = np.empty((mt, k), dtype=np.int32)
        w = np.empty((mt, k), dtype=np.float32)
        n = C.c_int32()
        self._ck(self.L.wisp_last_topk(self.ctx, layer, ids.ctypes.data_as(C.c_void_p), w.ctypes.data_as(C.c_void_p),
                                       C.byref(n)), "wisp_last_topk")
        return ids[:n.value].copy(), w[:n.value].copy()

    def last_logits(self, n_tokens):
        import numpy as np
        z = np.empty((n_tokens, self.cfg.n_experts), dtype=np.float32)
        self._ck(self.L.wisp_last_logits(self.ctx, z.ctypes.data_as(C.c_void_p), n_tokens), "wisp_last_logits")
        return z

    def debug_step_routing(self, layer, ids):
        arr = (C.c_int32 * len(ids))(*[int(i) for i in ids])
        self._ck(self.L.wisp_debug_step_routing(self.ctx, layer, arr, len(ids)), "wisp_debug_step_routing")

    def debug_reset_pool(self):
        self._ck(self.L.wisp_debug_reset_pool(self.ctx), "wisp_debug_reset_pool")

    def debug_ffn_launch(self, layer, hidden, stream):
        self._ck(self.L.wisp_debug_ffn_launch(self.ctx, layer, _ptr(hidden), hidden.shape[0], C.c_void_p(stream)), "wisp_debug_ffn_launch")

    def debug_residency(self, layer):
        import numpy as np
        Cn, E = self.stats().slots_per_layer, self.cfg.n_experts
        pi_inv = np.empty(Cn, dtype=np.int32)
        tau = np.empty(Cn, dtype=np.uint64)
        freq = np.empty(E, dtype=np.uint64)
        clock = C.c_uint64()
        self._ck(self.L.wisp_debug_residency(self.ctx, layer, pi_inv.ctypes.data_as(C.c_void_p), tau.ctypes.data_as(C.c_void_p),
                                             freq.ctypes.data_as(C.c_void_p), C.byref(clock)), "wisp_debug_residency")
        return pi_inv, tau, freq, clock.value

    def debug_verify_pool(self, layer) -> int:
        n = C.c_int32()
        self._ck(self.L.wisp_debug_verify_pool(self.ctx, layer, C.byref(n)), "wisp_debug_verify_pool")
        return n.value

    def timing_enable(self, level=2):
        self._ck(self.L.wisp_timing_enable(self.ctx, int(level)), "wisp_timing_enable")

    def timing_read(self, reset=True):
        ms = (C.c_double * N_KERNEL_CLASSES)()
        n = (C.c_uint64 * N_KERNEL_CLASSES)()
        self._ck(self.L.wisp_timing_read(self.ctx, ms, n, int(reset)), "wisp_timing_read")
        return {name: (ms[i], n[i]) for i, name in enumerate(KERNEL_CLASSES)}

    def kv_reserve(self, delta_blocks):
        self._ck(self.L.wisp_kv_reserve(self.ctx, delta_blocks), "wisp_kv_reserve")

    def mvwsa_track(self, on=True):
        self._ck(self.L.wisp_mvwsa_track(self.ctx, int(on)), "wisp_mvwsa_track")

    def mvwsa_miss_curve(self, n, decay=1.0):
        buf = (C.c_double * n)()
        self._ck(self.L.wisp_mvwsa_miss_curve(self.ctx, buf, n, decay), "wisp_mvwsa_miss_curve")
        return list(buf)

    def mvwsa_propose(self, *, mode=0, c_min=1, c_max=0, dead_zone=1, headroom=0.2, kv_peak_blocks=None, c_exp=0.0,
                      c_kv=0.0, m_kv=None):
        arr = None
        inp = WispMvwsaIn(mode, c_min, c_max, dead_zone, headroom, (1 << 64) - 1 if kv_peak_blocks is None else kv_peak_blocks,
                          c_exp, c_kv, None, 0)
        if m_kv is not None:
            arr = (C.c_double * len(m_kv))(*m_kv)
            inp.m_kv, inp.m_kv_len = arr, len(m_kv)
        eb, kb, mv = C.c_uint64(), C.c_uint64(), C.c_int32()
        self._ck(self.L.wisp_mvwsa_propose(self.ctx, C.byref(inp), C.byref(eb), C.byref(kb), C.byref(mv)), "wisp_mvwsa_propose")
        return eb.value, kb.value, bool(mv.value)
