"""Request scheduler of BASELINE.json config 5 (harness side): KV blocks are modelled as reservations.

This is the ONE harness implementation of the KV-reservation model that `bench.py --workload mvwsa` drives
(G12/G14/G15).  The paper only says "KV miss or recompute cost"; the model
is: a request holds ceil((prompt + generated) / block_tokens) blocks; admission is FCFS while the head's blocks fit;
when a running request needs one more block and none is free, the most recently admitted running request is preempted
(all its blocks released, back to the head of the queue, it re-prefills prompt + generated tokens on re-admission).
`tests/test_kv_sched.py` steps it by hand (tests/golden/hand_kv_schedule.txt) and against `oracle/mvwsa.py:KVScheduler`.

Holds no CUDA and no method arithmetic; reservations go out through the `reserve` callback (wisp_kv_reserve).
"""
from __future__ import annotations

from dataclasses import dataclass


@dataclass
class KvRequest:
    rid: int
    prompt: int
    target: int
    gen: int = 0
    blocks: int = 0
    t_first: float | None = None


class KvReservationScheduler:
    def __init__(self, kappa: int, requests, *, block_tokens: int = 16, reserve=None):
        self.kappa = int(kappa)               # cached: refresh with set_kappa() after a successful wisp_set_split
        self.block_tokens = block_tokens
        self._reserve = reserve or (lambda delta: None)
        self.waiting = list(requests)
        self.running: list[KvRequest] = []
        self.done: list[KvRequest] = []
        self.used = 0
        self.peak = 0                          # since construction
        self.window_peak = 0                   # since the last reset_window(): p of Eq. 6
        self.preemptions = 0
        self.reprefill_tokens = 0

    def set_kappa(self, kappa: int):
        self.kappa = int(kappa)

    def reset_window(self):
        self.window_peak = self.used

    def _blocks(self, tokens: int) -> int:
        return -(-tokens // self.block_tokens)

    def _take(self, delta: int):
        self._reserve(delta)
        self.used += delta
        self.peak = max(self.peak, self.used)
        self.window_peak = max(self.window_peak, self.used)

    def admit(self):
        """FCFS while the head fits.  Returns [(request, tokens to (re-)prefill)]."""
        out = []
        while self.waiting:
            r = self.waiting[0]
            n = self._blocks(r.prompt + r.gen)
            if self.used + n > self.kappa:
                break
            self.waiting.pop(0)
            self._take(n)
            r.blocks = n
            self.running.append(r)
            out.append((r, r.prompt + r.gen))
        return out

    def grow_for_decode(self):
        """Make room for one more token of every running request, preempting from the tail of the admission order.
        Returns the requests that decode in this iteration (admission order)."""
        i = 0
        while i < len(self.running):
            r = self.running[i]
            n = self._blocks(r.prompt + r.gen + 1)
            preempted_self = False
            while n > r.blocks and self.used + (n - r.blocks) > self.kappa and len(self.running) > 1:
                v = self.running.pop()
                self._take(-v.blocks)
                v.blocks = 0
                self.preemptions += 1
                self.reprefill_tokens += v.prompt + v.gen
                self.waiting.insert(0, v)
                if v is r:
                    preempted_self = True
                    break
            if preempted_self:
                continue
            if n > r.blocks:
                self._take(n - r.blocks)
                r.blocks = n
            i += 1
        return list(self.running)

    def finish_tick(self):
        """Every running request produced a token; requests that reached their target release their blocks."""
        for r in self.running:
            r.gen += 1
        for r in [x for x in self.running if x.gen >= x.target]:
            self._take(-r.blocks)
            r.blocks = 0
            self.running.remove(r)
            self.done.append(r)
