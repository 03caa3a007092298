"""Oracle O4: CPU simulation of the expert pager, Algorithm 1 `WISPLAYER.STEP(R)`.

TEST INFRASTRUCTURE (see oracle/__init__.py).  Pure Python integers, one layer per object.
Follows the algorithm line by line in the paper's notation (pi, pi^-1, tau, c); the readings the
paper leaves open are those of SURVEY.md §8(c) / DESIGN.md:
  G1  line 2 (lost in extraction):  M <- R \\ dom(pi)
  G2  victims "in increasing tau": ties -> lower slot index
  G3  ASSIGN: M in ascending expert id  <->  U in key order
  G4  empty slot: occupant is None (not in R), tau = 0  -> taken first
  G5  |R| > C: R sorted ascending is cut into consecutive waves of at most C ids; Alg. 1 per wave
  G6  LFU (not in the paper): key (f[occupant], tau, slot); f counts steps in which e was in R,
      survives eviction, never decays; an empty slot has f = -1
  G13 resize: keep the most-recently-used C~ residents, compact to slots < C~ (device move, byte-equal
      to the paper's re-page from host)
  G20 a reference = one (layer, step, distinct expert); hit iff resident when its wave begins
  G24 one tick per wave shared by all of R_w
  G25 wave order (PAPER.md:112 calls overflow handling an implementation detail):
      ASCENDING = G5; HITS_FIRST = only when |R| > C, R is listed as (members resident when the step
      begins, ascending id) followed by (the faults, ascending id) before it is cut into waves, so a
      resident member is never evicted by an earlier wave of the same step.  |R| <= C: identical to G5.
"""
from __future__ import annotations

from dataclasses import dataclass, field

HIT, MISS, RESIZE_DROP, RESIZE_MOVE, PREFETCH = 0, 1, 2, 3, 4
LRU, LFU = 0, 1
ASCENDING, HITS_FIRST = 0, 1


@dataclass
class Event:
    step: int
    wave: int
    expert: int
    slot: int
    evicted: int      # -1 none
    kind: int

    def key(self):
        return (self.step, self.wave, self.expert, self.slot, self.evicted, self.kind)


@dataclass
class PagerLayer:
    C: int
    E: int
    policy: int = LRU
    wave_order: int = ASCENDING
    pi: dict = field(default_factory=dict)        # expert -> slot
    pi_inv: list = field(default_factory=list)    # slot -> expert or None
    tau: list = field(default_factory=list)       # per-slot LRU tick
    f: list = field(default_factory=list)         # per-expert LFU count
    c: int = 0                                    # clock
    steps: int = 0
    hits: int = 0
    misses: int = 0
    evictions: int = 0
    references: int = 0
    prefetches: int = 0

    def __post_init__(self):
        self.pi_inv = [None] * self.C
        self.tau = [0] * self.C
        self.f = [0] * self.E

    # -- Algorithm 1 -------------------------------------------------------------------------
    def _victim_key(self, s: int):
        if self.policy == LRU:
            return (self.tau[s], s)
        occ = self.pi_inv[s]
        return (-1 if occ is None else self.f[occ], self.tau[s], s)

    def step(self, routed) -> list[Event]:
        """One forward of this layer.  `routed` = expert ids routed by all tokens (any order, repeats
        allowed); R is their set.  Returns the trace events in emission order."""
        R = sorted(set(int(e) for e in routed))
        if not R:
            return []                                   # n_tokens = 0: no-op, no tick (G23)
        if self.wave_order == HITS_FIRST and len(R) > self.C:      # G25
            R = [e for e in R if e in self.pi] + [e for e in R if e not in self.pi]
        events: list[Event] = []
        step_no = self.steps
        for wv, lo in enumerate(range(0, len(R), self.C)):
            Rw = R[lo:lo + self.C]
            in_wave = set(Rw)
            # 2: M <- R \ dom(pi)   (faults)
            M = [e for e in Rw if e not in self.pi]
            hit_set = [e for e in Rw if e in self.pi]
            # 3: U <- {s : pi^-1(s) not in R} in increasing tau   (victims; ties -> lower slot)
            U = sorted((s for s in range(self.C) if self.pi_inv[s] not in in_wave), key=self._victim_key)
            # 4-8: assign each e in M a victim slot; copy; update maps
            assign = {}
            for i, e in enumerate(M):
                s = U[i]
                old = self.pi_inv[s]
                if old is not None:
                    del self.pi[old]
                    self.evictions += 1
                self.pi[e] = s
                self.pi_inv[s] = e
                assign[e] = (s, -1 if old is None else old)
            # 9: c <- c+1; tau[pi(e)] <- c for e in R ; LFU count
            self.c += 1
            for e in Rw:
                self.tau[self.pi[e]] = self.c
                self.f[e] += 1
            self.hits += len(hit_set)
            self.misses += len(M)
            self.references += len(Rw)
            for e in Rw:                                 # wave order (ascending expert id under G5)
                if e in assign:
                    events.append(Event(step_no, wv, e, assign[e][0], assign[e][1], MISS))
                else:
                    events.append(Event(step_no, wv, e, self.pi[e], -1, HIT))
        self.steps += 1
        return events

    # -- speculative prefetch ----------------------------------
    def prefetch(self, experts) -> list[Event]:
        """Bring the predicted experts (best first) into the pool BEFORE this layer's next step.  Reading (G27):
        a resident expert is skipped; each other one takes the next victim in increasing policy key over ALL slots (no member
        of R protects a slot: the layer is not running; slots filled by this call are not victims again); the slot's tau
        becomes the current clock c (no tick: a prefetch is not a reference), f is untouched.  At a tight cap this can evict
        an expert the next step still needs -- the effect the paper reports."""
        events: list[Event] = []
        taken = set()
        for e in experts:
            e = int(e)
            if e in self.pi:
                continue
            free = [s for s in range(self.C) if s not in taken]
            if not free:
                break
            s = min(free, key=self._victim_key)
            old = self.pi_inv[s]
            if old is not None:
                del self.pi[old]
                self.evictions += 1
            self.pi[e] = s
            self.pi_inv[s] = e
            self.tau[s] = self.c
            taken.add(s)
            self.prefetches += 1
            events.append(Event(self.steps, 0, e, s, -1 if old is None else old, PREFETCH))
        return events

    # -- resize (a7) ---------------------------------------------------------------------------
    def resize(self, C_new: int) -> list[Event]:
        events: list[Event] = []
        step_no = self.steps
        if C_new < self.C:
            occ = [s for s in range(self.C) if self.pi_inv[s] is not None]
            if self.policy == LRU:
                occ.sort(key=lambda s: (-self.tau[s], s))
            else:
                occ.sort(key=lambda s: (-self.f[self.pi_inv[s]], -self.tau[s], s))
            keep, drop = occ[:C_new], occ[C_new:]
            for s in sorted(drop):
                e = self.pi_inv[s]
                del self.pi[e]
                self.pi_inv[s] = None
                self.tau[s] = 0
                events.append(Event(step_no, 0, e, s, -1, RESIZE_DROP))
            for s in sorted(x for x in keep if x >= C_new):
                dst = next(t for t in range(C_new) if self.pi_inv[t] is None)
                e = self.pi_inv[s]
                self.pi_inv[dst], self.tau[dst] = e, self.tau[s]
                self.pi_inv[s], self.tau[s] = None, 0
                self.pi[e] = dst
                events.append(Event(step_no, 0, e, dst, s, RESIZE_MOVE))   # `evicted` carries the source slot
            self.pi_inv = self.pi_inv[:C_new]
            self.tau = self.tau[:C_new]
        elif C_new > self.C:
            self.pi_inv += [None] * (C_new - self.C)
            self.tau += [0] * (C_new - self.C)
        self.C = C_new
        return events

    def slots(self) -> list:
        return list(self.pi_inv)

    def check_invariants(self):
        """P9: pi and pi^-1 mutually inverse; distinct slots."""
        for e, s in self.pi.items():
            assert self.pi_inv[s] == e
        for s, e in enumerate(self.pi_inv):
            if e is not None:
                assert self.pi[e] == s
            else:
                assert self.tau[s] == 0
        assert len(set(self.pi.values())) == len(self.pi)


# -- static layer-level offload: the paper's comparison arm (Table 2) --------------
def static_offload_bytes_per_forward(n_layers: int, n_experts: int, expert_bytes: int, budget_bytes: int) -> int:
    """Bytes a static layer-offload engine moves over the host link for ONE forward of the stack: it "streams the whole
    expert layer" for every layer the budget does not hold, whatever the routing.  Reading (G26):
    the budget holds whole layers of E * M_e bytes, two of them are bounce buffers (layer l+1 streams while layer l
    computes), the first floor(B / (E * M_e)) - 2 layers stay resident."""
    layer_bytes = n_experts * expert_bytes
    resident = max(0, min(n_layers, budget_bytes // layer_bytes - 2))
    return (n_layers - resident) * layer_bytes
