"""Oracle O5: MV-WSA restatement (§3.2-3.5, Eq. 2-5; App. B, Eq. 6-8).

TEST INFRASTRUCTURE (see oracle/__init__.py).  Pure Python, integers and fp64.
Readings (SURVEY.md §8(c) / DESIGN.md): G10 floor brackets in Eq. 7, 8; G11 constants h = 0.2,
Delta = 1, C_min = k, lambda = 0.5; G12 KV cost model = reservation/preemption scheduler below.
Pins (tests/): Table 4 (P6), hand-stepped KV schedule (tests/golden/hand_kv_schedule.txt), two-period decay hand case,
Mattson k = 1 equality (P7), brute-force argmin == greedy (P10).  Still "parity unpinned": the k > 1 reuse-distance
ESTIMATOR of Algorithm 1's miss count beyond monotonicity and its limits (P7), and the VALUES of the constants lambda = 0.5,
h = 0.2, Delta = 1 (G11: the paper gives none).
"""
from __future__ import annotations

import math
from collections import deque
from dataclasses import dataclass, field

INF = math.inf


# -- reuse-distance histograms and miss curves ------------------------------------
def stack_distances(stream) -> list:
    """Stack (reuse) distance of every reference of a linear reference stream: the number of DISTINCT
    items referenced since the previous reference to the same item, counting the item itself
    (1 = immediate re-reference, INF = first reference).  Textbook Mattson LRU stack."""
    stack: list = []          # most recent first
    out = []
    for e in stream:
        if e in stack:
            i = stack.index(e)
            out.append(i + 1)
            del stack[i]
        else:
            out.append(INF)
        stack.insert(0, e)
    return out


def linearise(steps) -> list:
    """One layer's reference stream: steps in order, distinct ids ascending within a step."""
    out = []
    for R in steps:
        out.extend(sorted(set(R)))
    return out


def histogram(distances, max_d: int) -> list:
    """hist[d] for d = 1..max_d (index 0 unused), hist[max_d+1] = count of distances > max_d (incl. INF)."""
    h = [0.0] * (max_d + 2)
    for d in distances:
        h[d if d <= max_d else max_d + 1] += 1.0
    return h


def miss_curve_from_hist(hist, max_d: int) -> list:
    """m(C) = #{refs with distance > C} for C = 0..max_d."""
    total = sum(hist[1:])
    out, acc = [], 0.0
    for C in range(0, max_d + 1):
        if C >= 1:
            acc += hist[C]
        out.append(total - acc)
    return out


def miss_curve(layer_streams, max_c: int) -> list:
    """m_exp(C) = sum over layers of #{refs with stack distance > C}, C = 0..max_c."""
    tot = [0.0] * (max_c + 1)
    for steps in layer_streams:
        mc = miss_curve_from_hist(histogram(stack_distances(linearise(steps)), max_c), max_c)
        tot = [a + b for a, b in zip(tot, mc)]
    return tot


def decay(hist, lam: float) -> list:
    """'Decayed' histograms: multiply all bins by lambda at each controller period."""
    return [lam * v for v in hist]


# -- Eq. 2-5: cost and configurator ---------------------------------------------------------------
def kappa_of(C: int, B: int, a: int, b: int) -> int:
    """kappa(C) = floor((B - C*a) / b)."""
    return (B - C * a) // b


def kappa_min(W: int, l_ctx: int, b_tok: int) -> int:
    """Eq. 4: kappa_min = W * ceil(l_ctx / b_tok)."""
    return W * -(-l_ctx // b_tok)


def cost(C: int, *, B, a, b, c_exp, c_kv, m_exp, m_kv) -> float:
    """Eq. 2: T = c_exp * m_exp(C) + c_kv * m_kv(kappa(C)).
    m_exp: sequence indexed by C; m_kv: callable kappa -> cost count."""
    return c_exp * m_exp[C] + c_kv * m_kv(kappa_of(C, B, a, b))


def configurator(*, B, a, b, kappa_floor, c_exp, c_kv, m_exp, m_kv, C_min, C_max):
    """Eq. 3-5: C_feas = floor((B - kappa_min*b)/a);
    C^ = argmin_{C_min <= C <= min(C_max, C_feas)} T(C), ties -> smaller C; B_kv = B - C*a.
    Exhaustive argmin (brute-force statement of the equimarginal point).  Returns (C, B_kv) or None."""
    C_feas = (B - kappa_floor * b) // a
    hi = min(C_max, C_feas)
    if hi < C_min:
        return None
    best_C, best_T = None, None
    for C in range(C_min, hi + 1):
        T = cost(C, B=B, a=a, b=b, c_exp=c_exp, c_kv=c_kv, m_exp=m_exp, m_kv=m_kv)
        if best_T is None or T < best_T:
            best_C, best_T = C, T
    return best_C, B - best_C * a


def greedy_marginal_walk(*, B, a, b, kappa_floor, c_exp, c_kv, m_exp, m_kv, C_min, C_max):
    """'Move bytes toward whichever pool currently removes more latency per byte':
    start at C_min and give `a` more bytes to experts while that lowers T.  Equals the argmin on
    convex curves (pin P10)."""
    C_feas = (B - kappa_floor * b) // a
    hi = min(C_max, C_feas)
    if hi < C_min:
        return None
    kw = dict(B=B, a=a, b=b, c_exp=c_exp, c_kv=c_kv, m_exp=m_exp, m_kv=m_kv)
    C = C_min
    while C + 1 <= hi and cost(C + 1, **kw) < cost(C, **kw):
        C += 1
    return C, B - C * a


# -- Eq. 6-8: live dual-resize law -------------------------------------------
def live_law(*, B, a, b, kappa_floor, p, h, C_min, C_max, C_cur, delta):
    """kappa~ = max(kappa_min, ceil((1+h) p));  C~ = clip(floor((B - kappa~ b)/a), C_min, C_max);
    kappa~ <- floor((B - C~ a)/b);  apply only if |C~ - C| >= Delta.  B, a, b may be ints (bytes)
    or floats (GiB, for the Table 4 pin).  Returns (C_new, kappa_new, moved)."""
    k1 = max(kappa_floor, math.ceil((1.0 + h) * p))
    Ct = math.floor((B - k1 * b) / a)
    Ct = max(C_min, min(C_max, Ct))
    k2 = math.floor((B - Ct * a) / b)
    if abs(Ct - C_cur) < delta:
        return C_cur, math.floor((B - C_cur * a) / b), False
    return Ct, k2, True


# -- KV-reservation scheduler model (config 5; harness-level; parity unpinned) --------------------
@dataclass
class Request:
    rid: int
    prompt: int
    target: int
    generated: int = 0
    blocks: int = 0


@dataclass
class KVScheduler:
    """FCFS admission on block reservations; a running request holds ceil((P+g)/block_tokens) blocks;
    when a block is needed and none is free, the most recently admitted running request is preempted
    (releases all blocks, goes to the head of the waiting queue, re-prefills P+g tokens)."""
    kappa: int
    block_tokens: int = 16
    waiting: deque = field(default_factory=deque)
    running: list = field(default_factory=list)
    used: int = 0
    peak: int = 0
    preemptions: int = 0
    reprefill_tokens: int = 0

    def need(self, r: Request) -> int:
        return -(-(r.prompt + r.generated) // self.block_tokens)

    def admit(self) -> list:
        """Admit FCFS while the head's blocks fit; returns [(request, tokens_to_prefill)]."""
        out = []
        while self.waiting:
            r = self.waiting[0]
            n = self.need(r)
            if self.used + n > self.kappa:
                break
            self.waiting.popleft()
            r.blocks = n
            self.used += n
            self.peak = max(self.peak, self.used)
            self.running.append(r)
            out.append((r, r.prompt + r.generated))
        return out

    def decode_tick(self) -> list:
        """Every running request produces one token; grows reservations, preempting if needed.
        Returns the requests that decoded this tick (in running order)."""
        i = 0
        while i < len(self.running):
            r = self.running[i]
            n = -(-(r.prompt + r.generated + 1) // self.block_tokens)
            while n > r.blocks and self.used + (n - r.blocks) > self.kappa and len(self.running) > 1:
                v = self.running.pop()                     # most recently admitted
                self.used -= v.blocks
                v.blocks = 0
                self.preemptions += 1
                self.reprefill_tokens += v.prompt + v.generated
                self.waiting.appendleft(v)
                if v is r:
                    break
            if r.blocks == 0 and r not in self.running:
                continue
            if n > r.blocks:
                self.used += n - r.blocks
                r.blocks = n
                self.peak = max(self.peak, self.used)
            i += 1
        done = list(self.running)
        for r in done:
            r.generated += 1
        for r in [x for x in self.running if x.generated >= x.target]:
            self.used -= r.blocks
            self.running.remove(r)
        return done
