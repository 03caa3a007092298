"""Oracle for SURVEY.md 8(f) f3: the online co-activation predictor of App. E that drives the speculative
expert prefetch of Section 4.

TEST INFRASTRUCTURE (see oracle/__init__.py).  Pure Python, integer tables, fp64 scores.  Follows the construction in the
paper's notation:

    A_{l,l'}(e, e')          counts how often source expert e at layer l and target expert e' at layer l' > l fire in the
                             same forward pass
    P_{l,l'}(e' | e)       = A_{l,l'}(e, e') / sum_j A_{l,l'}(e, j)
    s_{l'}(e')             = sum_{l < l'} gamma^{l'-l} sum_{e in R_l} P_{l,l'}(e' | e)
    "The highest-scoring experts are used as the predicted target-layer experts."

Readings (G27; the paper gives no numbers or tie rules here):
  * the table starts empty and is learned online ("can start empty"); a forward pass is added to the table of
    target layer l' when layer l' has routed, so the prediction for l' (made when layer l'-1 has routed) sees earlier
    passes only;
  * sources are the `window` layers before the target (window = None: all earlier layers, the paper's sum);
  * gamma^dist is the running product g_1 = gamma, g_d = g_{d-1} * gamma (fp64);
  * the score is accumulated in this order: distance 1, 2, ... (nearest source layer first), source experts in ascending id,
    each term (A / rowsum) * g_dist added to s with IEEE fp64 round-to-nearest operations and no fused multiply-add -- the
    CUDA path does the same operations in the same order, so the ranking is bit-identical ("where floating point decides an
    integer, both sides take that decision in the same precision");
  * a source expert whose row is empty contributes nothing; candidates with score 0 are never predicted;
  * ranking: score descending, ties -> lower expert id.
"""
from __future__ import annotations


class CoActivationPredictor:
    def __init__(self, n_layers: int, n_experts: int, gamma: float = 0.5, window: int | None = 1):
        self.L, self.E = n_layers, n_experts
        self.window = n_layers if window is None else window
        self.gpow = [1.0]
        for _ in range(self.window):
            self.gpow.append(self.gpow[-1] * gamma)
        # tables of target layer l2 and distance dist = l2 - l (1..window): A[l2][dist][e][e2], row[l2][dist][e]
        self.A = {}
        self.row = {}
        self.R = [None] * n_layers          # routed sets of the forward pass in progress

    def _tab(self, l2, dist):
        key = (l2, dist)
        if key not in self.A:
            self.A[key] = [[0] * self.E for _ in range(self.E)]
            self.row[key] = [0] * self.E
        return self.A[key], self.row[key]

    def begin_pass(self):
        self.R = [None] * self.L

    def observe(self, layer: int, routed):
        """Layer `layer` of the pass in progress has routed to `routed`: record R_layer and add the pass to the tables whose
        TARGET is this layer."""
        R2 = sorted(set(int(e) for e in routed))
        self.R[layer] = R2
        for dist in range(1, self.window + 1):
            l = layer - dist
            if l < 0 or self.R[l] is None:
                continue
            A, row = self._tab(layer, dist)
            for e in self.R[l]:
                for e2 in R2:
                    A[e][e2] += 1
                row[e] += len(R2)

    def scores(self, target: int) -> list:
        """s_target(e') for every candidate e', from the layers of the pass in progress observed so far."""
        s = [0.0] * self.E
        for dist in range(1, self.window + 1):
            l = target - dist
            if l < 0 or self.R[l] is None or (target, dist) not in self.A:
                continue
            A, row = self.A[(target, dist)], self.row[(target, dist)]
            g = self.gpow[dist]
            for e in self.R[l]:
                if row[e] == 0:
                    continue
                for e2 in range(self.E):
                    s[e2] = s[e2] + (A[e][e2] / row[e]) * g
        return s

    def predict(self, target: int, n: int, resident=()) -> list:
        """The n highest-scoring experts of layer `target` that are not resident and have a positive score, best first."""
        s = self.scores(target)
        res = set(resident)
        cand = [e for e in range(self.E) if s[e] > 0.0 and e not in res]
        cand.sort(key=lambda e: (-s[e], e))
        return cand[:n]
