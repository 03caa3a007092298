"""CPU oracle for the WiSP hot path -- TEST INFRASTRUCTURE, NOT PRODUCT.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference` legs
may import anything from this package.  It shares no code with `paper_2606_21868_b200/` (the CUDA
path) and never imports it; the only module both sides use is `synth_inputs` (seeded input
generators, no method arithmetic).

Parts (every function cites the PAPER.md passage or DESIGN.md reading it follows):
  moe_forward.py  O1 router/top-k/softmax, O2 SwiGLU FFN + weighted combine, O3 residual stack
  paging.py       O4 Algorithm 1 with LRU/LFU, overflow waves, resize
  mvwsa.py        O5 reuse-distance miss curves, Eq. 2-8, KV model

Pins (tests/test_oracle_*.py, `-m "not gpu"`): hand-worked cases, brute force, the paper's printed
numbers (tests/golden/*.txt).  Unpinned parts ("parity unpinned"): the k>1 reuse-distance
*estimator* of Algorithm 1's misses beyond monotonicity/limits (P7), and the KV-reservation
scheduler model and the controller constants lambda / hysteresis: this build's
own readings with no paper value to check against.
"""
