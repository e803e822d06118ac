"""CPU ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.

A plain, slow, obviously-correct fp64 restatement of what the ProMoE hot path computes (PAPER.md =
/root/reference/PAPER.md of arxiv 2410.22134; `P:NNN` = its line NNN), written from the paper and SURVEY.md §8(c):

  forward.py    O1  decoder forward pass (the "original model" ProMoE must stay equivalent to)
  predictor.py  O2  learned stride predictor inference (§4.3, §4.4)
  permute.py        token→expert permutation definition (histogram / offsets / stable order)
  cache_sim.py  O3  logical-time ProMoE cache + prefetcher state machine (Alg. 1, Alg. 2)
  accounting.py     byte / roofline accounting (P:85 worked numbers)
  compare.py        parity protocol P1-P4: compares arrays read back from the CUDA path with the three parts above

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may import this
package.  It shares no code with `paper_2410_22134_b200/` and never imports it; inputs come from `synth/`.

Pins (tests/test_oracle_*.py, `-m "not gpu"`): every function here is pinned to something other than itself —
closed forms, brute force, library cross-checks (torch fp64 SDPA / rms_norm), the paper's Fig. 9 worked example
and P:85 byte counts, a textbook LRU, the `max_spec` knob's special cases, and the method's invariants (outputs independent of cache
parameters).
Parity unpinned: none of the functions here; FetchRate / hidden-copy fraction / tokens/s are GPU-only timing
statistics with no oracle counterpart.
"""
