"""Token→expert permutation (ORACLE; test infrastructure).

Definition (the paper leaves this to the framework, P:277 only fixes that expert
outputs are "simply summed"): for a step with T tokens and selections sel[t, j] (j < k),
  count[e]  = #{(t, j) : sel[t, j] = e}
  offset[e] = sum_{e' < e} count[e']            (groups laid out in ascending expert id), offset[E] = T·k
  pos(t, j) = offset[e] + #{(t', j') : sel[t', j'] = e, t' < t}     with e = sel[t, j]
              (a token selects an expert at most once, so t' < t orders the group token-ascending)
  perm[pos(t, j)] = t·k + j          inv[t·k + j] = pos(t, j)
"""
from __future__ import annotations

from typing import List, Tuple


def permutation(sel: List[List[int]], n_experts: int) -> Tuple[List[int], List[int], List[int], List[int]]:
    T = len(sel)
    k = len(sel[0]) if T else 0
    count = [0] * n_experts
    for t in range(T):
        for j in range(k):
            count[sel[t][j]] += 1
    offset = [0] * (n_experts + 1)
    for e in range(n_experts):
        offset[e + 1] = offset[e] + count[e]
    fill = [0] * n_experts
    perm = [-1] * (T * k)
    inv = [-1] * (T * k)
    for t in range(T):                      # token-ascending inside every group
        for j in range(k):
            e = sel[t][j]
            p = offset[e] + fill[e]
            fill[e] += 1
            perm[p] = t * k + j
            inv[t * k + j] = p
    return count, offset, perm, inv
