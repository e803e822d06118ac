"""O2 — learned stride predictor, online inference (ORACLE; test infrastructure).

PAPER.md §4.3: a small MLP per layer reads "the input for each layer" and outputs, "similar to a gate's
output", a priority per expert; it "selects the same number of experts that the model would activate for one token"
(P:163).  §6.3: a 2-layer MLP.  §4.4: stride prefetching = predict a layer further ahead.
Readings: input = u_l (the post-attention RMSNorm output the router of layer l
reads), p = W2·ReLU(W1·u), no biases; top-k by score, ties → lower index, listed by descending score;
T > 1 tokens (prefill): per-token top-k → vote histogram → experts by votes descending (ties → lower id) → the first
min(#voted, cap) of them, cap = slots of the target layer.
"""
from __future__ import annotations

from typing import List

import torch


def topk_desc(scores: torch.Tensor, k: int) -> List[int]:
    """Indices of the k largest entries, by descending value, ties → lower index (plain selection)."""
    vals = scores.tolist()
    order = sorted(range(len(vals)), key=lambda i: (-vals[i], i))
    return order[:k]


def predictor_scores(u: torch.Tensor, w1: torch.Tensor, w2: torch.Tensor) -> torch.Tensor:
    """u [T, H] fp64; w1 [ph, H], w2 [E, ph] (any float dtype, widened exactly) → scores [T, E] fp64."""
    h = torch.relu(u @ w1.to(torch.float64).T)
    return h @ w2.to(torch.float64).T


def predict_experts(scores: torch.Tensor, k: int, cap: int) -> List[int]:
    """scores [T, E] → predicted expert list for the target layer (decode T = 1: the top-k list)."""
    T, E = scores.shape
    if T == 1:
        return topk_desc(scores[0], k)[:cap]
    votes = [0] * E
    for t in range(T):
        for e in topk_desc(scores[t], k):
            votes[e] += 1
    order = sorted((e for e in range(E) if votes[e] > 0), key=lambda e: (-votes[e], e))
    return order[:cap]
