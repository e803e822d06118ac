"""O1 — plain fp64 forward pass of the MoE decoder (ORACLE; test infrastructure).

ProMoE "performs computations that are equivalent to the original model"; the expert order is
interchangeable because expert outputs "are simply summed together".  So the oracle for OUTPUTS is the plain
offload-free model.  Structure: PAPER.md §2.1 and Fig. 2: each layer = self-attention + FFN, the FFN
being an MoE block "gate → top-k → experts → weighted sum"; prefill processes the whole prompt, decode one token per
iteration with a KV cache.  The paper gives no equations; the formulae are the standard ones of the named model
families under the readings of SURVEY.md §8(c) (G1, G8, G9, G11) restated in DESIGN.md:

    x = Emb[id]
    for each layer l:
       u1 = rmsnorm(x; ln1)                  y = x·rsqrt(mean(x²)+eps)·w
       q,k,v = Wqkv·u1 ; rope(q), rope(k) (rotate-half pairs (i, i+d/2), angle pos·θ^(−2i/d)) ; append k,v
       o_h = softmax(q_h·K_gᵀ/√d over positions ≤ pos)·V_g,  kv head g = ⌊h / (nq/nkv)⌋
       h = x + Wo·o ;  u = rmsnorm(h; ln2)
       dense layer:  y = FFN(u) = Wd·(silu(Wg·u) ⊙ (Wu·u))
       MoE layer:    z = R·u (+ b);  sel = top-k(z) (ties → lower index, by descending z)
                     g = softmax(z[sel])                                  (renormalised, Σg = 1; G8)
                     y = Σ_j (in j order) g_j·FFN_{sel_j}(u)  [+ σ(wsg·u)·FFN_sh(u) | + FFN_sh(u)]
       x = h + y
    logits = lm_head·rmsnorm(x_last; final_norm)

Weights are widened exactly (bf16/fp32 → fp64); activations are fp64 and never rounded (G1).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Dict, List, Optional, Tuple

import torch

from .predictor import predict_experts, predictor_scores, topk_desc
from .quant import dequant_expert

F64 = torch.float64


def rmsnorm(x: torch.Tensor, w: torch.Tensor, eps: float) -> torch.Tensor:
    return x * torch.rsqrt((x * x).mean(dim=-1, keepdim=True) + eps) * w.to(F64)


def rope(x: torch.Tensor, pos: torch.Tensor, theta: float) -> torch.Tensor:
    """x [T, n_heads, d]; pos [T] absolute positions.  Pair (i, i+d/2) rotated by angle pos·θ^(−2i/d)."""
    d = x.shape[-1]
    half = d // 2
    i = torch.arange(half, dtype=F64)
    freq = theta ** (-2.0 * i / d)
    ang = pos.to(F64)[:, None] * freq[None, :]            # [T, half]
    c, s = torch.cos(ang)[:, None, :], torch.sin(ang)[:, None, :]
    x1, x2 = x[..., :half], x[..., half:]
    return torch.cat([x1 * c - x2 * s, x2 * c + x1 * s], dim=-1)


def swiglu_ffn(u: torch.Tensor, wg: torch.Tensor, wu: torch.Tensor, wd: torch.Tensor) -> torch.Tensor:
    """u [n, H] → [n, H]:  Wd·(silu(Wg·u) ⊙ (Wu·u)),  silu(a) = a·σ(a)."""
    a = u @ wg.to(F64).T
    b = u @ wu.to(F64).T
    return ((a * torch.sigmoid(a)) * b) @ wd.to(F64).T


def route(z: torch.Tensor, k: int) -> Tuple[List[int], List[float], float]:
    """z [E] logits → (sel by descending z, ties → lower index; gates = softmax over the k selected; margin =
    z_(k) − z_(k+1), +inf when k = E)."""
    sel = topk_desc(z, k)
    zs = z[sel]
    g = torch.exp(zs - zs.max())
    g = g / g.sum()
    rest = [z[i].item() for i in range(z.numel()) if i not in sel]
    margin = (zs[-1].item() - max(rest)) if rest else float("inf")
    return sel, g.tolist(), margin


@dataclass
class LayerTrace:
    sel: List[List[int]]                 # [T][k]
    gates: List[List[float]]             # [T][k]
    margin: List[float]                  # [T]
    logits: torch.Tensor                 # router logits z [T, E]
    pred_scores: Optional[torch.Tensor]  # predictor scores [T, E] (predictor AT this layer)
    pred: Optional[List[int]]            # predicted list for MoE layer (this + stride), uncapped by G5


@dataclass
class StepTrace:
    layers: List[LayerTrace]             # one per MoE layer
    hidden: torch.Tensor                 # [T, H] residual stream after the full stack (before the final norm)
    logits: torch.Tensor                 # [vocab] of the last token
    next_token: int                      # argmax, ties → lower id


class OracleModel:
    """Plain decoder with KV cache.  `weights` is a synth.Weights; nothing here touches the expert cache."""

    def __init__(self, weights, stride: int = 1, slots_per_layer: Optional[int] = None, use_predictor: bool = True):
        self.w = weights
        self.s = weights.shape
        self.stride = stride
        self.cap = slots_per_layer if slots_per_layer is not None else self.s.n_experts
        self.use_predictor = use_predictor
        self.reset()
        self.overrides: Dict[Tuple[int, int, int], List[int]] = {}   # (step, moe_layer, token) → forced selection

    def reset(self) -> None:
        s = self.s
        self.kcache = [torch.zeros(0, s.n_kv_heads, s.head_dim, dtype=F64) for _ in range(s.n_layers)]
        self.vcache = [torch.zeros(0, s.n_kv_heads, s.head_dim, dtype=F64) for _ in range(s.n_layers)]
        self.pos = 0
        self.step_idx = 0

    # ---------------------------------------------------------------------------------------------------------
    def _attention(self, l: int, u1: torch.Tensor) -> torch.Tensor:
        s, D = self.s, self.w.dense
        T = u1.shape[0]
        nq, nkv, d = s.n_q_heads, s.n_kv_heads, s.head_dim
        qkv = u1 @ D[f"l{l}.wqkv"].to(F64).T
        q = qkv[:, :nq * d].reshape(T, nq, d)
        k = qkv[:, nq * d:(nq + nkv) * d].reshape(T, nkv, d)
        v = qkv[:, (nq + nkv) * d:].reshape(T, nkv, d)
        pos = torch.arange(self.pos, self.pos + T)
        q, k = rope(q, pos, s.rope_theta), rope(k, pos, s.rope_theta)
        self.kcache[l] = torch.cat([self.kcache[l], k], 0)
        self.vcache[l] = torch.cat([self.vcache[l], v], 0)
        K, V = self.kcache[l], self.vcache[l]              # [P, nkv, d], P = pos + T
        P = K.shape[0]
        out = torch.empty(T, nq, d, dtype=F64)
        causal = torch.arange(P)[None, :] <= pos[:, None]  # [T, P]
        for h in range(nq):
            g = h // (nq // nkv)
            sc = (q[:, h, :] @ K[:, g, :].T) / math.sqrt(d)
            sc = sc.masked_fill(~causal, float("-inf"))
            p = torch.exp(sc - sc.max(dim=-1, keepdim=True).values)
            out[:, h, :] = (p @ V[:, g, :]) / p.sum(dim=-1, keepdim=True)
        return out.reshape(T, nq * d) @ D[f"l{l}.wo"].to(F64).T

    def _moe(self, l: int, m: int, u: torch.Tensor) -> Tuple[torch.Tensor, LayerTrace]:
        s, D = self.s, self.w.dense
        T = u.shape[0]
        z = u @ D[f"l{l}.router"].to(F64).T
        if s.router_bias:
            z = z + D[f"l{l}.router_bias"].to(F64)
        sel, gates, margin = [], [], []
        for t in range(T):
            st, gt, mt = route(z[t], s.top_k)
            forced = self.overrides.get((self.step_idx, m, t))
            if forced is not None:                      # parity protocol P2: swap near-ties only
                st = list(forced)
                zs = z[t][st]
                g = torch.exp(zs - zs.max())
                gt = (g / g.sum()).tolist()
            sel.append(st); gates.append(gt); margin.append(mt)
        y = torch.zeros_like(u)
        # per expert, over the tokens that selected it; summed into y in fixed j order per token
        contrib = torch.zeros(T, s.top_k, s.hidden, dtype=F64)
        by_expert: Dict[int, List[Tuple[int, int]]] = {}
        for t in range(T):
            for j, e in enumerate(sel[t]):
                by_expert.setdefault(e, []).append((t, j))
        for e, pairs in sorted(by_expert.items()):
            if s.wdtype == 2:      # INT4 experts: dequantise, then the plain definition
                wg, wu, wd = dequant_expert(self.w.experts[m, e], s.hidden, s.expert_inter)
            else:
                wg, wu, wd = self.w.expert_views(m, e)
            rows = torch.tensor([t for t, _ in pairs])
            out = swiglu_ffn(u[rows], wg, wu, wd)
            for i, (t, j) in enumerate(pairs):
                contrib[t, j] = out[i]
        for j in range(s.top_k):
            y = y + torch.tensor([gates[t][j] for t in range(T)], dtype=F64)[:, None] * contrib[:, j]
        if s.n_shared_inter:
            sh = swiglu_ffn(u, D[f"l{l}.ffn_gate"], D[f"l{l}.ffn_up"], D[f"l{l}.ffn_down"])
            if s.shared_gate:
                sh = torch.sigmoid(u @ D[f"l{l}.shared_gate_w"].to(F64).T) * sh
            y = y + sh
        scores, pred = None, None
        if self.use_predictor:
            scores = predictor_scores(u, D[f"l{l}.pred_w1"], D[f"l{l}.pred_w2"])
            pred = predict_experts(scores, s.top_k, self.cap)
        return y, LayerTrace(sel=sel, gates=gates, margin=margin, logits=z, pred_scores=scores, pred=pred)

    def forward(self, ids) -> StepTrace:
        s, D = self.s, self.w.dense
        ids = torch.as_tensor(ids, dtype=torch.long).reshape(-1)
        x = D["emb"][ids].to(F64)
        traces: List[LayerTrace] = []
        m = 0
        for l in range(s.n_layers):
            u1 = rmsnorm(x, D[f"l{l}.ln1"], s.rms_eps)
            h = x + self._attention(l, u1)
            u = rmsnorm(h, D[f"l{l}.ln2"], s.rms_eps)
            if l < s.n_dense_layers:
                y = swiglu_ffn(u, D[f"l{l}.ffn_gate"], D[f"l{l}.ffn_up"], D[f"l{l}.ffn_down"])
            else:
                y, tr = self._moe(l, m, u)
                traces.append(tr)
                m += 1
            x = h + y
        self.pos += ids.numel()
        self.step_idx += 1
        xf = rmsnorm(x[-1:], D["final_norm"], s.rms_eps)
        logits = (xf @ D["lm_head"].to(F64).T)[0]
        nxt = int(torch.argmax(logits).item())   # torch.argmax returns the first maximal index
        mx = logits.max()
        nxt = int((logits == mx).nonzero()[0].item())
        return StepTrace(layers=traces, hidden=x, logits=logits, next_token=nxt)

    prefill = forward

    def decode(self, token_id: int) -> StepTrace:
        return self.forward([int(token_id)])


def needed_sets(step: StepTrace) -> List[List[int]]:
    return [sorted({e for row in lt.sel for e in row}) for lt in step.layers]


def pred_lists(step: StepTrace) -> List[Optional[List[int]]]:
    return [lt.pred for lt in step.layers]
