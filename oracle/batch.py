"""Batched decode (ORACLE; test infrastructure): B independent sequences that share one expert cache.

PAPER.md §7.5 varies the batch size from 1 to 4: "more experts are activated" per step, which stresses the
cache.  The MODEL is unchanged — each sequence is the plain decoder of oracle/forward.py with its own KV cache and position
(outputs equivalent to the original model) — so the oracle for outputs is B independent `OracleModel`s.  What the
batch shares is the MoE step state: one gate per layer sees the B new tokens, `needed` = the union of their selections,
and the stride predictor of a layer reads the B hidden states and votes (reading G7, the T > 1 rule of O2).

`OracleBatch.forward(ids)` therefore returns ONE StepTrace with T = B rows per layer, built from the B single-token
steps; it offers the attributes `oracle/compare.py`'s near-tie protocol (P2) uses (`overrides`, `step_idx`, snapshot /
restore through `kcache` / `vcache` / `pos`), mapping a forced selection of batch row b to sequence b's own step.
"""
from __future__ import annotations

from typing import Dict, List, Sequence, Tuple

import torch

from .forward import LayerTrace, OracleModel, StepTrace
from .predictor import predict_experts


class OracleBatch:
    def __init__(self, weights, n_seq: int, stride: int = 1, slots_per_layer=None, use_predictor: bool = True):
        self.seqs = [OracleModel(weights, stride=stride, slots_per_layer=slots_per_layer, use_predictor=use_predictor)
                     for _ in range(n_seq)]
        self.s = weights.shape
        self.cap = self.seqs[0].cap
        self.use_predictor = use_predictor
        self.step_idx = 0
        self.overrides: Dict[Tuple[int, int, int], List[int]] = {}   # (batch step, moe layer, batch row) → forced selection

    # ---- what snapshot() / restore() of oracle/compare.py touch ----------------------------------------------
    @property
    def kcache(self):
        return [t for o in self.seqs for t in o.kcache]

    @kcache.setter
    def kcache(self, flat):
        L = self.s.n_layers
        for i, o in enumerate(self.seqs):
            o.kcache = list(flat[i * L:(i + 1) * L])

    @property
    def vcache(self):
        return [t for o in self.seqs for t in o.vcache]

    @vcache.setter
    def vcache(self, flat):
        L = self.s.n_layers
        for i, o in enumerate(self.seqs):
            o.vcache = list(flat[i * L:(i + 1) * L])

    @property
    def pos(self):
        return tuple((o.pos, o.step_idx) for o in self.seqs)

    @pos.setter
    def pos(self, v):
        for o, (p, si) in zip(self.seqs, v):
            o.pos, o.step_idx = p, si

    # ---- steps -----------------------------------------------------------------------------------------------
    def prefill_seq(self, b: int, ids) -> StepTrace:
        """The prompt of sequence b (an ordinary single-sequence step, compared like one)."""
        return self.seqs[b].forward(ids)

    def forward(self, ids: Sequence[int]) -> StepTrace:
        """One batched decode step: ids[b] is the new token of sequence b."""
        assert len(ids) == len(self.seqs)
        subs = []
        for b, (o, tok) in enumerate(zip(self.seqs, ids)):
            for (st_no, m, t), forced in self.overrides.items():
                if st_no == self.step_idx and t == b:
                    o.overrides[(o.step_idx, m, 0)] = forced
            subs.append(o.forward([int(tok)]))
        self.step_idx += 1
        k = self.s.top_k
        layers = []
        for m in range(len(subs[0].layers)):
            rows = [st.layers[m] for st in subs]
            scores, pred = None, None
            if self.use_predictor:
                scores = torch.cat([r.pred_scores for r in rows], 0)          # [B, E]
                pred = predict_experts(scores, k, self.cap)                     # B = 1: the top-k list; B > 1: votes (G7)
            layers.append(LayerTrace(sel=[r.sel[0] for r in rows], gates=[r.gates[0] for r in rows],
                                     margin=[r.margin[0] for r in rows], logits=torch.cat([r.logits for r in rows], 0),
                                     pred_scores=scores, pred=pred))
        last = subs[-1]
        st = StepTrace(layers=layers, hidden=torch.cat([s_.hidden for s_ in subs], 0), logits=last.logits,
                       next_token=last.next_token)
        st.seq_logits = [s_.logits for s_ in subs]          # per-sequence logits / next tokens
        st.seq_next = [s_.next_token for s_ in subs]
        return st
