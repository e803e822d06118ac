"""Parity protocol P1-P4 (ORACLE side; test infrastructure): compares plain arrays read back from the CUDA path
with the oracle's StepTrace / cache simulator.  Imports nothing from the product package.

Rules (BASELINE.json north_star):
  * selections / permutations / cache traces bit-exact; a selection that differs from the oracle's is tolerated
    (counted, then forced into the oracle through `overrides` so nothing cascades, P2) only when every ordering
    decision it changes has an oracle logit margin < 1e-3;
  * gates: |gpu - cpu| <= 1e-4 (softmax over k fp32 logits); hidden: |gpu - cpu| <= 1e-2 + 1e-2*|cpu|;
  * logits top-1 equal unless the oracle's top-1/top-2 margin < 1e-3 (counted);
  * cache traces: O3 is a pure function of (routing, predictions), so it is driven with the GPU's own routing and
    prediction lists and compared with no tolerance (P3).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence

import numpy as np
import torch

from .cache_sim import ProMoECacheSim
from .forward import OracleModel, StepTrace
from .permute import permutation

MARGIN = 1e-3


@dataclass
class ParityReport:
    steps: int = 0
    token_layers: int = 0
    sel_near_tie: int = 0          # selections that differed inside the 1e-3 margin (counted, not failed)
    pred_near_tie: int = 0
    top1_near_tie: int = 0
    max_gate_err: float = 0.0
    max_hidden_ratio: float = 0.0  # max |gpu-cpu| / (1e-2 + 1e-2|cpu|)
    max_logit_err: float = 0.0
    reruns: int = 0
    notes: List[str] = field(default_factory=list)


def _consistent(order: Sequence[int], z: torch.Tensor, k: int) -> bool:
    """Is `order` (k experts, claimed descending) a valid top-k of z up to MARGIN?  Every ordering decision the list
    makes — adjacent entries, and its weakest entry against the strongest expert left out — must hold in the oracle's
    logits to within MARGIN.  A duplicate, a wrong length or an expert id outside [0, E) is never consistent."""
    E = z.numel()
    order = [int(e) for e in order]
    if len(order) != k or len(set(order)) != k or any(e < 0 or e >= E for e in order):
        return False
    zs = [z[e].item() for e in order]
    for a, b in zip(zs, zs[1:]):
        if a < b - MARGIN:
            return False
    rest = [z[i].item() for i in range(E) if i not in order]
    return not rest or min(zs) >= max(rest) - MARGIN


def snapshot(o: OracleModel):
    return ([t.clone() for t in o.kcache], [t.clone() for t in o.vcache], o.pos, o.step_idx)


def restore(o: OracleModel, snap) -> None:
    o.kcache = [t.clone() for t in snap[0]]
    o.vcache = [t.clone() for t in snap[1]]
    o.pos, o.step_idx = snap[2], snap[3]


def oracle_step_matching(o: OracleModel, ids, gpu_sel: np.ndarray, rep: ParityReport, max_reruns: int = 8) -> StepTrace:
    """Run one oracle step; where the GPU's selection differs inside the margin, force it (P2) and re-run so that
    everything downstream is compared exactly.  A difference outside the margin raises."""
    step_no = o.step_idx
    for attempt in range(max_reruns + 1):
        snap = snapshot(o)
        st = o.forward(ids)
        bad = []
        for m, lt in enumerate(st.layers):
            for t, row in enumerate(lt.sel):
                g = [int(x) for x in gpu_sel[m, t]]
                if g != row:
                    bad.append((m, t, g))
            if bad:
                break                      # later layers saw a different input; fix the first layer first
        if not bad:
            return st
        for m, t, g in bad:
            z = st.layers[m].logits[t]
            if not _consistent(g, z, len(g)):
                raise AssertionError(f"selection mismatch outside the {MARGIN} margin at step {step_no} layer {m} token {t}: "
                                     f"gpu {g} oracle {st.layers[m].sel[t]} margin {st.layers[m].margin[t]:.3e}")
            o.overrides[(step_no, m, t)] = g
            rep.sel_near_tie += 1
        restore(o, snap)
        rep.reruns += 1
    raise AssertionError("too many near-tie reruns")


def vote_bounds(scores: torch.Tensor, k: int):
    """Per-expert vote interval [lo, hi] of the prefill predictor (reading G7) when every token's top-k is only known
    up to MARGIN.  For one token with sorted scores s_(1) >= ... >= s_(E): an expert of the top-k with s_e > s_(k+1) + MARGIN
    is in every margin-consistent top-k (it votes in lo and hi); any other expert with s_e >= s_(k) - MARGIN MAY be in
    one (hi only); everything else never votes.  With no near tie at the k/(k+1) boundary lo == hi == the
    plain vote count."""
    T, E = scores.shape
    lo, hi = [0] * E, [0] * E
    for t in range(T):
        row = scores[t].tolist()
        srt = sorted(row, reverse=True)
        kth = srt[k - 1]
        nxt = srt[k] if k < E else float("-inf")
        for e in range(E):
            if row[e] >= kth and row[e] > nxt + MARGIN:     # no margin-consistent top-k leaves e out
                lo[e] += 1; hi[e] += 1
            elif row[e] >= kth - MARGIN:                    # some margin-consistent top-k contains e
                hi[e] += 1
    return lo, hi


def pred_list_acceptable(gpu_list: Sequence[int], scores: torch.Tensor, k: int, cap: int) -> bool:
    """Per-decision check of a predicted list that differs from the oracle's (O2, reading G7).

    Decode (T = 1): the list must be a margin-consistent top-min(k, cap) of the token's scores (`_consistent`).
    Prefill (T > 1): the list must be a possible outcome of "experts by votes descending, ties -> lower id, first
    min(#voted, cap)" for SOME vote vector inside `vote_bounds` (only tokens whose own k/(k+1) score gap is below
    MARGIN can move a vote): every ordering decision the list makes — each listed expert against each later listed
    one and against every voted expert left out — must be attainable, and its length must be attainable."""
    T, E = scores.shape
    gl = [int(e) for e in gpu_list]
    if len(set(gl)) != len(gl) or any(e < 0 or e >= E for e in gl):
        return False
    if T == 1:
        return _consistent(gl, scores[0], min(k, cap))
    lo, hi = vote_bounds(scores, k)
    n_lo, n_hi = min(cap, sum(1 for v in lo if v > 0)), min(cap, sum(1 for v in hi if v > 0))
    if not (n_lo <= len(gl) <= n_hi):
        return False
    if any(hi[e] == 0 for e in gl):
        return False

    def may_precede(a: int, b: int) -> bool:      # can a rank before b?  votes_a > votes_b, or equal and a < b
        return hi[a] > lo[b] or (hi[a] == lo[b] and a < b)

    for i, a in enumerate(gl):
        for b in gl[i + 1:]:
            if not may_precede(a, b):
                return False
    if len(gl) == cap:                              # the list is full: every expert left out ranks after all of it
        for b in range(E):
            if b in gl or lo[b] == 0:
                continue
            if not all(may_precede(a, b) for a in gl):
                return False
    else:                                           # shorter than cap: every expert left out must be able to have no vote
        if any(lo[b] > 0 for b in range(E) if b not in gl):
            return False
    return True


def compare_step(gpu: Dict[str, np.ndarray], st: StepTrace, n_experts: int, rep: ParityReport,
                 gpu_logits: Optional[np.ndarray] = None, check_pred: bool = True, pred_cap: Optional[int] = None) -> None:
    Lm = len(st.layers)
    T = len(st.layers[0].sel)
    k = len(st.layers[0].sel[0])
    rep.steps += 1
    rep.token_layers += Lm * T
    for m, lt in enumerate(st.layers):
        assert gpu["sel"][m].tolist() == lt.sel, f"layer {m}: selections differ after overrides"
        ge = np.abs(gpu["gates"][m].astype(np.float64) - np.asarray(lt.gates)).max()
        rep.max_gate_err = max(rep.max_gate_err, float(ge))
        assert ge <= 1e-4, f"layer {m}: gate error {ge}"
        zerr = np.abs(gpu["z"][m].astype(np.float64) - lt.logits.numpy()).max()
        assert zerr <= MARGIN, f"layer {m}: router logit error {zerr}"
        if T > 1:   # P4 permutation, bit-exact given equal selections
            cnt, off, perm, inv = permutation(lt.sel, n_experts)
            row = gpu["perm"][m]
            E = n_experts
            assert row[:E].tolist() == cnt, f"layer {m}: histogram"
            assert row[E:2 * E + 1].tolist() == off, f"layer {m}: offsets"
            assert row[2 * E + 1:2 * E + 1 + T * k].tolist() == perm, f"layer {m}: perm"
            assert row[2 * E + 1 + T * k:].tolist() == inv, f"layer {m}: inv"
        if check_pred and lt.pred is not None:
            n = int(gpu["predlist"][m, 0])
            gl = gpu["predlist"][m, 1:1 + n].tolist()
            if gl != lt.pred:
                assert pred_list_acceptable(gl, lt.pred_scores, k, pred_cap if pred_cap is not None else n_experts), \
                    f"layer {m}: predicted list {gl} != oracle {lt.pred} and not explained by score gaps < {MARGIN}"
                rep.pred_near_tie += 1
    hid = st.hidden.numpy()
    ratio = np.abs(gpu["hidden"].astype(np.float64) - hid) / (1e-2 + 1e-2 * np.abs(hid))
    rep.max_hidden_ratio = max(rep.max_hidden_ratio, float(ratio.max()))
    assert ratio.max() <= 1.0, f"hidden state outside 1e-2 + 1e-2|cpu| (ratio {ratio.max():.3f})"
    if gpu_logits is not None:
        lo = st.logits.numpy()
        rep.max_logit_err = max(rep.max_logit_err, float(np.abs(gpu_logits - lo).max()))
        g1 = int(np.flatnonzero(gpu_logits == gpu_logits.max())[0])
        if g1 != st.next_token:
            srt = np.sort(lo)
            assert srt[-1] - srt[-2] < MARGIN, f"logits top-1 differs: gpu {g1} oracle {st.next_token}"
            rep.top1_near_tie += 1


def compare_cache(sim: ProMoECacheSim, gpu: Dict[str, np.ndarray], stride: int, use_pred: bool,
                  max_spec: Optional[int] = None) -> None:
    """P3: drive O3 with the GPU's own routing + prediction lists for one step; records must match bit for bit."""
    Lm, E = sim.L, sim.E
    needed = [sorted(set(int(e) for e in gpu["sel"][m].reshape(-1))) for m in range(Lm)]
    preds = []
    for m in range(Lm):
        n = int(gpu["predlist"][m, 0])
        preds.append(gpu["predlist"][m, 1:1 + n].tolist() if use_pred else None)
    out = sim.run_step(needed, preds, stride, max_spec)
    for m, (prec, _) in enumerate(out):
        row = gpu["precise"][m]
        n = int(row[0])
        got = [tuple(int(x) for x in row[1 + 5 * i:6 + 5 * i]) for i in range(n)]
        assert got == prec.as_tuples(), f"layer {m}: PushPrecise trace differs\n gpu    {got}\n oracle {prec.as_tuples()}"
    # row mt of the GPU pred trace = the push INTO layer mt (made at layer mt - stride)
    for m, (_, pr) in enumerate(out):
        mt = m + stride
        if mt >= Lm:
            continue
        row = gpu["pred"][mt]
        n = int(row[0])
        got = [tuple(int(x) for x in row[1 + 4 * i:5 + 4 * i]) for i in range(n)]
        want = pr.as_tuples() if pr is not None else []
        assert got == want, f"push into layer {mt}: PushPredicted trace differs\n gpu    {got}\n oracle {want}"


STAT_KEYS = ("accesses", "hits_resident", "hits_prefetch", "misses", "evictions", "predicted", "predicted_correct",
             "pred_allocs", "need_experts")


def compare_stats(sim: ProMoECacheSim, gpu_stats: Dict[str, float]) -> None:
    for key in STAT_KEYS:
        assert int(gpu_stats[key]) == getattr(sim.stats, key), f"stat {key}: gpu {gpu_stats[key]} oracle {getattr(sim.stats, key)}"
