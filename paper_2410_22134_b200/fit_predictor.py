"""Offline fitting of the learned stride predictor (§4.3: "we collect traces ... offline, split 9:1 into
a training and a test set and train the predictor"; §6.3: a 2-layer MLP per layer; §4.4: stride).

    python -m paper_2410_22134_b200.fit_predictor --config c2 [--stride 2] [--prompts 16]

What is fitted: for every MoE layer m with m + stride < n_moe, the MLP  p = W2·ReLU(W1·u_m)  (hidden → pred_hidden → E, no
biases; the shape the hot path runs, A5) against the experts the gate of layer m + stride selects for the same token.
Where the traces come from: the synthetic model itself (there are no ShareGPT prompts or checkpoints here) —
seeded random prompts, DISJOINT from the prompt and decode ids bench.py and the tests use, run through the library's own
prefill with PROMOE_F_TRACE_U; u_m and the selections are read back through promoe_get_trace.  This is the method's
offline step, not its hot path: the optimiser is torch's (on the GPU when there is one).

Start point = the training-free `skip` construction the weights already hold (W1 = [R; −R; 0], W2 = [I, −I, 0], R the
router of the target layer); the free hidden units start from small random rows.  Loss = cross-entropy between
softmax(p) and the uniform distribution over the k selected experts (the predictor's output is "similar to a gate's
output"); Adam; the 9:1 split is by PROMPT (whole prompts held out: tokens of one prompt share their attention
context); the checkpoint with the best held-out accuracy is kept, and a layer whose fitted MLP does not beat `skip` on the
held-out prompts keeps the `skip` weights — "fitted" is never worse than its start point on held-out prompts.
Accuracy = |top-k(p) ∩ selected| / k, measured with the weights rounded to the model's dtype, as the GPU sees them.
"""
from __future__ import annotations

import argparse
import json
import time
from dataclasses import replace
from typing import Dict, List, Tuple

import numpy as np
import torch

from . import binding as B
from .engine import ProMoE


def collect_traces(weights, cfg, n_prompts: int, prompt_len: int, seed: int = 777) -> Tuple[torch.Tensor, torch.Tensor]:
    """u [n_moe, N, H] fp32 and sel [n_moe, N, k] int64 (CPU tensors), N = n_prompts * prompt_len tokens of seeded random
    prompts (generator seed `seed` + prompt index: not the bench's prompt/decode streams, which use cfg.seed + 1 / + 2)."""
    s = weights.shape
    flags = B.F_PREEMPT | B.F_REORDER | B.F_WARM | B.F_TRACE | B.F_TRACE_U | (B.F_TENSOR if s.wdtype >= 1 else 0)
    eng = ProMoE(weights, cache_slots=cfg.cache_slots, stride=cfg.stride, predictor_mode=B.PRED_NONE, flags=flags)
    us, sels = [], []
    try:
        Lm, k, H = eng.n_moe, s.top_k, s.hidden
        for i in range(n_prompts):
            g = torch.Generator().manual_seed(seed + i)
            ids = torch.randint(0, s.vocab, (prompt_len,), generator=g, dtype=torch.int32).numpy()
            eng.reset()
            eng.prefill(ids, want_logits=False)
            us.append(torch.from_numpy(B.promoe_get_trace(eng.h, B.TRACE_U, np.float32).reshape(Lm, prompt_len, H)))
            sels.append(torch.from_numpy(B.promoe_get_trace(eng.h, B.TRACE_SEL, np.int32).reshape(Lm, prompt_len, k)).long())
    finally:
        eng.close()
    return torch.cat(us, 1), torch.cat(sels, 1)


def _round_like_model(w: torch.Tensor, wdtype: int) -> torch.Tensor:
    return w.to(torch.bfloat16).to(torch.float32) if wdtype == 1 else w


def topk_accuracy(u: torch.Tensor, w1: torch.Tensor, w2: torch.Tensor, target: torch.Tensor, k: int) -> float:
    """mean |top-k(W2·ReLU(W1·u)) ∩ target| / k;  target [N, E] 0/1."""
    p = torch.relu(u @ w1.T) @ w2.T
    top = p.topk(k, dim=1).indices
    return float(target.gather(1, top).sum(1).mean().item() / k)


def fit_layer(u: torch.Tensor, sel: torch.Tensor, w1_0: torch.Tensor, w2_0: torch.Tensor, E: int, k: int, wdtype: int,
              seed: int, steps: int = 240, lr: float = 2e-4, n_test_tail: int = 0) -> Dict:
    """One MLP: u [N, H] fp32, sel [N, k] (targets), start weights (skip construction).  Returns the chosen weights
    (fp32, already rounded to the model's dtype) and the accuracies on the 9:1 split.
    n_test_tail > 0: the LAST n_test_tail rows (whole held-out prompts) are the test split — tokens of one prompt share
    their attention context, so a random split over tokens leaks it and flatters the fitted MLP (measured: 0.69 on a
    token split against 0.58 on the decode stream of another prompt); 0: a random 9:1 split over rows."""
    dev = u.device
    N = u.shape[0]
    g = torch.Generator().manual_seed(seed)
    if n_test_tail > 0:
        n_tr = N - n_test_tail
        tr, te = torch.arange(n_tr, device=dev), torch.arange(n_tr, N, device=dev)
    else:
        perm = torch.randperm(N, generator=g).to(dev)
        n_tr = (N * 9) // 10
        tr, te = perm[:n_tr], perm[n_tr:]
    tgt = torch.zeros(N, E, device=dev)
    tgt.scatter_(1, sel, 1.0)
    w1_0, w2_0 = w1_0.float().to(dev), w2_0.float().to(dev)
    acc_skip_te = topk_accuracy(u[te], w1_0, w2_0, tgt[te], k)
    acc_skip_tr = topk_accuracy(u[tr], w1_0, w2_0, tgt[tr], k)
    # free hidden units (all-zero rows of the start point) begin as small random features
    free = (w1_0.abs().sum(1) == 0)
    w1 = w1_0.clone()
    w1[free] = torch.randn(int(free.sum()), w1.shape[1], generator=g).to(dev) * (w1.shape[1] ** -0.5)
    w2 = w2_0.clone()
    w1.requires_grad_(True); w2.requires_grad_(True)
    opt = torch.optim.Adam([w1, w2], lr=lr, weight_decay=0.0)
    best = {"acc": -1.0}
    bs = min(4096, n_tr)
    for it in range(steps):
        idx = tr[torch.randint(0, n_tr, (bs,), generator=g).to(dev)]
        p = torch.relu(u[idx] @ w1.T) @ w2.T
        loss = -(torch.log_softmax(p, dim=1) * tgt[idx]).sum(1).mean() / k
        opt.zero_grad(set_to_none=True)
        loss.backward()
        opt.step()
        if (it + 1) in (5, 10, 20) or (it + 1) % 40 == 0 or it + 1 == steps:
            with torch.no_grad():
                r1, r2 = _round_like_model(w1.detach(), wdtype), _round_like_model(w2.detach(), wdtype)
                a = topk_accuracy(u[te], r1, r2, tgt[te], k)
                if a > best["acc"]:
                    best = {"acc": a, "w1": r1.clone(), "w2": r2.clone(), "step": it + 1, "loss": float(loss.item())}
    with torch.no_grad():
        acc_fit_tr = topk_accuracy(u[tr], best["w1"], best["w2"], tgt[tr], k)
    use_fit = best["acc"] > acc_skip_te
    return {"w1": best["w1"] if use_fit else _round_like_model(w1_0, wdtype), "w2": best["w2"] if use_fit else _round_like_model(w2_0, wdtype),
            "kept": "fitted" if use_fit else "skip", "acc_test_fitted": best["acc"], "acc_test_skip": acc_skip_te,
            "acc_train_fitted": acc_fit_tr, "acc_train_skip": acc_skip_tr, "best_step": best["step"], "n_train": n_tr, "n_test": N - n_tr}


def fit_predictor(weights, cfg, stride: int, n_prompts: int = 20, prompt_len: int = 0, steps: int = 240, seed: int = 777,
                  traces=None) -> Dict:
    """Replace weights.dense['l*.pred_w1' / 'l*.pred_w2'] (which must hold the `skip` construction for `stride`) by the
    fitted MLPs, in place.  Returns the report (per layer and mean accuracies on the 9:1 split, timings)."""
    s = weights.shape
    if weights.predictor != "skip" or weights.stride != stride:
        raise ValueError("fit_predictor starts from synth.make_weights(cfg with this stride, predictor='skip')")
    t0 = time.perf_counter()
    pl = prompt_len or min(cfg.prompt_len, s.max_seq)
    u, sel = traces if traces is not None else collect_traces(weights, cfg, n_prompts, pl, seed)
    t1 = time.perf_counter()
    dev = torch.device("cuda") if torch.cuda.is_available() else torch.device("cpu")
    moe_ids = list(range(s.n_dense_layers, s.n_layers))
    Lm = len(moe_ids)
    dt = torch.float32 if s.wdtype == 0 else torch.bfloat16
    n_test = max(1, round(n_prompts / 10))       # 9:1 by PROMPT: the last prompts are held out whole
    layers = []
    for m in range(Lm - stride):
        l = moe_ids[m]
        r = fit_layer(u[m].to(dev), sel[m + stride].to(dev), weights.dense[f"l{l}.pred_w1"], weights.dense[f"l{l}.pred_w2"],
                      s.n_experts, s.top_k, min(s.wdtype, 1), seed + 1000 + m, steps, n_test_tail=n_test * pl)
        weights.dense[f"l{l}.pred_w1"] = r.pop("w1").to(dt).cpu().contiguous()
        weights.dense[f"l{l}.pred_w2"] = r.pop("w2").to(dt).cpu().contiguous()
        r["moe_layer"] = m
        layers.append(r)
    weights.predictor = "fitted"
    t2 = time.perf_counter()
    mean = lambda key: float(np.mean([r[key] for r in layers])) if layers else 0.0
    return {"stride": stride, "tokens": int(u.shape[1]), "prompts": n_prompts, "prompt_len": pl,
            "split": f"9:1 by prompt ({n_prompts - n_test} train / {n_test} held-out prompts)",
            "acc_test_fitted": mean("acc_test_fitted"), "acc_test_skip": mean("acc_test_skip"),
            "acc_train_fitted": mean("acc_train_fitted"), "acc_train_skip": mean("acc_train_skip"),
            "layers_kept_fitted": sum(r["kept"] == "fitted" for r in layers), "layers": len(layers),
            "collect_s": t1 - t0, "train_s": t2 - t1, "per_layer": layers}


def main():
    import synth
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", default="c2")
    ap.add_argument("--stride", type=int, default=0)
    ap.add_argument("--prompts", type=int, default=20)
    ap.add_argument("--steps", type=int, default=240)
    a = ap.parse_args()
    cfg = synth.get_config(a.config)
    if a.stride:
        cfg = replace(cfg, stride=a.stride)
    w = synth.make_weights(cfg, predictor="skip")
    rep = fit_predictor(w, cfg, cfg.stride, a.prompts, steps=a.steps)
    rep.pop("per_layer")
    print(json.dumps(rep))


if __name__ == "__main__":
    main()
