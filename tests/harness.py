"""Side-by-side driver: the CUDA path (through the C-ABI binding) against the CPU oracle on the same seeded inputs.

Used by the `-m gpu` parity tests, `__graft_entry__.smoke()` and nothing in the product.  Decode is teacher-forced
with the ORACLE's greedy tokens (P1), or with seeded random ids.
"""
from __future__ import annotations

from typing import Dict, List, Optional

import numpy as np

from oracle.cache_sim import ProMoECacheSim
from oracle.compare import ParityReport, compare_cache, compare_stats, compare_step, oracle_step_matching
from oracle.forward import OracleModel


def run_parity(cfg, weights, prompt, decode_steps: int, *, cache_slots: Optional[int] = None,
               stride: Optional[int] = None, chunk_bytes: int = 0, predictor_mode: int = 1, flags: Optional[int] = None,
               decode_ids: Optional[List[int]] = None, max_inflight: int = 0, warm: bool = True, high_group: int = 0,
               max_spec_decode: int = 0, max_spec_prefill: int = 0, static_slots: int = 0) -> Dict:
    from paper_2410_22134_b200 import binding as B
    from paper_2410_22134_b200.engine import ProMoE

    s = cfg.shape
    cache_slots = cfg.cache_slots if cache_slots is None else cache_slots
    stride = cfg.stride if stride is None else stride
    if flags is None:
        flags = B.F_PREEMPT | B.F_REORDER | B.F_TRACE | (B.F_WARM if warm else 0)
    n_moe = s.n_layers - s.n_dense_layers
    C = cache_slots // n_moe
    eng = ProMoE(weights, cache_slots=cache_slots, stride=stride, chunk_bytes=chunk_bytes,
                 predictor_mode=predictor_mode, flags=flags, max_inflight=max_inflight, high_group=high_group,
                 max_spec_decode=max_spec_decode, max_spec_prefill=max_spec_prefill, static_slots=static_slots)
    use_pred = predictor_mode == B.PRED_MLP
    ora = OracleModel(weights, stride=stride, slots_per_layer=C, use_predictor=use_pred)
    sim = ProMoECacheSim(n_moe, s.n_experts, C, warm=bool(flags & B.F_WARM), reorder=bool(flags & B.F_REORDER),
                         demote=bool(flags & B.F_DEMOTE), static_slots=static_slots)
    rep = ParityReport()
    # library defaults (include/promoe.h): decode top_k allocations per push, prefill none
    ms_dec = s.top_k if max_spec_decode == 0 else max(0, max_spec_decode)
    ms_pre = max(0, max_spec_prefill)
    all_logits = []
    try:
        ids = [int(x) for x in prompt]
        T = len(ids)
        logits = eng.prefill(ids)
        tr = eng.trace(T)
        st = oracle_step_matching(ora, ids, tr["sel"], rep)
        compare_step(tr, st, s.n_experts, rep, gpu_logits=logits, check_pred=use_pred, pred_cap=C)
        compare_cache(sim, tr, stride, use_pred, ms_pre)
        all_logits.append(logits)
        nxt = st.next_token
        for i in range(decode_steps):
            tok = int(decode_ids[i]) if decode_ids is not None else nxt
            logits = eng.decode(tok)
            tr = eng.trace(1)
            st = oracle_step_matching(ora, [tok], tr["sel"], rep)
            compare_step(tr, st, s.n_experts, rep, gpu_logits=logits, check_pred=use_pred, pred_cap=C)
            compare_cache(sim, tr, stride, use_pred, ms_dec)
            all_logits.append(logits)
            nxt = st.next_token
        stats = eng.stats()
        compare_stats(sim, stats)
        for m in range(n_moe):
            assert eng.slots(m).tolist() == sim.slot_expert[m], f"final slot table of layer {m} differs"
    finally:
        eng.close()
    return {"report": rep, "stats": stats, "logits": all_logits, "sim": sim}


def run_gpu_only(cfg, weights, prompt, decode_ids, **kw) -> Dict:
    """GPU-only run (no oracle): logits per step + stats, for the bitwise-invariance tests (P5)."""
    from paper_2410_22134_b200 import binding as B
    from paper_2410_22134_b200.engine import ProMoE

    flags = kw.pop("flags", B.F_PREEMPT | B.F_REORDER | B.F_WARM | B.F_TRACE)
    eng = ProMoE(weights, cache_slots=kw.pop("cache_slots", cfg.cache_slots), stride=kw.pop("stride", cfg.stride),
                 flags=flags, **kw)
    try:
        out = [eng.prefill([int(x) for x in prompt])]
        for t in decode_ids:
            out.append(eng.decode(int(t)))
        stats = eng.stats()
    finally:
        eng.close()
    return {"logits": out, "stats": stats}


def run_parity_batch(cfg, weights, prompts, decode_ids, *, cache_slots: Optional[int] = None, stride: Optional[int] = None,
                     predictor_mode: int = 1, flags: Optional[int] = None, max_spec_decode: int = 0, chunk_bytes: int = 0) -> Dict:
    """Batched decode: len(prompts) sequences are prefilled one by one (ordinary single-sequence steps), then
    every entry of decode_ids ([steps][B]) is ONE promoe_decode_batch call over all of them, compared with oracle/batch.py:
    rows = sequences, needed = union, predictions = votes; cache traces against O3 driven with the GPU's lists."""
    from oracle.batch import OracleBatch
    from paper_2410_22134_b200 import binding as B
    from paper_2410_22134_b200.engine import ProMoE

    s = cfg.shape
    nb = len(prompts)
    cache_slots = cfg.cache_slots if cache_slots is None else cache_slots
    stride = cfg.stride if stride is None else stride
    if flags is None:
        flags = B.F_PREEMPT | B.F_REORDER | B.F_TRACE | B.F_WARM
    n_moe = s.n_layers - s.n_dense_layers
    C = cache_slots // n_moe
    eng = ProMoE(weights, cache_slots=cache_slots, stride=stride, chunk_bytes=chunk_bytes, predictor_mode=predictor_mode,
                 flags=flags, max_spec_decode=max_spec_decode, max_batch=nb)
    use_pred = predictor_mode == B.PRED_MLP
    ora = OracleBatch(weights, nb, stride=stride, slots_per_layer=C, use_predictor=use_pred)
    sim = ProMoECacheSim(n_moe, s.n_experts, C, warm=bool(flags & B.F_WARM), reorder=bool(flags & B.F_REORDER),
                         demote=bool(flags & B.F_DEMOTE))
    rep = ParityReport()
    ms_dec = s.top_k if max_spec_decode == 0 else max(0, max_spec_decode)
    try:
        for b, pr in enumerate(prompts):
            ids = [int(x) for x in pr]
            logits = eng.prefill_seq(b, ids)
            tr = eng.trace(len(ids))
            st = oracle_step_matching(ora.seqs[b], ids, tr["sel"], rep)
            compare_step(tr, st, s.n_experts, rep, gpu_logits=logits, check_pred=use_pred, pred_cap=C)
            compare_cache(sim, tr, stride, use_pred, 0 if len(ids) > 1 else ms_dec)
        for toks in decode_ids:
            toks = [int(t) for t in toks]
            logits = eng.decode_batch(list(range(nb)), toks)
            tr = eng.trace(nb)
            st = oracle_step_matching(ora, toks, tr["sel"], rep)
            compare_step(tr, st, s.n_experts, rep, gpu_logits=logits[-1], check_pred=use_pred, pred_cap=C)
            for b in range(nb):          # every row's logits against its own sequence
                lo = st.seq_logits[b].numpy()
                g1 = int(np.flatnonzero(logits[b] == logits[b].max())[0])
                if g1 != st.seq_next[b]:
                    srt = np.sort(lo)
                    assert srt[-1] - srt[-2] < 1e-3, f"row {b}: logits top-1 differs"
                rep.max_logit_err = max(rep.max_logit_err, float(np.abs(logits[b] - lo).max()))
            compare_cache(sim, tr, stride, use_pred, ms_dec)
        stats = eng.stats()
        compare_stats(sim, stats)
        for m in range(n_moe):
            assert eng.slots(m).tolist() == sim.slot_expert[m], f"final slot table of layer {m} differs"
    finally:
        eng.close()
    return {"report": rep, "stats": stats, "sim": sim}
