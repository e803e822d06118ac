#!/usr/bin/env python
"""bench.py — ProMoE hot path on B200: prefill & decode tokens/s at a fixed expert-cache budget, % of roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config c2]

A "step" is ONE REQUEST of the workload BASELINE.json's metric is quoted on (configs[1]: Qwen1.5-MoE-A2.7B-shaped
decoder, 50 % expert cache, stride-2 predictor): promoe_reset → promoe_prefill(512 seeded random ids) → 128 ×
promoe_decode, i.e. one pass of the whole hot path (all SURVEY §8(a) rows) through the C-ABI.  Routed experts
(24.9 GB) live in pinned host memory, so every step moves its missing experts host→device (L2 is irrelevant: each
request streams ≫ 126 MB of weights).  `value` = decode tokens/s from the library's CUDA events (device time of
the step); `e2e` = the same requests by host wall clock around the C-ABI calls with HOST buffers (ids in, logits
out, experts copied inside).  Multi-GPU: replicas only — every rank serves its own request stream,
no data-path collective, "scaling": "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


# ---------------------------------------------------------------------------------------------------------------
def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "bf16_tflops": d["bf16_tflops"], "bf16_tflops_sustained":
                d.get("bf16_tflops_sustained", d["bf16_tflops"]), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        self.proc.terminate()
        self.t.join(timeout=2)
        sm = sorted(int(r[0]) for r in self.rows if r and r[0].isdigit())
        mx = [int(r[1]) for r in self.rows if len(r) > 1 and r[1].isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 2 + i and r[2 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(sm)}


# ---- algorithmic work of one step -----------------------------
def expert_image_bytes(s) -> int:
    """Bytes of one routed expert image (what a slot fill moves): 3·H·I weights at 4 / 2 bytes, or INT4 codes + one
    bf16 scale per 128 (wdtype 2, G18)."""
    n = 3 * s.hidden * s.expert_inter
    return n // 2 + n // 128 * 2 if s.wdtype == 2 else n * (4 if s.wdtype == 0 else 2)


def dense_bytes_per_token(s) -> int:
    """Always-resident weight bytes one decode step streams from HBM (each touched once)."""
    wb = 4 if s.wdtype == 0 else 2
    qkv = (s.n_q_heads + 2 * s.n_kv_heads) * s.head_dim * s.hidden
    wo = s.hidden * s.n_q_heads * s.head_dim
    per_moe = s.n_experts * s.hidden + s.pred_hidden * s.hidden + s.n_experts * s.pred_hidden \
        + 3 * s.hidden * s.n_shared_inter + (s.hidden if s.shared_gate else 0)
    n_moe = s.n_layers - s.n_dense_layers
    total = s.n_layers * (qkv + wo) + n_moe * per_moe + s.n_dense_layers * 3 * s.hidden * s.dense_inter \
        + s.vocab * s.hidden + s.hidden      # lm_head + one embedding row
    return total * wb


def step_work(s, T: int, pos0: int, distinct_experts: int, need_experts: int):
    """(B_hbm, FLOPs) of one step with T tokens starting at position pos0.  distinct_experts = Σ_layers |needed|,
    need_experts = those not resident at step start (their bytes are also WRITTEN into the slot region)."""
    wb = 4 if s.wdtype == 0 else 2
    Be = expert_image_bytes(s)
    n_moe = s.n_layers - s.n_dense_layers
    kv_read = sum(2 * s.n_layers * s.n_kv_heads * s.head_dim * 4 * (pos0 + t + 1) for t in range(T)) if T == 1 else \
        2 * s.n_layers * s.n_kv_heads * s.head_dim * 4 * (pos0 + T)
    kv_write = 2 * s.n_layers * s.n_kv_heads * s.head_dim * 4 * T
    lm = s.vocab * s.hidden * wb
    b_hbm = dense_bytes_per_token(s) + distinct_experts * Be + need_experts * Be + kv_read + kv_write
    elems_per_tok = (dense_bytes_per_token(s) - lm) // wb + n_moe * s.top_k * 3 * s.hidden * s.expert_inter
    attn = sum(4 * (pos0 + t + 1) * s.n_q_heads * s.head_dim for t in range(T)) * s.n_layers
    flops = 2 * elems_per_tok * T + 2 * s.vocab * s.hidden + attn
    return b_hbm, flops


def roofline_time(b_need, b_hbm, flops, h2d_gbs, hbm_gbs, tflops):
    terms = {"h2d": b_need / (h2d_gbs * 1e9), "hbm": b_hbm / (hbm_gbs * 1e9), "tensor": flops / (tflops * 1e12)}
    bound = max(terms, key=terms.get)
    return terms[bound], bound, terms


# ---------------------------------------------------------------------------------------------------------------
def oracle_sample(cfg, weights, prompt_len: int, decode_steps: int):
    """Time the CPU oracle AS IT STANDS on a bounded sample of the workload (test infrastructure used as the
    reported CPU baseline; never on the product path)."""
    import torch
    import synth
    from oracle.forward import OracleModel
    ora = OracleModel(weights, stride=cfg.stride, slots_per_layer=cfg.slots_per_layer)
    prompt = synth.make_prompt(cfg, prompt_len).tolist()
    t0 = time.perf_counter()
    st = ora.forward(prompt)
    t1 = time.perf_counter()
    tok = st.next_token
    for _ in range(decode_steps):
        tok = ora.decode(tok).next_token
    t2 = time.perf_counter()
    return {"prefill_tok_s": prompt_len / (t1 - t0), "decode_tok_s": decode_steps / (t2 - t1),
            "cores": torch.get_num_threads(), "seconds": t2 - t0}


def run_reference(args, cfg, rank):
    """--impl reference: this tier's reference arm is the oracle on the host cores (rank 0 only)."""
    if rank != 0:
        return
    import synth
    weights = synth.make_weights(cfg, predictor="skip")
    pl, ds = ref_sample(args, cfg)
    for _ in range(args.warmup):          # warm-up of a CPU program: page in the weights, start the thread pool
        oracle_sample(cfg, weights, min(pl, 32), 1)
    t0 = time.perf_counter()
    dec, pre, cores = [], [], 0
    for _ in range(args.steps):
        r = oracle_sample(cfg, weights, pl, ds)
        dec.append(r["decode_tok_s"]); pre.append(r["prefill_tok_s"]); cores = r["cores"]
    dt = time.perf_counter() - t0
    v = len(dec) / sum(1.0 / x for x in dec)
    sample = ref_sample_text(cfg, pl, ds)
    conf = workload_config(cfg, args)
    conf["reference_sample"] = {"prompt_tokens": pl, "decode_tokens": ds, "decode_positions": [pl, pl + ds - 1],
                                "of_prompt": cfg.prompt_len, "of_decode": cfg.decode_steps}
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": "tokens/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": conf, "prefill_tokens_per_s": len(pre) / sum(1.0 / x for x in pre),
            "cpu_baseline": {"value": v, "unit": "tokens/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": "tokens/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def ref_sample(args, cfg):
    """Bounded oracle sample at the GPU arm's own token positions: the whole prompt when it is at most 512 tokens (so
    that the decode tokens sit at the positions the GPU arm decodes at), then a few decode tokens."""
    pl = args.ref_prompt if args.ref_prompt > 0 else min(cfg.prompt_len, 512)
    return pl, args.ref_decode


def ref_sample_text(cfg, pl, ds):
    same = "the GPU arm's positions" if pl == cfg.prompt_len else f"SHORTER than the GPU arm's prompt of {cfg.prompt_len}"
    return (f"per step: prefill {pl} tokens ({same}) + {ds} decode tokens at positions {pl}..{pl + ds - 1} of {cfg.name} "
            f"(GPU arm: {cfg.prompt_len} + {cfg.decode_steps})")


METRIC = "decode tokens/s at fixed expert-cache budget (prefill tokens/s and % of per-step roofline alongside)"


def workload_config(cfg, args):
    s = cfg.shape
    return {"workload": f"{cfg.name}: BASELINE.json configs[{ {'c1': 0, 'c2': 1, 'c3': 2, 'c4': 3}.get(cfg.name, '?') }] "
                        f"{s.n_layers}L H{s.hidden} E{s.n_experts} top{s.top_k} I{s.expert_inter}, batch 1, "
                        f"prompt {cfg.prompt_len} + {cfg.decode_steps} decode",
            "cache_slots": cfg.cache_slots, "cache_fraction": cfg.slots_per_layer / s.n_experts, "stride": cfg.stride,
            "predictor": args.predictor, "decode_ids": args.decode, "chunk_bytes": args.chunk_kb << 10, "max_spec_decode": args.max_spec_decode,
            "max_spec_prefill": args.max_spec_prefill, "low_cap_chunks": args.low_cap, "max_inflight": args.inflight, "fetch_ctas": args.fetch_ctas, "demote": args.demote, "int4_experts": args.int4,
            "l2": "inputs larger than L2 (each request streams >> 126 MB of expert weights)"}


def shard_requests(n_requests_per_rank: int, world: int):
    """Replicas only: every rank serves n requests of the same shape (weak scaling); no data-path collective."""
    return [n_requests_per_rank] * world


def aggregate(local_tokens: float, local_seconds: float, dist=None):
    """Whole-job throughput = tokens of all ranks ÷ max-over-ranks device time."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local_tokens, local_seconds
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    tok = torch.tensor([local_tokens], dtype=torch.float64, device=dev)
    sec = torch.tensor([local_seconds], dtype=torch.float64, device=dev)
    dist.all_reduce(tok, op=dist.ReduceOp.SUM)
    dist.all_reduce(sec, op=dist.ReduceOp.MAX)
    return float(tok.item()), float(sec.item())


def run_request(eng, cfg, prompt, decode_ids, greedy: bool, record=None, inject=None):
    """reset → prefill → decode_steps × decode.  Returns per-phase device ms, wall s, stats deltas.
    record: list that receives, per step, the needed experts of every MoE layer (from the library's routing trace);
    inject: such a list from an earlier pass — step t's predictor at layer m is given the TRUE needed set of layer
    m+stride (oracle-routing predictor, the upper bound of BASELINE.json configs[4]); routing does not depend on
    the cache, so a reactive pass and the injected pass see the same selections."""
    import numpy as np
    eng.reset()
    Lm, k = eng.n_moe, eng.s.top_k

    def needed_of_last_step(T):
        from paper_2410_22134_b200 import binding as B
        sel = B.promoe_get_trace(eng.h, B.TRACE_SEL, np.int32).reshape(Lm, T * k)
        return [sorted(set(int(e) for e in row)) for row in sel]

    def inject_step(t):
        need, st = inject[t], eng.stride
        eng.set_prediction_trace([need[m + st][:eng.slots_per_layer] if m + st < Lm else None for m in range(Lm)])

    s0 = eng.stats()
    if inject is not None:
        inject_step(0)
    w0 = time.perf_counter()
    logits = eng.prefill(prompt)
    w1 = time.perf_counter()
    s1 = eng.stats()
    if record is not None:
        record.append(needed_of_last_step(len(prompt)))
    tok = int(np.argmax(logits))
    dec_ms = []
    for i in range(cfg.decode_steps):
        if not greedy:
            tok = int(decode_ids[i])
        if inject is not None:
            inject_step(1 + i)
        logits = eng.decode(tok)
        if record is not None:
            record.append(needed_of_last_step(1))
        dec_ms.append(eng.stats()["last_step_ms"])
        if greedy:
            tok = int(np.argmax(logits))
    w2 = time.perf_counter()
    s2 = eng.stats()
    d = lambda a, b, k: b[k] - a[k]
    return {"prefill_ms": s1["step_ms"] - s0["step_ms"], "decode_ms": s2["step_ms"] - s1["step_ms"],
            "prefill_wall": w1 - w0, "decode_wall": w2 - w1, "dec_ms": dec_ms,
            "pre": {k: d(s0, s1, k) for k in s0}, "dec": {k: d(s1, s2, k) for k in s1}}


def also_config(args, name, h2d_gbs, flags, local):
    """One request of another BASELINE.json config (after one warm-up request): ProMoE with the run's settings and the reactive
    cache, decode / prefill tokens/s and the H2D roofline fractions (every bf16 config is H2D-bound)."""
    import synth
    from paper_2410_22134_b200 import binding as B
    from paper_2410_22134_b200.engine import ProMoE
    cfg = synth.get_config(name)
    s = cfg.shape
    Be = expert_image_bytes(s)
    w = synth.make_weights(cfg, predictor="skip")
    prompt = synth.make_prompt(cfg).tolist()
    decode_ids = synth.make_decode_ids(cfg).tolist()
    out = {"workload": f"{name}: prompt {cfg.prompt_len} + {cfg.decode_steps} decode, cache {cfg.slots_per_layer}/{s.n_experts} per layer, stride {cfg.stride}"}
    need_reactive = None
    for label, pm in (("reactive_no_prefetch", B.PRED_NONE), ("promoe", B.PRED_MLP)):
        eng = ProMoE(w, cache_slots=cfg.cache_slots, stride=cfg.stride, chunk_bytes=args.chunk_kb << 10, predictor_mode=pm, flags=flags,
                     max_inflight=args.inflight, max_spec_decode=args.max_spec_decode, max_spec_prefill=args.max_spec_prefill,
                     fetch_ctas=args.fetch_ctas, device=f"cuda:{local}")
        run_request(eng, cfg, prompt, decode_ids, False)
        r = run_request(eng, cfg, prompt, decode_ids, False)
        eng.close()
        dec_s, pre_s = r["decode_ms"] / 1e3, r["prefill_ms"] / 1e3
        need_d, need_p = r["dec"]["need_experts"] * Be, r["pre"]["need_experts"] * Be
        if pm == B.PRED_NONE:
            need_reactive = (need_d, need_p)
        out[label] = {"decode_tokens_per_s": cfg.decode_steps / dec_s, "prefill_tokens_per_s": cfg.prompt_len / pre_s,
                      "decode_roofline_frac": need_d / (h2d_gbs * 1e9) / dec_s, "prefill_roofline_frac": need_p / (h2d_gbs * 1e9) / pre_s,
                      "decode_frac_vs_reactive_need": need_reactive[0] / (h2d_gbs * 1e9) / dec_s,
                      "prefill_frac_vs_reactive_need": need_reactive[1] / (h2d_gbs * 1e9) / pre_s,
                      "hit_rate": (r["dec"]["hits_resident"] + r["dec"]["hits_prefetch"]) / max(1, r["dec"]["accesses"]),
                      "predictor_accuracy": r["dec"]["predicted_correct"] / max(1, r["dec"]["predicted"])}
    return out


def replica_weights(cfg, pred_kind, local, world, dist, tag=None):
    """Weights of one replica.  world > 1: the replicas of a node share ONE host copy of the routed experts — a /dev/shm
    mapping drawn by local rank 0 and mapped by the others (every rank's library registers it with cudaHostRegister);
    8 private pinned copies of 25-90 GB would not fit the host."""
    import torch
    import synth
    if world <= 1:
        return synth.make_weights(cfg, predictor=pred_kind)
    s = cfg.shape
    n_moe = s.n_layers - s.n_dense_layers
    per = expert_image_bytes(s) if s.wdtype == 2 else 3 * s.hidden * s.expert_inter
    dt = {0: torch.float32, 1: torch.bfloat16, 2: torch.uint8}[s.wdtype]
    path = f"/dev/shm/promoe_experts_{tag or os.environ.get('MASTER_PORT', '0')}_{cfg.name}"
    if local == 0:
        buf = torch.from_file(path, shared=True, size=n_moe * s.n_experts * per, dtype=dt).view(n_moe, s.n_experts, per)
        weights = synth.make_weights(cfg, predictor=pred_kind, experts_buf=buf, fill_experts=True)
    dist.barrier()
    if local != 0:
        buf = torch.from_file(path, shared=True, size=n_moe * s.n_experts * per, dtype=dt).view(n_moe, s.n_experts, per)
        weights = synth.make_weights(cfg, predictor=pred_kind, experts_buf=buf, fill_experts=False)
    dist.barrier()
    if local == 0:
        os.unlink(path)          # the mappings keep the memory alive until the processes exit
    return weights


def run_ours(args, cfg, rank, world, dist):
    import numpy as np
    import torch
    import synth
    from paper_2410_22134_b200 import binding as B
    from paper_2410_22134_b200.engine import ProMoE

    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    peaks = load_peaks()
    s = cfg.shape
    pred_kind = "skip" if args.predictor in ("none", "trace", "fitted") else args.predictor
    weights = replica_weights(cfg, pred_kind, local, world, dist)
    Be = expert_image_bytes(s)
    h2d_gbs = B.promoe_bench_h2d(256 << 20, 2, 5)
    prompt = synth.make_prompt(cfg).tolist()
    decode_ids = synth.make_decode_ids(cfg).tolist()
    greedy = args.decode == "greedy"
    flags = B.F_PREEMPT | B.F_REORDER | B.F_WARM | (B.F_TENSOR if args.tensor else 0) | (B.F_DEMOTE if args.demote else 0)
    fit_report = None
    if args.predictor == "fitted":     # N1: the offline step of §4.3 on the model's own traces, before any timing
        from paper_2410_22134_b200.fit_predictor import fit_predictor
        fit_report = fit_predictor(weights, cfg, cfg.stride, n_prompts=args.fit_prompts, steps=args.fit_steps)
        fit_report.pop("per_layer")
    inject = None
    if args.predictor == "trace":      # pass 0: reactive run that records the routing of every step
        rec_eng = ProMoE(weights, cache_slots=cfg.cache_slots, stride=cfg.stride, predictor_mode=B.PRED_NONE,
                         flags=flags | B.F_TRACE, device=f"cuda:{local}")
        inject = []
        run_request(rec_eng, cfg, prompt, decode_ids, greedy, record=inject)
        rec_eng.close()
    pmode = {"none": B.PRED_NONE, "trace": B.PRED_TRACE}.get(args.predictor, B.PRED_MLP)
    eng = ProMoE(weights, cache_slots=cfg.cache_slots, stride=cfg.stride, chunk_bytes=args.chunk_kb << 10,
                 predictor_mode=pmode, flags=flags,
                 max_inflight=args.inflight, max_spec_decode=args.max_spec_decode, max_spec_prefill=args.max_spec_prefill,
                 low_cap_chunks=args.low_cap, fetch_ctas=args.fetch_ctas, device=f"cuda:{local}")
    for _ in range(args.warmup):
        run_request(eng, cfg, prompt, decode_ids, greedy, inject=inject)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    clocks = ClockSampler(local)
    clocks.start()
    launches0 = eng.stats()["kernel_launches"]
    t0 = time.perf_counter()
    reqs = [run_request(eng, cfg, prompt, decode_ids, greedy, inject=inject) for _ in range(args.steps)]
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    wall = time.perf_counter() - t0
    launches = eng.stats()["kernel_launches"] - launches0
    clk = clocks.stop()

    K = args.steps
    dec_tokens, pre_tokens = K * cfg.decode_steps, K * cfg.prompt_len
    dec_s = sum(r["decode_ms"] for r in reqs) / 1e3
    pre_s = sum(r["prefill_ms"] for r in reqs) / 1e3
    g_dec_tok, g_dec_s = aggregate(dec_tokens, dec_s, dist)
    g_pre_tok, g_pre_s = aggregate(pre_tokens, pre_s, dist)
    g_dec_wtok, g_dec_wall = aggregate(dec_tokens, sum(r["decode_wall"] for r in reqs), dist)
    g_pre_wtok, g_pre_wall = aggregate(pre_tokens, sum(r["prefill_wall"] for r in reqs), dist)

    # ---- per-step roofline (north_star): max(B_need / H2D, B_hbm / HBM, F / bf16 peak), summed over the steps
    def phase_roof(key, T_of_step, n_steps, pos_start):
        b_need = sum(r[key]["need_experts"] for r in reqs) * Be
        b_hbm = fl = 0.0
        for r in reqs:
            acc, need = r[key]["accesses"], r[key]["need_experts"]
            for i in range(n_steps):
                bh, f = step_work(s, T_of_step, pos_start + i, acc / n_steps, need / n_steps)
                b_hbm += bh; fl += f
        t, bound, terms = roofline_time(b_need, b_hbm, fl, h2d_gbs, peaks["hbm_gbs"], peaks["bf16_tflops_sustained"])
        t8, _, _ = roofline_time(b_need, b_hbm, fl, h2d_gbs, 8000.0, peaks["bf16_tflops_sustained"])
        return {"bound": bound, "t_roof_s": t, "terms_s": terms, "b_need_bytes": b_need, "b_hbm_bytes": b_hbm,
                "flops": fl, "t_roof_s_at_8TBs": t8}
    roof_dec = phase_roof("dec", 1, cfg.decode_steps, cfg.prompt_len)
    roof_pre = phase_roof("pre", cfg.prompt_len, 1, 0)
    roof_dec["frac"] = roof_dec["t_roof_s"] / dec_s
    roof_pre["frac"] = roof_pre["t_roof_s"] / pre_s
    # `frac` takes B_need from THIS run's cache state, which a prefetching run pollutes with its own mispredictions;
    # `frac_vs_reactive_need` (filled in below from the reactive pass over the same routing) uses the B_need of a plain
    # LRU cache — a function of routing and budget only (re-fetches caused by pollution are overhead)
    roof_dec["frac_vs_reactive_need"] = roof_pre["frac_vs_reactive_need"] = None

    def cache_stats(key):
        a = {k: sum(r[key][k] for r in reqs) for k in reqs[0][key]}
        acc = max(1, a["accesses"])
        return {"hit_rate": (a["hits_resident"] + a["hits_prefetch"]) / acc, "hit_rate_resident": a["hits_resident"] / acc,
                # byte-accurate: class A / B accesses whose whole image had landed when the gate was processed (a logical hit on a
                # partially fetched image still owes bytes: `owed_bytes_per_access`)
                "hit_rate_landed": a["hits_landed"] / acc, "owed_bytes_per_access": a["owed_bytes_at_gate"] / acc,
                "miss_rate": a["misses"] / acc,
                "predictor_accuracy": a["predicted_correct"] / max(1, a["predicted"]),
                "fetch_rate": a["fetched_at_gate"] / max(1, a["fetched_at_gate_of"]),
                # partial-fetch form: chunks of the class-B images that had landed at their gate / chunks per image
                "fetch_rate_chunks": a["landed_chunks_at_gate"] / max(1, a["landed_chunks_of"]),
                "good_pred": a["predicted_correct"] / max(1, a["predicted"]) * a["fetched_at_gate"] / max(1, a["fetched_at_gate_of"]),
                "good_pred_chunks": a["predicted_correct"] / max(1, a["predicted"]) * a["landed_chunks_at_gate"] / max(1, a["landed_chunks_of"]),
                "pred_allocs": a["pred_allocs"], "low_bytes": a["low_bytes"], "low_bytes_useful": a["low_bytes_useful"],
                "h2d_bytes_moved": a["h2d_bytes"], "h2d_bytes_needed": a["need_experts"] * Be,
                "byte_efficiency": a["need_experts"] * Be / max(1, a["h2d_bytes"]),
                "copy_busy_ms": a["copy_busy_ms"], "link_utilisation": a["h2d_bytes"] / 1e6 / max(1e-9, a["copy_busy_ms"]) / h2d_gbs,
                "chunks_cancelled": a["chunks_cancelled"], "timeouts": a["timeouts"]}
    cs_dec, cs_pre = cache_stats("dec"), cache_stats("pre")

    # ---- dominant kernel, timed live with CUDA events on the launching stream (resident slots ≫ L2)
    ms_gu, bytes_gu = B.promoe_bench_kernel_time(eng.h, 0, 300)
    ms_dn, bytes_dn = B.promoe_bench_kernel_time(eng.h, 1, 300)
    ach = bytes_gu / (ms_gu * 1e-3) / 1e9
    kernel_roof = {"kernel": "ffn_gateup_gemv_kernel (A9 decode: gate/up SwiGLU GEMV over top_k resident experts)",
                   "bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": ach / peaks["hbm_gbs"],
                   "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peaks['source']}, burst: kernel timed alone)",
                   "bytes_per_launch": bytes_gu, "avg_launch_us": ms_gu * 1e3, "traffic": None,
                   "down_gemv": {"achieved": bytes_dn / (ms_dn * 1e-3) / 1e9, "avg_launch_us": ms_dn * 1e3,
                                 "bytes_per_launch": bytes_dn}}
    prof = os.path.join(ROOT, "profiles", "traffic.txt")
    if os.path.exists(prof):
        try:
            kernel_roof["traffic"] = json.load(open(prof)).get(cfg.name, {}).get("ffn_gateup_gemv_kernel")
            kernel_roof["traffic_source"] = ("stored constant: dram__bytes_read.sum + dram__bytes_write.sum per launch from the "
                                             "ncu --set full capture named in profiles/README.md (not measured in this run)")
        except Exception:
            pass
    eng.close()

    # ---- compute-only time of the same decode stream (every expert resident): hidden-copy fraction + HBM view
    hidden = None
    allhit = None
    if rank == 0 and not args.no_allhit:
        n_moe = s.n_layers - s.n_dense_layers
        full = ProMoE(weights, cache_slots=n_moe * s.n_experts, stride=cfg.stride, predictor_mode=B.PRED_NONE if args.predictor in ("none", "trace") else B.PRED_MLP,
                      flags=flags, chunk_bytes=args.chunk_kb << 10, device=f"cuda:{local}")
        run_request(full, cfg, prompt, decode_ids, greedy)
        r = run_request(full, cfg, prompt, decode_ids, greedy)
        full.close()
        comp_dec_s = r["decode_ms"] / 1e3
        bh = sum(step_work(s, 1, cfg.prompt_len + i, n_moe * s.top_k, 0)[0] for i in range(cfg.decode_steps))
        allhit = {"decode_tokens_per_s": cfg.decode_steps / comp_dec_s, "prefill_tokens_per_s": cfg.prompt_len / (r["prefill_ms"] / 1e3),
                  "decode_hbm_gbs": bh / comp_dec_s / 1e9, "decode_hbm_frac": bh / comp_dec_s / 1e9 / peaks["hbm_gbs"]}
        copy_s = cs_dec["copy_busy_ms"] / 1e3 / K
        exposed = max(0.0, dec_s / K - comp_dec_s)
        hidden = max(0.0, 1.0 - exposed / copy_s) if copy_s > 0 else None

    # ---- context points (one request each, not the headline): reactive LRU cache without prefetch (BASELINE.json
    # configs[4] "no-prefetch reactive baseline") and the oracle-routing predictor (its upper bound)
    variants = None
    if rank == 0 and args.variants:
        variants = {}
        for name, pm in (("reactive_no_prefetch", B.PRED_NONE), ("oracle_routing_predictor", B.PRED_TRACE)):
            inj = None
            if pm == B.PRED_TRACE:
                rec = ProMoE(weights, cache_slots=cfg.cache_slots, stride=cfg.stride, predictor_mode=B.PRED_NONE,
                             flags=flags | B.F_TRACE, device=f"cuda:{local}")
                inj = []
                run_request(rec, cfg, prompt, decode_ids, greedy, record=inj)
                rec.close()
            v = ProMoE(weights, cache_slots=cfg.cache_slots, stride=cfg.stride, chunk_bytes=args.chunk_kb << 10,
                       predictor_mode=pm, flags=flags, max_inflight=args.inflight, device=f"cuda:{local}")
            run_request(v, cfg, prompt, decode_ids, greedy, inject=inj)
            r = run_request(v, cfg, prompt, decode_ids, greedy, inject=inj)
            v.close()
            need_d, need_p = r["dec"]["need_experts"] * Be, r["pre"]["need_experts"] * Be
            if pm == B.PRED_NONE:       # pollution-free B_need of the same requests → the headline fraction
                for roof, need, t_meas, key in ((roof_dec, need_d, dec_s, "dec"), (roof_pre, need_p, pre_s, "pre")):
                    t_r, bound_r, _ = roofline_time(need * K, roof["b_hbm_bytes"], roof["flops"], h2d_gbs, peaks["hbm_gbs"],
                                                    peaks["bf16_tflops_sustained"])
                    roof["b_need_reactive_bytes"] = need * K
                    roof["frac_vs_reactive_need"] = t_r / t_meas
                    roof["bound_vs_reactive_need"] = bound_r
            variants[name] = {
                "decode_tokens_per_s": cfg.decode_steps / (r["decode_ms"] / 1e3),
                "prefill_tokens_per_s": cfg.prompt_len / (r["prefill_ms"] / 1e3),
                "decode_roofline_frac": need_d / (h2d_gbs * 1e9) / (r["decode_ms"] / 1e3),
                "prefill_roofline_frac": need_p / (h2d_gbs * 1e9) / (r["prefill_ms"] / 1e3),
                "hit_rate": (r["dec"]["hits_resident"] + r["dec"]["hits_prefetch"]) / max(1, r["dec"]["accesses"]),
                "h2d_bytes_needed_per_token": need_d / cfg.decode_steps,
                "h2d_bytes_moved_per_token": r["dec"]["h2d_bytes"] / cfg.decode_steps}

    cpu = None
    if rank == 0 and not args.no_cpu:
        rpl, rds = ref_sample(args, cfg)
        o = oracle_sample(cfg, weights, rpl, rds)
        cpu = {"value": o["decode_tok_s"], "unit": "tokens/s", "cores": o["cores"], "kind": "oracle",
               "prefill_tokens_per_s": o["prefill_tok_s"], "seconds": o["seconds"],
               "sample": ref_sample_text(cfg, rpl, rds)}
    also = None
    if rank == 0 and world == 1 and args.also and args.also != cfg.name:
        # a second BASELINE.json config in the same run (one request each for ProMoE and the reactive cache), so that the round's
        # bench record carries more than the headline workload; not part of `value`
        del weights
        import gc
        gc.collect(); torch.cuda.empty_cache()
        also = {args.also: also_config(args, args.also, h2d_gbs, flags, local)}
    if rank != 0:
        return
    line = {"metric": METRIC, "value": g_dec_tok / g_dec_s, "unit": "tokens/s", "n_gpus": world, "steps": K,
            "warmup": args.warmup, "ms_per_step": 1e3 * wall / K, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": {0: "f32", 1: "f32 activations x bf16 weights, f32 accumulate",
                                          2: "f32 activations x (bf16 dense weights, int4 group-quantised experts), f32 accumulate"}[s.wdtype],
            "data": "synthetic", "config": workload_config(cfg, args),
            "prefill_tokens_per_s": g_pre_tok / g_pre_s, "decode_ms_per_token": 1e3 * g_dec_s / g_dec_tok * world,
            "ttft_ms": 1e3 * pre_s / K,
            "e2e": {"value": g_dec_wtok / g_dec_wall, "unit": "tokens/s", "prefill_tokens_per_s": g_pre_wtok / g_pre_wall,
                    "h2d_bytes_per_step": int((cs_dec["h2d_bytes_moved"] + cs_pre["h2d_bytes_moved"]) / K + 4 * (cfg.prompt_len + cfg.decode_steps)),
                    "d2h_bytes_per_step": 4 * s.vocab * (1 + cfg.decode_steps)},
            "gpu_launches": int(launches), "clocks": clk,
            "roofline": kernel_roof,
            "step_roofline": {"h2d_gbs_measured": h2d_gbs, "hbm_gbs": peaks["hbm_gbs"], "bf16_tflops": peaks["bf16_tflops_sustained"],
                              "peaks": peaks["source"], "decode": roof_dec, "prefill": roof_pre},
            "cache": {"decode": cs_dec, "prefill": cs_pre, "hidden_copy_fraction_decode": hidden},
            "all_resident": allhit, "variants": variants, "predictor_fit": fit_report, "also": also, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)


def run_sweep(args):
    """BASELINE.json configs[4]: sweep on the DeepSeek-MoE-16B-shaped decoder — expert-cache budget 25/50/75 % x
    predictor stride 1/2/3 x H2D chunk 1/4/16 MiB, plus the oracle-routing predictor and the reactive cache per
    budget; prompts 128 / 2048, 256 decode steps.  One JSON line per point (tokens/s, hit rate, hidden-copy
    fraction, % of the per-step roofline)."""
    import dataclasses
    import torch
    import synth
    from paper_2410_22134_b200 import binding as B
    from paper_2410_22134_b200.engine import ProMoE
    torch.cuda.set_device(0)
    peaks = load_peaks()
    base = synth.get_config("c3", shape_overrides={"max_seq": 2048 + 256, **({"wdtype": 2} if args.int4 else {})},
                            decode_steps=args.decode_steps or 256)
    s = base.shape
    n_moe = s.n_layers - s.n_dense_layers
    Be = expert_image_bytes(s)
    h2d = B.promoe_bench_h2d(256 << 20, 2, 5)
    w0 = synth.make_weights(base, predictor="skip")
    decode_ids = synth.make_decode_ids(base).tolist()
    prompts = {n: synth.make_prompt(base, n).tolist() for n in (128, 2048)}
    flags = B.F_PREEMPT | B.F_REORDER | B.F_WARM | B.F_TENSOR | (B.F_DEMOTE if args.demote else 0)
    wcache = {1: w0}

    def weights_for(stride):
        if stride not in wcache:      # the skip predictor's weights depend on the stride; the experts are shared
            wcache[stride] = synth.make_weights(dataclasses.replace(base, stride=stride), predictor="skip",
                                                experts_buf=w0.experts, fill_experts=False)
        return wcache[stride]

    def one(cfg, eng, prompt, inject=None):
        run_request(eng, dataclasses.replace(cfg, decode_steps=4), prompt[:64], decode_ids, False)       # warm-up
        return run_request(eng, cfg, prompt, decode_ids, False, inject=inject)

    compute = {}
    full = ProMoE(w0, cache_slots=n_moe * s.n_experts, stride=1, predictor_mode=B.PRED_MLP, flags=flags)
    for n, pr in prompts.items():
        r = one(dataclasses.replace(base, prompt_len=n), full, pr)
        compute[n] = (r["prefill_ms"], r["decode_ms"])
    full.close()
    routing = {}
    points = []
    for frac in (0.25, 0.5, 0.75):
        slots = int(s.n_experts * frac) * n_moe
        grid = [("mlp", st, ch) for st in (1, 2, 3) for ch in (1, 4, 16)] + [("trace", 1, 4), ("none", 1, 4)]
        for mode, stride, chunk in grid:
            w = weights_for(stride if mode == "mlp" else 1)
            pm = {"mlp": B.PRED_MLP, "trace": B.PRED_TRACE, "none": B.PRED_NONE}[mode]
            for n, pr in prompts.items():
                cfg = dataclasses.replace(base, prompt_len=n, cache_slots=slots, stride=stride)
                inj = None
                if mode == "trace":
                    if n not in routing:     # routing does not depend on the cache: record it once per prompt
                        rec = ProMoE(w, cache_slots=slots, stride=1, predictor_mode=B.PRED_NONE, flags=flags | B.F_TRACE)
                        routing[n] = []
                        run_request(rec, cfg, pr, decode_ids, False, record=routing[n])
                        rec.close()
                    inj = routing[n]
                eng = ProMoE(w, cache_slots=slots, stride=stride, chunk_bytes=chunk << 20, predictor_mode=pm, flags=flags,
                             max_inflight=args.inflight, max_spec_decode=0 if mode == "trace" else args.max_spec_decode)
                r = one(cfg, eng, pr, inject=inj)
                eng.close()
                d, p = r["dec"], r["pre"]
                dec_s, pre_s = r["decode_ms"] / 1e3, r["prefill_ms"] / 1e3
                copy_s = d["copy_busy_ms"] / 1e3
                exposed = max(0.0, dec_s - compute[n][1] / 1e3)
                pt = {"budget": frac, "predictor": mode, "stride": stride, "chunk_mib": chunk, "prompt": n, "demote": args.demote,
                      "int4": args.int4, "fetch_rate": d["fetched_at_gate"] / max(1, d["fetched_at_gate_of"]),
                      "fetch_rate_chunks": d["landed_chunks_at_gate"] / max(1, d["landed_chunks_of"]),
                      "decode_tokens_per_s": cfg.decode_steps / dec_s, "prefill_tokens_per_s": n / pre_s,
                      "hit_rate": (d["hits_resident"] + d["hits_prefetch"]) / max(1, d["accesses"]),
                      "hit_rate_resident": d["hits_resident"] / max(1, d["accesses"]),
                      "predictor_accuracy": d["predicted_correct"] / max(1, d["predicted"]),
                      "hidden_copy_fraction": max(0.0, 1.0 - exposed / copy_s) if copy_s > 0 else None,
                      "byte_efficiency": d["need_experts"] * Be / max(1, d["h2d_bytes"]),
                      "decode_roofline_frac": d["need_experts"] * Be / (h2d * 1e9) / dec_s,
                      "prefill_roofline_frac": p["need_experts"] * Be / (h2d * 1e9) / pre_s}
                points.append(pt)
                print(json.dumps(pt), flush=True)
    print(json.dumps({"sweep": "c5", "points": len(points), "h2d_gbs": h2d, "hbm_gbs": peaks["hbm_gbs"],
                      "compute_only_ms": {str(k): v for k, v in compute.items()}}), flush=True)


def run_modes(args):
    """--ladder: PAPER.md §7.3 / Fig. 12 — Base (LRU, ID order, no prefetch) → +prefetch (un-chunked, no early
    preemption) → +chunked → +early preemption → +reordered inference, and this build's own additions (demotion of
    mispredictions, the fitted predictor).  --goodpred: §4.1 Accuracy, FetchRate, GoodPred of the `skip` and the
    fitted predictor at strides 1-3.  One request (after one warm-up request) per row, one JSON line per row."""
    import dataclasses
    import torch
    import synth
    from paper_2410_22134_b200 import binding as B
    from paper_2410_22134_b200.engine import ProMoE
    from paper_2410_22134_b200.fit_predictor import fit_predictor
    torch.cuda.set_device(0)
    over = {}
    if args.prompt_len:
        over["prompt_len"] = args.prompt_len
    if args.decode_steps:
        over["decode_steps"] = args.decode_steps
    if args.int4:
        over["shape_overrides"] = {"wdtype": 2}
    base = synth.get_config(args.config, **over)
    s = base.shape
    Be = expert_image_bytes(s)
    h2d = B.promoe_bench_h2d(256 << 20, 2, 5)
    prompt = synth.make_prompt(base).tolist()
    decode_ids = synth.make_decode_ids(base).tolist()
    wcache = {}

    def weights_for(stride, kind):
        key = (stride, kind)
        if key not in wcache:
            cfg = dataclasses.replace(base, stride=stride)
            first = next(iter(wcache.values()))[0] if wcache else None
            w = synth.make_weights(cfg, predictor="skip", experts_buf=first.experts if first is not None else None,
                                   fill_experts=first is None)
            rep = None
            if kind == "fitted":
                rep = fit_predictor(w, cfg, stride, n_prompts=args.fit_prompts, steps=args.fit_steps)
                rep.pop("per_layer")
            wcache[key] = (w, rep)
        return wcache[key]

    P, R, D, U, TN, W = B.F_PREEMPT, B.F_REORDER, B.F_DEMOTE, B.F_UNCHUNKED, (B.F_TENSOR if args.tensor else 0), B.F_WARM
    if args.ladder:
        st = base.stride
        rows = [("static cache (fixed set + top_k staging buffers, P:317)", "static", st, W | TN, 0),
                ("base: LRU, ID order, no prefetch", "none", st, W | TN, 0),
                ("+prefetch (un-chunked, no preemption)", "skip", st, W | TN | U, args.max_spec_decode),
                ("+chunked", "skip", st, W | TN, args.max_spec_decode),
                ("+early preemption", "skip", st, W | TN | P, args.max_spec_decode),
                ("+reordered inference (= ProMoE)", "skip", st, W | TN | P | R, args.max_spec_decode),
                ("reordered, no prefetch (reactive)", "none", st, W | TN | P | R, 0),
                ("ProMoE + demotion (G17)", "skip", st, W | TN | P | R | D, args.max_spec_decode),
                ("ProMoE + demotion + fitted predictor", "fitted", st, W | TN | P | R | D, args.max_spec_decode)]
    else:
        rows = [(f"{kind} stride {st}", kind, st, W | TN | P | R | (D if args.demote else 0), args.max_spec_decode)
                for st in (1, 2, 3) for kind in ("skip", "fitted")]
    for label, kind, stride, flags, ms in rows:
        w, rep = weights_for(stride, "fitted" if kind == "fitted" else "skip")
        cfg = dataclasses.replace(base, stride=stride)
        eng = ProMoE(w, cache_slots=cfg.cache_slots, stride=stride, chunk_bytes=args.chunk_kb << 10,
                     predictor_mode=B.PRED_NONE if kind in ("none", "static") else B.PRED_MLP, flags=flags, max_inflight=args.inflight,
                     max_spec_decode=ms, max_spec_prefill=args.max_spec_prefill, fetch_ctas=args.fetch_ctas,
                     static_slots=cfg.slots_per_layer - s.top_k if kind == "static" else 0)
        run_request(eng, cfg, prompt, decode_ids, False)
        r = run_request(eng, cfg, prompt, decode_ids, False)
        eng.close()
        d, p = r["dec"], r["pre"]
        dec_s, pre_s = r["decode_ms"] / 1e3, r["prefill_ms"] / 1e3
        acc = d["predicted_correct"] / max(1, d["predicted"])
        fr = d["fetched_at_gate"] / max(1, d["fetched_at_gate_of"])
        frc = d["landed_chunks_at_gate"] / max(1, d["landed_chunks_of"])
        row = {"mode": label, "config": cfg.name, "stride": stride, "predictor": kind,
               "decode_tokens_per_s": cfg.decode_steps / dec_s, "prefill_tokens_per_s": cfg.prompt_len / pre_s,
               "decode_roofline_frac": d["need_experts"] * Be / (h2d * 1e9) / dec_s,
               "prefill_roofline_frac": p["need_experts"] * Be / (h2d * 1e9) / pre_s,
               "hit_rate": (d["hits_resident"] + d["hits_prefetch"]) / max(1, d["accesses"]),
               "miss_rate_prefill": p["misses"] / max(1, p["accesses"]),
               "accuracy": acc, "fetch_rate": fr, "fetch_rate_chunks": frc, "good_pred": acc * fr, "good_pred_chunks": acc * frc,
               "need_mb_per_token": d["need_experts"] * Be / 1e6 / cfg.decode_steps,
               "moved_mb_per_token": d["h2d_bytes"] / 1e6 / cfg.decode_steps,
               "prefill_moved_gb": p["h2d_bytes"] / 1e9, "prefill_need_gb": p["need_experts"] * Be / 1e9,
               "fit": rep}
        print(json.dumps(row), flush=True)
    print(json.dumps({"modes": "ladder" if args.ladder else "goodpred", "rows": len(rows), "h2d_gbs": h2d}), flush=True)


def run_batch_sweep(args):
    """PAPER.md §7.5: decode at batch sizes 1-4.  nb sequences with their own seeded prompts are prefilled one
    by one, then every decode step is ONE promoe_decode_batch call (one gate / slot-table step per layer over the union of
    the rows' experts).  One JSON line per batch size: tokens/s = nb x steps / device time."""
    import dataclasses
    import torch
    import synth
    from paper_2410_22134_b200 import binding as B
    from paper_2410_22134_b200.engine import ProMoE
    torch.cuda.set_device(0)
    over = {}
    if args.prompt_len:
        over["prompt_len"] = args.prompt_len
    if args.decode_steps:
        over["decode_steps"] = args.decode_steps
    if args.int4:
        over["shape_overrides"] = {"wdtype": 2}
    cfg = synth.get_config(args.config, **over)
    s = cfg.shape
    Be = expert_image_bytes(s)
    h2d = B.promoe_bench_h2d(256 << 20, 2, 5)
    w = synth.make_weights(cfg, predictor="skip")
    flags = B.F_PREEMPT | B.F_REORDER | B.F_WARM | (B.F_TENSOR if args.tensor else 0) | (B.F_DEMOTE if args.demote else 0)
    pm = B.PRED_NONE if args.predictor == "none" else B.PRED_MLP
    for nb in (1, 2, 3, 4):
        g = torch.Generator().manual_seed(4242)
        prompts = [torch.randint(0, s.vocab, (cfg.prompt_len,), generator=g, dtype=torch.int32).tolist() for _ in range(nb)]
        dec = torch.randint(0, s.vocab, (cfg.decode_steps, nb), generator=g, dtype=torch.int32).tolist()
        eng = ProMoE(w, cache_slots=cfg.cache_slots, stride=cfg.stride, chunk_bytes=args.chunk_kb << 10, predictor_mode=pm, flags=flags,
                     max_spec_decode=args.max_spec_decode, max_spec_prefill=args.max_spec_prefill, fetch_ctas=args.fetch_ctas,
                     max_batch=nb)
        res = None
        for rep_ in range(2):                     # one warm-up pass, one timed
            eng.reset()
            for b in range(nb):
                eng.prefill_seq(b, prompts[b], want_logits=False)
            s1 = eng.stats()
            for row in dec:
                eng.decode_batch(list(range(nb)), row)
            s2 = eng.stats()
            res = {k: s2[k] - s1[k] for k in s1}
        eng.close()
        dec_s = res["step_ms"] / 1e3
        line = {"mode": "batched decode", "config": cfg.name, "batch": nb, "int4": args.int4, "predictor": args.predictor,
                "decode_tokens_per_s": nb * cfg.decode_steps / dec_s, "ms_per_step": 1e3 * dec_s / cfg.decode_steps,
                "experts_needed_per_layer_step": res["accesses"] / (cfg.decode_steps * (s.n_layers - s.n_dense_layers)),
                "hit_rate": (res["hits_resident"] + res["hits_prefetch"]) / max(1, res["accesses"]),
                "need_mb_per_step": res["need_experts"] * Be / 1e6 / cfg.decode_steps,
                "moved_mb_per_step": res["h2d_bytes"] / 1e6 / cfg.decode_steps,
                "decode_roofline_frac": res["need_experts"] * Be / (h2d * 1e9) / dec_s,
                "path": "fused decode step + device-side fetch worker" if nb == 1 else "T > 1 layer loop (copy-engine fills, per-row fused attention)"}
        print(json.dumps(line), flush=True)


def spawn_command(n_gpus: int, argv):
    """Command line that runs this script as n_gpus ranks on one node (127.0.0.1 rendezvous, a free port)."""
    import socket
    sk = socket.socket(); sk.bind(("127.0.0.1", 0)); port = sk.getsockname()[1]; sk.close()
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n_gpus}", "--master-addr", "127.0.0.1",
            "--master-port", str(port), os.path.abspath(__file__), *argv]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="c2")
    ap.add_argument("--predictor", default="skip", choices=["skip", "fitted", "random", "none", "trace"],
                    help="skip: training-free MLP weights; fitted: the MLP fitted offline on the model's own traces (fit_predictor.py); "
                         "none: reactive cache; trace: oracle-routing upper bound")
    ap.add_argument("--demote", type=int, default=1, help="PROMOE_F_DEMOTE: a mispredicted prefetch becomes the next LRU victim (G17)")
    ap.add_argument("--fit-prompts", type=int, default=20, help="--predictor fitted: prompts of prompt_len tokens to collect traces from")
    ap.add_argument("--fit-steps", type=int, default=240, help="--predictor fitted: optimiser steps per layer")
    ap.add_argument("--cache-all", type=int, default=0, help="every routed expert resident (compute-only step; with --fetch-ctas -1 "
                    "this is the configuration ncu can profile: a kernel-serialising profiler cannot run the persistent fetch worker)")
    ap.add_argument("--also", default="c3", help="a second config measured briefly in the same run and reported under `also` ('' = none)")
    ap.add_argument("--stride", type=int, default=0, help="predictor stride (0 = the config's: c2 2, c3 / c4 1)")
    ap.add_argument("--int4", type=int, default=0, help="routed experts as INT4 group-quantised images (SURVEY N3; wdtype 2)")
    ap.add_argument("--ladder", action="store_true", help="ablation ladder of PAPER.md §7.3 / Fig. 12 (one JSON line per rung)")
    ap.add_argument("--batch-sweep", action="store_true", help="decode at batch sizes 1-4 (PAPER.md §7.5), one JSON line per batch size")
    ap.add_argument("--goodpred", action="store_true", help="Accuracy / FetchRate / GoodPred of skip vs fitted at strides 1-3 (one JSON line per row)")
    ap.add_argument("--decode", default="random", choices=["random", "greedy"],
                    help="decode ids: seeded random (locality-neutral, default) or greedy argmax")
    ap.add_argument("--chunk-kb", type=int, default=0, help="chunk size in KiB: granularity of the ready flags, of LOW copies and of preemption (0 = library default 256)")
    ap.add_argument("--inflight", type=int, default=0, help="LOW chunks kept in flight (bounded preemption delay, P:191)")
    ap.add_argument("--max-spec-decode", type=int, default=1, help="allocations per PushPredicted in decode (0 = top_k as in Alg. 2, <0 = none); default 1: on a B200 one layer of\n                    compute hides about half an expert copy (profiles/r01_sweep_c2.md)")
    ap.add_argument("--max-spec-prefill", type=int, default=0, help="allocations per PushPredicted in prefill (<=0 = none)")
    ap.add_argument("--low-cap", type=int, default=0, help="a LOW fill stops after this many chunks (0 = no cap)")
    ap.add_argument("--fetch-ctas", type=int, default=0, help="CTAs of the device-side fetch worker (0 = library default 2)")
    ap.add_argument("--tensor", type=int, default=1, help="prefill GEMMs on tcgen05 (bf16 weights)")
    ap.add_argument("--prompt-len", type=int, default=0)
    ap.add_argument("--decode-steps", type=int, default=0)
    ap.add_argument("--ref-prompt", type=int, default=0, help="oracle sample: prompt tokens (0 = the whole prompt, capped at 512)")
    ap.add_argument("--ref-decode", type=int, default=2, help="oracle sample: decode tokens")
    ap.add_argument("--sweep", action="store_true", help="BASELINE.json configs[4] grid on the c3 shape (one JSON line per point)")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-allhit", action="store_true")
    ap.add_argument("--variants", type=int, default=1, help="also measure the reactive and oracle-routing context points")
    args = ap.parse_args()

    if args.sweep:
        run_sweep(args)
        return
    if args.ladder or args.goodpred:
        run_modes(args)
        return
    if args.batch_sweep:
        run_batch_sweep(args)
        return
    import synth
    over = {}
    if args.prompt_len:
        over["prompt_len"] = args.prompt_len
    if args.decode_steps:
        over["decode_steps"] = args.decode_steps
    if args.int4:
        over["shape_overrides"] = {"wdtype": 2}
    if args.stride:
        over["stride"] = args.stride
    cfg = synth.get_config(args.config, **over)
    if args.cache_all:
        import dataclasses
        cfg = dataclasses.replace(cfg, cache_slots=(cfg.shape.n_layers - cfg.shape.n_dense_layers) * cfg.shape.n_experts)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # launched as a plain `python bench.py --gpus N`: start the N ranks ourselves, one process per GPU, the way the
        # driver does (replicas only; NCCL carries the two aggregate all-reduces, nothing on the data path)
        sys.exit(subprocess.call(spawn_command(args.gpus, sys.argv[1:])))
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, cfg, rank)
        return
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl")
    run_ours(args, cfg, rank, world, dist)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
