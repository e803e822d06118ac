"""Model shapes and run parameters of BASELINE.json configs 1-5 (shapes only).

Citations: BASELINE.json `configs[0..4]`; Table 1 names the model
families whose *shapes* configs 2-4 take (QW-1, DS-1, Mixt).  Vocabulary sizes for
c2-c4 are the public values of those families; c1's is
BASELINE.json's 1000.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace, asdict
from typing import Dict, List


@dataclass(frozen=True)
class Shape:
    """Mirror of `promoe_shape_t` (include/promoe.h)."""
    n_layers: int
    hidden: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    vocab: int
    max_seq: int
    n_experts: int
    top_k: int
    expert_inter: int
    n_shared_inter: int = 0     # 0 = no shared expert
    shared_gate: int = 0        # 1 = sigmoid scalar gate on the shared expert (c2)
    n_dense_layers: int = 0     # leading layers with a dense FFN instead of MoE (c3: 1)
    dense_inter: int = 0
    router_bias: int = 0        # c3: per-expert logit bias
    pred_hidden: int = 128
    wdtype: int = 1             # 0 fp32 (c1), 1 bf16, 2 bf16 with INT4 group-quantised routed experts
    rope_theta: float = 10000.0
    rms_eps: float = 1e-6

    @property
    def n_moe_layers(self) -> int:
        return self.n_layers - self.n_dense_layers


@dataclass(frozen=True)
class RunConfig:
    name: str
    shape: Shape
    seed: int
    cache_slots: int            # TOTAL slots (per layer = cache_slots / n_moe_layers)
    stride: int
    prompt_len: int
    decode_steps: int
    zipf_s: float = 0.0         # c3: router bias ~ Zipf(s) popularity

    @property
    def slots_per_layer(self) -> int:
        return self.cache_slots // self.shape.n_moe_layers


def expert_elems(s: Shape) -> int:
    """Elements in one routed expert image [Wgate | Wup | Wdown] (3 linears)."""
    return 3 * s.hidden * s.expert_inter


INT4_GROUP = 128   # elements per quantisation group (along the reduction dimension)


def expert_bytes(s: Shape) -> int:
    if s.wdtype == 2:   # 4-bit codes, two per byte, + one bf16 scale per group of 128
        return expert_elems(s) // 2 + expert_elems(s) // INT4_GROUP * 2
    return expert_elems(s) * (4 if s.wdtype == 0 else 2)


def moe_layer_ids(s: Shape) -> List[int]:
    return list(range(s.n_dense_layers, s.n_layers))


_C1 = Shape(n_layers=2, hidden=256, n_q_heads=4, n_kv_heads=4, head_dim=64, vocab=1000, max_seq=64,
            n_experts=8, top_k=2, expert_inter=512, pred_hidden=128, wdtype=0)
_C2 = Shape(n_layers=24, hidden=2048, n_q_heads=16, n_kv_heads=16, head_dim=128, vocab=151936, max_seq=768,
            n_experts=60, top_k=4, expert_inter=1408, n_shared_inter=5632, shared_gate=1,
            pred_hidden=512, wdtype=1)
_C3 = Shape(n_layers=28, hidden=2048, n_q_heads=16, n_kv_heads=16, head_dim=128, vocab=102400, max_seq=1280,
            n_experts=64, top_k=6, expert_inter=1408, n_shared_inter=2816, shared_gate=0,
            n_dense_layers=1, dense_inter=10944, router_bias=1, pred_hidden=512, wdtype=1)
_C4 = Shape(n_layers=32, hidden=4096, n_q_heads=32, n_kv_heads=8, head_dim=128, vocab=32000, max_seq=768,
            n_experts=8, top_k=2, expert_inter=14336, pred_hidden=1024, wdtype=1)

CONFIGS: Dict[str, RunConfig] = {
    # BASELINE.json configs[0]: toy, fp32, 8 slots of 16 experts, stride 1, 32-token prompt + 16 decode steps.
    "c1": RunConfig("c1", _C1, seed=0, cache_slots=8, stride=1, prompt_len=32, decode_steps=16),
    # c1 with bf16 weights (exercises the tensor-core path in seconds).
    "c1b": RunConfig("c1b", replace(_C1, wdtype=1), seed=0, cache_slots=8, stride=1, prompt_len=32, decode_steps=16),
    # configs[1]: Qwen1.5-MoE-A2.7B-shaped, 50 % cache, stride 2, 512 + 128.
    "c2": RunConfig("c2", _C2, seed=1234, cache_slots=24 * 30, stride=2, prompt_len=512, decode_steps=128),
    # configs[2]: DeepSeek-MoE-16B-shaped, 50 % cache, stride 1, 1024 + 256, Zipf(0.3) router bias.
    "c3": RunConfig("c3", _C3, seed=1234, cache_slots=27 * 32, stride=1, prompt_len=1024, decode_steps=256, zipf_s=0.3),
    # configs[3]: Mixtral-8x7B-shaped, 25 % cache (64 of 256), stride 1, 512 + 128.
    "c4": RunConfig("c4", _C4, seed=1234, cache_slots=64, stride=1, prompt_len=512, decode_steps=128),
}


def get_config(name: str, **overrides) -> RunConfig:
    """Return a named config; `overrides` may replace RunConfig fields, `shape_overrides=dict` Shape fields."""
    cfg = CONFIGS[name]
    shape_over = overrides.pop("shape_overrides", None)
    if shape_over:
        cfg = replace(cfg, shape=replace(cfg.shape, **shape_over))
    return replace(cfg, **overrides) if overrides else cfg


def mini(name: str) -> RunConfig:
    """Reduced-depth variants of c2-c4 (same per-layer shapes, fewer layers, small vocab) for
    parity tests the oracle finishes in seconds.  Not bench workloads."""
    cfg = CONFIGS[name]
    s = cfg.shape
    nl = {"c2": 4, "c3": 4, "c4": 2}[name]
    shape = replace(s, n_layers=nl, vocab=2048, max_seq=256)
    per = cfg.slots_per_layer
    return replace(cfg, name=name + "-mini", shape=shape, cache_slots=per * shape.n_moe_layers,
                   prompt_len=96, decode_steps=8)
