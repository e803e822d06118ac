"""Seeded random weights, prompts and decode ids (inputs only; no method arithmetic).

Recipe (BASELINE.json: "Weights and embeddings N(0, 1/fan_in)"):
  * linear weights  W[out, in] ~ N(0, 1/in), stored row-major [out_features, in_features];
  * embeddings ~ N(0, 1)  (a lookup's fan-in is 1);
  * RMSNorm gains = 1 + 0.1*N(0,1), fp32 (so that a dropped gain is visible in tests);
  * c3: router bias b_e = ln p_e - mean(ln p), p_e ∝ (π(e)+1)^-s, π a seeded permutation;
  * predictor weights, by `predictor=`:
      "random": W1, W2 ~ N(0, 1/fan_in)                       (BASELINE.json-literal, accuracy ≈ k/E)
      "skip"  : W1 = [R; -R; 0], W2 = [I, -I, 0] with R the router of the TARGET layer (l+stride), so the
                MLP output equals R·u exactly (one ReLU branch is zero) — the paper's skip-based predictor
                (§4.2) in the learned predictor's shape (SURVEY finding 3).  Needs ph >= 2E.
  * every tensor has its own generator seeded with (seed, tensor name), so shapes can change independently.
Weights are cast to bf16 (round-to-nearest-even) when shape.wdtype == 1; both sides see the same bits.

Each routed expert is ONE contiguous image [Wgate (I×H) | Wup (I×H) | Wdown (H×I)] (three linears);
all images live in one [n_moe_layers, E, 3·H·I] host tensor, pinned when CUDA is present ("routed experts live in
pinned host memory", BASELINE.json configs[1]).

INT4 experts (shape.wdtype == 2, PAPER.md P:313 / §7.6 P:417-433 — the paper's QW-2 and Mixt run GPTQ-style
4-bit experts): the routed experts are drawn as above (bf16) and then packed by `pack_int4` — the stand-in for the
offline quantiser, an input-preparation step: per row, groups of 128 consecutive elements of the reduction dimension share
one bf16 scale = max|w| / 7 of the group (1 for an all-zero group); code = clamp(round_half_even(w / scale), −8, 7) + 8,
two codes per byte (even element in the low nibble).  Image = [gate codes | up codes | down codes | gate scales | up
scales | down scales] (uint8).  The dense weights of such a model stay bf16.  Dequantisation — value = (code − 8)·scale —
is method arithmetic and lives on the two sides separately (oracle/quant.py; csrc/kernels_q4.cu).

Large tensors are drawn with torch's CUDA Philox generator when a GPU is present (25-90 GB of normals are too slow
on the host); small configs always use the CPU generator so CPU-only tests see the same values everywhere.
"""
from __future__ import annotations

import hashlib
import math
from dataclasses import dataclass, field
from typing import Dict, List, Optional

import torch

from .configs import INT4_GROUP, RunConfig, Shape, expert_bytes, expert_elems, moe_layer_ids

_GPU_GEN_THRESHOLD = 1 << 26   # tensors above 64 Mi elements are drawn on the GPU when there is one


def _seed_for(seed: int, name: str) -> int:
    h = hashlib.sha256(f"{seed}:{name}".encode()).digest()
    return int.from_bytes(h[:8], "little") & ((1 << 63) - 1)


def _normal(seed: int, name: str, shape, std: float, dtype: torch.dtype, out: Optional[torch.Tensor] = None,
            allow_gpu: bool = True) -> torch.Tensor:
    n = 1
    for d in shape:
        n *= d
    use_gpu = allow_gpu and n >= _GPU_GEN_THRESHOLD and torch.cuda.is_available()
    dev = "cuda" if use_gpu else "cpu"
    g = torch.Generator(device=dev)
    g.manual_seed(_seed_for(seed, name))
    t = torch.randn(shape, generator=g, device=dev, dtype=torch.float32)
    t.mul_(std)
    t = t.to(dtype)
    if out is not None:
        out.copy_(t)
        return out
    return t.cpu()


def pack_int4(w: torch.Tensor, group: int = 128):
    """w [..., N, K] float (K a multiple of `group`) → (codes uint8 [..., N, K/2], scales bf16 [..., N, K/group])."""
    shp = w.shape
    K = shp[-1]
    assert K % group == 0
    g = w.to(torch.float32).reshape(*shp[:-1], K // group, group)
    amax = g.abs().amax(dim=-1, keepdim=True)
    scale = (amax / 7.0).to(torch.bfloat16)
    scale = torch.where(scale.to(torch.float32) == 0, torch.ones_like(scale), scale)
    code = torch.clamp(torch.round(g / scale.to(torch.float32)), -8, 7).to(torch.int16) + 8
    code = code.reshape(*shp[:-1], K // 2, 2)
    packed = (code[..., 0] | (code[..., 1] << 4)).to(torch.uint8)
    return packed, scale.reshape(*shp[:-1], K // group)


@dataclass
class Weights:
    shape: Shape
    dense: Dict[str, torch.Tensor]          # CPU tensors, names documented in make_weights
    experts: torch.Tensor                   # [n_moe_layers, E, 3*H*I], CPU (pinned if CUDA present)
    predictor: str = "skip"
    stride: int = 1

    def expert_views(self, m: int, e: int):
        """(Wgate [I,H], Wup [I,H], Wdown [H,I]) views of routed expert e of MoE layer m (fp32 / bf16 images; an INT4
        image is raw bytes — the oracle unpacks it itself, oracle/quant.py)."""
        s = self.shape
        if s.wdtype == 2:
            raise TypeError("INT4 expert images have no tensor views: unpack self.experts[m, e] (uint8)")
        img = self.experts[m, e]
        hi = s.hidden * s.expert_inter
        return (img[:hi].view(s.expert_inter, s.hidden),
                img[hi:2 * hi].view(s.expert_inter, s.hidden),
                img[2 * hi:].view(s.hidden, s.expert_inter))


def make_weights(cfg: RunConfig, predictor: str = "skip", pin: Optional[bool] = None,
                 experts_buf: Optional[torch.Tensor] = None, fill_experts: bool = True) -> Weights:
    """experts_buf: caller-provided [n_moe, E, 3·H·I] host tensor (e.g. a shared-memory mapping used by all ranks of a
    node); fill_experts=False: the buffer already holds the values (another rank drew them)."""
    s = cfg.shape
    seed = cfg.seed
    dt = torch.float32 if s.wdtype == 0 else torch.bfloat16     # dense weights (wdtype 2: bf16 dense, INT4 experts)
    H, d = s.hidden, s.head_dim
    nq, nkv = s.n_q_heads, s.n_kv_heads
    D: Dict[str, torch.Tensor] = {}

    def lin(name, out_f, in_f):
        D[name] = _normal(seed, name, (out_f, in_f), in_f ** -0.5, dt)

    def gain(name):
        D[name] = (1.0 + 0.1 * _normal(seed, name, (H,), 1.0, torch.float32)).contiguous()

    D["emb"] = _normal(seed, "emb", (s.vocab, H), 1.0, dt)
    lin("lm_head", s.vocab, H)
    gain("final_norm")
    moe_ids = moe_layer_ids(s)
    for l in range(s.n_layers):
        p = f"l{l}."
        gain(p + "ln1")
        gain(p + "ln2")
        lin(p + "wqkv", (nq + 2 * nkv) * d, H)      # rows: [q heads | k heads | v heads]
        lin(p + "wo", H, nq * d)
        if l < s.n_dense_layers:
            lin(p + "ffn_gate", s.dense_inter, H)
            lin(p + "ffn_up", s.dense_inter, H)
            lin(p + "ffn_down", H, s.dense_inter)
            continue
        lin(p + "router", s.n_experts, H)
        if s.router_bias:
            g = torch.Generator().manual_seed(_seed_for(seed, p + "router_bias"))
            perm = torch.randperm(s.n_experts, generator=g).to(torch.float64)
            logp = -cfg.zipf_s * torch.log(perm + 1.0)
            D[p + "router_bias"] = (logp - logp.mean()).to(torch.float32).contiguous()
        if s.n_shared_inter:
            lin(p + "ffn_gate", s.n_shared_inter, H)
            lin(p + "ffn_up", s.n_shared_inter, H)
            lin(p + "ffn_down", H, s.n_shared_inter)
            if s.shared_gate:
                lin(p + "shared_gate_w", 1, H)
    # predictors (one per MoE layer; the one at MoE index m targets MoE index m+stride)
    ph, E = s.pred_hidden, s.n_experts
    for mi, l in enumerate(moe_ids):
        p = f"l{l}."
        if predictor == "random":
            lin(p + "pred_w1", ph, H)
            lin(p + "pred_w2", E, ph)
        elif predictor == "skip":
            if ph < 2 * E:
                raise ValueError("skip predictor needs pred_hidden >= 2*n_experts")
            tgt = mi + cfg.stride
            w1 = torch.zeros(ph, H, dtype=dt)
            w2 = torch.zeros(E, ph, dtype=dt)
            if tgt < len(moe_ids):
                R = D[f"l{moe_ids[tgt]}.router"]
                w1[:E] = R
                w1[E:2 * E] = -R
                w2[:, :E] = torch.eye(E, dtype=dt)
                w2[:, E:2 * E] = -torch.eye(E, dtype=dt)
            D[p + "pred_w1"], D[p + "pred_w2"] = w1, w2
        else:
            raise ValueError(f"unknown predictor variant {predictor!r}")

    # routed experts: one contiguous host tensor, pinned if possible
    n_moe = s.n_moe_layers
    q4 = s.wdtype == 2
    per = expert_bytes(s) if q4 else expert_elems(s)
    edt = torch.uint8 if q4 else dt
    if pin is None:
        pin = torch.cuda.is_available()
    if experts_buf is not None:
        assert tuple(experts_buf.shape) == (n_moe, E, per) and experts_buf.dtype == edt
        experts = experts_buf
    else:
        experts = torch.empty((n_moe, E, per), dtype=edt, pin_memory=bool(pin))
    hi = H * s.expert_inter
    for mi, l in enumerate(moe_ids if fill_experts else []):
        # gate/up rows have fan-in H, down rows fan-in I; one draw per (layer, matrix) over all experts
        for k, (name, std) in enumerate((("gate", H ** -0.5), ("up", H ** -0.5), ("down", s.expert_inter ** -0.5))):
            if not q4:
                _normal(seed, f"l{l}.experts.{name}", (E, hi), std, dt, out=experts[mi, :, k * hi:(k + 1) * hi])
                continue
            dev = "cuda" if torch.cuda.is_available() and E * hi >= _GPU_GEN_THRESHOLD else "cpu"
            w = _normal(seed, f"l{l}.experts.{name}", (E, hi), std, dt).to(dev)
            kdim = H if k < 2 else s.expert_inter
            codes, scales = pack_int4(w.view(E, hi // kdim, kdim), INT4_GROUP)
            experts[mi, :, k * (hi // 2):(k + 1) * (hi // 2)].copy_(codes.reshape(E, hi // 2))
            so = 3 * (hi // 2) + k * (hi // INT4_GROUP) * 2
            experts[mi, :, so:so + (hi // INT4_GROUP) * 2].copy_(scales.reshape(E, hi // INT4_GROUP).contiguous().view(torch.uint8).reshape(E, -1))
    return Weights(shape=s, dense=D, experts=experts, predictor=predictor, stride=cfg.stride)


def make_prompt(cfg: RunConfig, length: Optional[int] = None) -> torch.Tensor:
    """Uniform random token ids in [0, vocab); seed = config seed + 1."""
    n = cfg.prompt_len if length is None else length
    g = torch.Generator().manual_seed(_seed_for(cfg.seed + 1, "prompt"))
    return torch.randint(0, cfg.shape.vocab, (n,), generator=g, dtype=torch.int32)


def make_decode_ids(cfg: RunConfig, n: Optional[int] = None) -> torch.Tensor:
    """Seeded random decode ids: the locality-neutral teacher-forced decode stream."""
    n = cfg.decode_steps if n is None else n
    g = torch.Generator().manual_seed(_seed_for(cfg.seed + 2, "decode"))
    return torch.randint(0, cfg.shape.vocab, (n,), generator=g, dtype=torch.int32)
