"""Byte and roofline accounting (ORACLE; test infrastructure).

expert_bytes: one routed expert = three linears of H×I weights ("three linear layers").
P:85 worked example: DS-1 decode needs 27 MoE layers × 6 experts × 3·2048·1408·2 B = 2673 MiB per token ("2.67 GiB"
in the paper, which divides MiB by 1000) and half of it, 1336 MiB ("1.33 GiB"), crosses PCIe at a 50 % cache.
Per-step roofline (BASELINE.json north_star):
   t_roof = max(B_need / BW_h2d, B_hbm / BW_hbm, F / peak_flops)
"""
from __future__ import annotations


def expert_bytes(hidden: int, inter: int, wbytes: int) -> int:
    return 3 * hidden * inter * wbytes


def decode_expert_bytes_per_token(n_moe_layers: int, top_k: int, hidden: int, inter: int, wbytes: int) -> int:
    return n_moe_layers * top_k * expert_bytes(hidden, inter, wbytes)


def step_roofline_seconds(b_need: float, b_hbm: float, flops: float, bw_h2d: float, bw_hbm: float, peak_flops: float):
    terms = {"h2d": b_need / bw_h2d, "hbm": b_hbm / bw_hbm, "tensor": flops / peak_flops}
    bound = max(terms, key=terms.get)
    return terms[bound], bound, terms
