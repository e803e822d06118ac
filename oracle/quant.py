"""INT4 group-quantised routed experts: dequantisation (ORACLE; test infrastructure).

PAPER.md P:313 ("QW-2 and Mixt are evaluated using INT4 precision"), §7.6 (GPTQ-quantised experts):
the expert parameters that travel over PCIe and sit in the cache are 4-bit; the computation is unchanged ("keeping the
amount of computation ... constant").  The paper does not fix the container format; reading G18 does:

  per weight matrix W [N, K] (K = the reduction dimension, a multiple of 128), row-major:
    codes  : N·K/2 bytes, element (n, k) in byte (n·K + k) / 2, EVEN k in the low nibble, odd k in the high nibble;
    scales : N·K/128 bf16 values, group g = k / 128 of row n at index n·(K/128) + g;
    value  : W[n, k] = (code − 8) · scale          (symmetric, zero point 8, code ∈ 0..15)
  expert image = [gate codes | up codes | down codes | gate scales | up scales | down scales], gate/up [I, H], down [H, I].

The oracle dequantises to fp64 and then runs the same fp64 FFN as for bf16 experts — "dequantise, then the plain
definition".  Written out with integer arithmetic on the bytes; shares nothing with synth's packer or the CUDA kernels.
"""
from __future__ import annotations

from typing import Tuple

import torch

GROUP = 128


def unpack_matrix(codes: torch.Tensor, scales_bf16_bytes: torch.Tensor, n_rows: int, k: int) -> torch.Tensor:
    """codes uint8 [n_rows·k/2], scale bytes uint8 [n_rows·k/128·2] (little-endian bf16) → W fp64 [n_rows, k]."""
    b = codes.to(torch.int64)
    lo = b & 15           # even k
    hi = b >> 4           # odd k
    q = torch.stack([lo, hi], dim=-1).reshape(n_rows, k) - 8
    sb = scales_bf16_bytes.to(torch.int64).reshape(-1, 2)
    bits16 = sb[:, 0] | (sb[:, 1] << 8)                          # bf16 bit pattern = upper half of an fp32
    scale = (bits16 << 16).to(torch.int32).view(torch.float32).to(torch.float64).reshape(n_rows, k // GROUP)
    return q.to(torch.float64) * scale.repeat_interleave(GROUP, dim=1)


def dequant_expert(img: torch.Tensor, hidden: int, inter: int) -> Tuple[torch.Tensor, torch.Tensor, torch.Tensor]:
    """img uint8 [3·H·I/2 + 3·H·I/128·2] → (Wgate [I,H], Wup [I,H], Wdown [H,I]) fp64."""
    hi = hidden * inter
    nc, ns = hi // 2, hi // GROUP * 2
    assert img.dtype == torch.uint8 and img.numel() == 3 * (nc + ns)
    s0 = 3 * nc
    wg = unpack_matrix(img[0:nc], img[s0:s0 + ns], inter, hidden)
    wu = unpack_matrix(img[nc:2 * nc], img[s0 + ns:s0 + 2 * ns], inter, hidden)
    wd = unpack_matrix(img[2 * nc:3 * nc], img[s0 + 2 * ns:s0 + 3 * ns], hidden, inter)
    return wg, wu, wd
