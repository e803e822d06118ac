"""Pins for oracle/quant.py (INT4 group-quantised experts, G18; §7.6) — CPU only.

The dequantiser is pinned to things other than itself: a group written out by hand, byte by byte; a layout test that
plants single non-zero codes at known addresses of a full expert image; the quantisation error bound of the packer
(|w − ŵ| ≤ scale/2 inside the clamp range); weights that are exactly representable in the format (so the INT4 model
must equal the bf16 model bit for bit in fp64); and the identity "quantised expert = FFN of its dequantised matrices".
"""
import struct

import torch

import synth
from oracle.forward import OracleModel, swiglu_ffn
from oracle.quant import GROUP, dequant_expert, unpack_matrix
from synth.weights import pack_int4


def _bf16_bytes(x: float):
    b = struct.pack("<f", x)
    assert b[0] == 0 and b[1] == 0, "value must be bf16-representable"
    return [b[2], b[3]]


def test_hand_written_group():
    """One row of 128 elements, scale 0.5: byte j holds elements 2j (low nibble) and 2j+1 (high nibble);
    value = (code − 8)·0.5.  Bytes 0x08, 0xF0, 0x7A, 0x19 → elements (8,0) (0,15) (10,7) (9,1) → 0, −4, −4, 3.5, 1, −0.5, 0.5, −3.5."""
    codes = torch.tensor([0x08, 0xF0, 0x7A, 0x19] + [0x88] * 60, dtype=torch.uint8)
    scales = torch.tensor(_bf16_bytes(0.5), dtype=torch.uint8)
    w = unpack_matrix(codes, scales, 1, 128)
    assert w.dtype == torch.float64 and w.shape == (1, 128)
    assert w[0, :8].tolist() == [0.0, -4.0, -4.0, 3.5, 1.0, -0.5, 0.5, -3.5]
    assert w[0, 8:].abs().max().item() == 0.0            # code 8 = zero
    # the 16 codes map to −8..7 times the scale
    allc = torch.tensor([(2 * j) | ((2 * j + 1) << 4) for j in range(8)] + [0x88] * 56, dtype=torch.uint8)
    w = unpack_matrix(allc, torch.tensor(_bf16_bytes(0.25), dtype=torch.uint8), 1, 128)
    assert w[0, :16].tolist() == [(c - 8) * 0.25 for c in range(16)]


def test_scale_index_is_row_major_per_group():
    """2 rows × 256 elements: 4 groups, scales 1, 2, 4, 8 in (row, group) order; every code = 9 (value +1·scale)."""
    codes = torch.full((2 * 256 // 2,), 0x99, dtype=torch.uint8)
    scales = torch.tensor(sum((_bf16_bytes(v) for v in (1.0, 2.0, 4.0, 8.0)), []), dtype=torch.uint8)
    w = unpack_matrix(codes, scales, 2, 256)
    assert w[0, :128].unique().tolist() == [1.0] and w[0, 128:].unique().tolist() == [2.0]
    assert w[1, :128].unique().tolist() == [4.0] and w[1, 128:].unique().tolist() == [8.0]


def test_image_layout_by_planting_single_codes():
    """[gate codes | up codes | down codes | gate scales | up scales | down scales]; gate/up [I, H], down [H, I]."""
    H, I = 256, 384
    hi = H * I
    nc, ns = hi // 2, hi // GROUP * 2
    img = torch.full((3 * (nc + ns),), 0x88, dtype=torch.uint8)
    one = torch.tensor(_bf16_bytes(1.0) * (hi // GROUP), dtype=torch.uint8)
    for k in range(3):
        img[3 * nc + k * ns:3 * nc + (k + 1) * ns] = one
    # gate (row 5, col 10): even col → low nibble, code 15 → +7
    img[(5 * H + 10) // 2] = 0x8F
    # up (row 7, col 33): odd col → high nibble, code 0 → −8
    img[nc + (7 * H + 33) // 2] = 0x08
    # down (row 200, col 383): odd → high nibble, code 12 → +4; its group (200, 383 // 128 = 2) gets scale 0.5
    img[2 * nc + (200 * I + 383) // 2] = 0xC8
    so = 3 * nc + 2 * ns + (200 * (I // GROUP) + 2) * 2
    img[so:so + 2] = torch.tensor(_bf16_bytes(0.5), dtype=torch.uint8)
    wg, wu, wd = dequant_expert(img, H, I)
    assert wg.shape == (I, H) and wu.shape == (I, H) and wd.shape == (H, I)
    assert wg[5, 10].item() == 7.0 and wg.abs().sum().item() == 7.0
    assert wu[7, 33].item() == -8.0 and wu.abs().sum().item() == 8.0
    assert wd[200, 383].item() == 2.0 and wd.abs().sum().item() == 2.0


def test_packer_error_bound_and_roundtrip():
    """synth.pack_int4 (the offline quantiser stand-in) followed by the oracle's unpack: |w − ŵ| ≤ scale/2 (+ the bf16
    rounding of the scale: the group maximum may be clamped by up to 7·2⁻⁹·scale), scale = bf16(max|w|/7)."""
    g = torch.Generator().manual_seed(3)
    w = torch.randn(24, 512, generator=g) * 0.05
    codes, scales = pack_int4(w)
    assert codes.shape == (24, 256) and scales.shape == (24, 4) and scales.dtype == torch.bfloat16
    what = unpack_matrix(codes.reshape(-1), scales.contiguous().view(torch.uint8).reshape(-1), 24, 512)
    sc = scales.to(torch.float64).repeat_interleave(GROUP, dim=1)
    assert ((w.double() - what).abs() <= sc * (0.5 + 7 * 2.0 ** -8)).all()
    assert (what / sc == torch.round(what / sc)).all() and (what / sc).abs().max() <= 8
    # all-zero group → scale 1, codes 8
    z = torch.zeros(1, 128)
    c0, s0 = pack_int4(z)
    assert s0.item() == 1.0 and (c0 == 0x88).all()


def test_exactly_representable_weights_give_the_bf16_model():
    """Special case that reduces to the existing (pinned) bf16 path: expert weights on the grid {−7..7}·2⁻⁶ with every
    group containing ±7 survive quantisation exactly, so the INT4 model's outputs equal the bf16 model's in fp64."""
    cfg = synth.get_config("c1b")
    w16 = synth.make_weights(cfg, pin=False)
    g = torch.Generator().manual_seed(11)
    grid = torch.randint(-7, 8, w16.experts.shape, generator=g).float()
    grid[..., ::GROUP] = 7.0                                          # every group of 128 starts with the maximum code
    w16.experts.copy_((grid * 2.0 ** -6).to(torch.bfloat16))
    s4 = synth.get_config("c1b", shape_overrides={"wdtype": 2})
    w4 = synth.make_weights(s4, pin=False)
    H, I = cfg.shape.hidden, cfg.shape.expert_inter
    hi = H * I
    for m in range(w16.experts.shape[0]):
        for k, kdim in enumerate((H, H, I)):
            mat = w16.experts[m, :, k * hi:(k + 1) * hi].float().view(-1, hi // kdim, kdim)
            codes, scales = pack_int4(mat)
            w4.experts[m, :, k * (hi // 2):(k + 1) * (hi // 2)] = codes.reshape(mat.shape[0], -1)
            so = 3 * (hi // 2) + k * (hi // GROUP) * 2
            w4.experts[m, :, so:so + (hi // GROUP) * 2] = scales.contiguous().view(torch.uint8).reshape(mat.shape[0], -1)
    w4.dense = w16.dense
    ids = synth.make_prompt(cfg, 9).tolist()
    a = OracleModel(w16, use_predictor=False).forward(ids)
    b = OracleModel(w4, use_predictor=False).forward(ids)
    assert torch.equal(a.hidden, b.hidden) and torch.equal(a.logits, b.logits)
    assert [lt.sel for lt in a.layers] == [lt.sel for lt in b.layers]


def test_int4_expert_is_the_ffn_of_its_dequantised_matrices():
    cfg = synth.get_config("c1", shape_overrides={"wdtype": 2})
    w = synth.make_weights(cfg, pin=False)
    s = cfg.shape
    assert w.experts.dtype == torch.uint8 and w.experts.shape[2] == synth.configs.expert_bytes(s) == 3 * s.hidden * s.expert_inter * 33 // 64
    wg, wu, wd = dequant_expert(w.experts[1, 3], s.hidden, s.expert_inter)
    # quantised values stay close to N(0, 1/fan_in) draws: the format loses at most half a step of max|w|/7 per group
    assert 0.8 * s.hidden ** -0.5 < wg.std().item() < 1.2 * s.hidden ** -0.5
    u = torch.randn(3, s.hidden, dtype=torch.float64, generator=torch.Generator().manual_seed(1))
    y = swiglu_ffn(u, wg, wu, wd)
    a, b = u @ wg.T, u @ wu.T
    assert torch.allclose(y, ((a / (1 + torch.exp(-a))) * b) @ wd.T, rtol=1e-12, atol=1e-14)
    # and the model runs end to end on INT4 experts
    st = OracleModel(w, use_predictor=True).forward(synth.make_prompt(cfg, 5).tolist())
    assert st.hidden.shape == (5, s.hidden) and torch.isfinite(st.logits).all()
