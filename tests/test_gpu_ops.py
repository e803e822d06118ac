"""-m gpu: kernel-level parity of the micro entry points (C-ABI) against the oracle's pieces.

Rows of SURVEY.md §8(a): A4 router/top-k/gates (bit-exact selections), A8 permutation (bit-exact), linear and
A9 expert FFN (fp32 accumulate vs fp64: |err| <= 1e-4·scale, far inside north_star's 1e-2 tolerance).
Sizes span several tiles and a ragged tail; edge cases: k = E, k = 1, exact ties, T = 1, empty expert groups.
"""
from __future__ import annotations

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2410_22134_b200 import binding
    binding.lib()
    return binding


def _w(shape, dtype, seed, std=None):
    g = torch.Generator().manual_seed(seed)
    t = torch.randn(shape, generator=g) * (std if std is not None else shape[-1] ** -0.5)
    return t.to(dtype)


@pytest.mark.parametrize("wdtype", [0, 1])
@pytest.mark.parametrize("T,N,K,path", [(1, 60, 2048, 1), (1, 1000, 256, 1), (3, 77, 264, 1), (5, 60, 2048, 2),
                                        (97, 200, 264, 2), (130, 64, 512, 2), (1, 8, 4096, 0), (64, 6144, 256, 0)])
def test_op_linear(B, wdtype, T, N, K, path):
    dt = torch.float32 if wdtype == 0 else torch.bfloat16
    x = _w((T, K), torch.float32, 1, 1.0)
    w = _w((N, K), dt, 2)
    xd, wd = x.cuda(), w.cuda()
    y = torch.full((T, N), float("nan"), device="cuda")
    rc = B.lib().promoe_op_linear(xd.data_ptr(), wd.data_ptr(), y.data_ptr(), T, N, K, wdtype, path, None)
    assert rc == 0
    torch.cuda.synchronize()
    ref = x.double() @ w.double().T
    err = (y.cpu().double() - ref).abs().max().item()
    assert err <= 1e-4 * max(1.0, ref.abs().max().item()), err


@pytest.mark.parametrize("wdtype", [0, 1])
@pytest.mark.parametrize("T,H,E,k,bias", [(1, 256, 8, 2, False), (33, 256, 8, 8, False), (1, 2048, 60, 4, False),
                                          (130, 2048, 64, 6, True), (7, 512, 8, 1, False), (65, 264, 200, 16, True)])
def test_op_route(B, wdtype, T, H, E, k, bias):
    from oracle.forward import route
    dt = torch.float32 if wdtype == 0 else torch.bfloat16
    u = _w((T, H), torch.float32, 3, 1.0)
    R = _w((E, H), dt, 4)
    b = _w((E,), torch.float32, 5, 0.5) if bias else None
    ud, Rd = u.cuda(), R.cuda()
    bd = b.cuda() if bias else None
    z = torch.empty((T, E), device="cuda")
    sel = torch.empty((T, k), dtype=torch.int32, device="cuda")
    gates = torch.empty((T, k), device="cuda")
    margin = torch.empty((T,), device="cuda")
    rc = B.lib().promoe_op_route(ud.data_ptr(), Rd.data_ptr(), bd.data_ptr() if bias else None, T, H, E, k, wdtype,
                                 z.data_ptr(), sel.data_ptr(), gates.data_ptr(), margin.data_ptr(), None)
    assert rc == 0
    torch.cuda.synchronize()
    zo = u.double() @ R.double().T
    if bias:
        zo = zo + b.double()
    assert (z.cpu().double() - zo).abs().max().item() <= 1e-4
    near = 0
    for t in range(T):
        so, go, mo = route(zo[t], k)
        sg = sel[t].tolist()
        if sg != so:
            assert mo < 1e-3 or min(abs(zo[t][a] - zo[t][b2]).item() for a, b2 in zip(so, so[1:])) < 1e-3
            near += 1
            continue
        assert np.abs(np.asarray(go) - gates[t].cpu().numpy()).max() <= 1e-5
        assert abs(gates[t].sum().item() - 1.0) <= 1e-5
        if k < E:
            assert abs(margin[t].item() - mo) <= 1e-4
    assert near <= max(1, T // 20)


def test_op_route_exact_ties(B):
    """Constructed exact ties → lower expert index wins (north_star), on logits handed over through a one-hot u."""
    E, H, k = 8, 16, 3
    R = torch.zeros(E, H)
    vals = [1.0, 2.0, 2.0, 0.5, 2.0, 1.0, 1.0, -1.0]       # three-way tie at 2.0, three-way at 1.0
    for e, v in enumerate(vals):
        R[e, 0] = v
    u = torch.zeros(1, H); u[0, 0] = 1.0
    z = torch.empty((1, E), device="cuda"); sel = torch.empty((1, k), dtype=torch.int32, device="cuda")
    gates = torch.empty((1, k), device="cuda"); margin = torch.empty((1,), device="cuda")
    ud, Rd = u.cuda(), R.cuda()
    assert B.lib().promoe_op_route(ud.data_ptr(), Rd.data_ptr(), None, 1, H, E, k, 0, z.data_ptr(), sel.data_ptr(),
                                   gates.data_ptr(), margin.data_ptr(), None) == 0
    torch.cuda.synchronize()
    assert sel[0].tolist() == [1, 2, 4]
    assert margin[0].item() == pytest.approx(1.0)
    k = 5
    sel = torch.empty((1, k), dtype=torch.int32, device="cuda"); gates = torch.empty((1, k), device="cuda")
    assert B.lib().promoe_op_route(ud.data_ptr(), Rd.data_ptr(), None, 1, H, E, k, 0, z.data_ptr(), sel.data_ptr(),
                                   gates.data_ptr(), margin.data_ptr(), None) == 0
    torch.cuda.synchronize()
    assert sel[0].tolist() == [1, 2, 4, 0, 5]
    assert margin[0].item() == 0.0


@pytest.mark.parametrize("T,k,E,seed", [(1, 2, 8, 0), (32, 2, 8, 1), (96, 4, 60, 2), (1024, 6, 64, 3), (2048, 6, 64, 4),
                                        (517, 2, 8, 5), (333, 16, 256, 6), (1500, 1, 3, 7)])
def test_op_permute(B, T, k, E, seed):
    from oracle.permute import permutation
    g = torch.Generator().manual_seed(seed)
    # distinct experts per token; skewed so that some groups are empty and some are large
    scores = torch.rand(T, E, generator=g) + (torch.arange(E) % 5 == 0).float() * 0.5
    if E > 4:
        scores[:, 3] = -1.0        # expert 3 never selected → empty group
    sel = torch.topk(scores, k, dim=1).indices.to(torch.int32)
    sd = sel.cuda()
    count = torch.empty(E, dtype=torch.int32, device="cuda"); offset = torch.empty(E + 1, dtype=torch.int32, device="cuda")
    perm = torch.full((T * k,), -7, dtype=torch.int32, device="cuda"); inv = torch.full((T * k,), -7, dtype=torch.int32, device="cuda")
    assert B.lib().promoe_op_permute(sd.data_ptr(), T, k, E, count.data_ptr(), offset.data_ptr(), perm.data_ptr(),
                                     inv.data_ptr(), None) == 0
    torch.cuda.synchronize()
    c, o, p, i = permutation(sel.tolist(), E)
    assert count.tolist() == c and offset.tolist() == o
    assert perm.tolist() == p and inv.tolist() == i


@pytest.mark.parametrize("wdtype", [0, 1])
@pytest.mark.parametrize("T,H,I,path", [(1, 256, 512, 1), (1, 2048, 1408, 1), (37, 256, 512, 2), (130, 2048, 1408, 2),
                                        (1, 4096, 14336, 1)])
def test_op_expert_ffn(B, wdtype, T, H, I, path):
    from oracle.forward import swiglu_ffn
    dt = torch.float32 if wdtype == 0 else torch.bfloat16
    x = _w((T, H), torch.float32, 7, 1.0)
    wg, wu, wdn = _w((I, H), dt, 8), _w((I, H), dt, 9), _w((H, I), dt, 10)
    xd, wgd, wud, wdd = x.cuda(), wg.cuda(), wu.cuda(), wdn.cuda()
    act = torch.empty((T, I), device="cuda"); y = torch.full((T, H), float("nan"), device="cuda")
    ws = torch.zeros(64, dtype=torch.uint8, device="cuda")
    rc = B.lib().promoe_op_expert_ffn(xd.data_ptr(), wgd.data_ptr(), wud.data_ptr(), wdd.data_ptr(), act.data_ptr(),
                                      y.data_ptr(), ws.data_ptr(), T, H, I, wdtype, path, 0, None)
    assert rc == 0
    torch.cuda.synchronize()
    ref = swiglu_ffn(x.double(), wg, wu, wdn)
    err = (y.cpu().double() - ref).abs().max().item()
    assert err <= 2e-4 * max(1.0, ref.abs().max().item()), err


def test_bad_arguments(B):
    L = B.lib()
    assert L.promoe_op_linear(None, None, None, 1, 1, 8, 0, 0, None) == B.PROMOE_EINVAL
    assert L.promoe_op_permute(None, 1, 1, 1, None, None, None, None, None) == B.PROMOE_EINVAL
    sh = B.promoe_shape_t(n_layers=2, hidden=250, n_q_heads=4, n_kv_heads=4, head_dim=64, vocab=10, max_seq=8,
                          n_experts=8, top_k=2, expert_inter=512, pred_hidden=128, wdtype=0)
    with pytest.raises(B.PromoeError) as e:
        B.promoe_create(sh, B.promoe_opts_t(cache_slots=8, stride=1))
    assert e.value.code == B.PROMOE_EINVAL
    sh.hidden = 256
    with pytest.raises(B.PromoeError):
        B.promoe_create(sh, B.promoe_opts_t(cache_slots=7, stride=1))      # not a multiple of n_moe_layers
    with pytest.raises(B.PromoeError):
        B.promoe_create(sh, B.promoe_opts_t(cache_slots=2, stride=1))      # fewer slots per layer than top_k
    h = B.promoe_create(sh, B.promoe_opts_t(cache_slots=8, stride=1))
    with pytest.raises(B.PromoeError) as e:
        B.promoe_decode(h, 0, None)                                         # decode before load
    assert e.value.code == B.PROMOE_ESTATE
    B.promoe_destroy(h)


# ---- tcgen05 / TMEM / TMA path (bf16 weights, activations as a bf16 hi/lo pair; G1) ---------------------
@pytest.mark.parametrize("T,N,K", [(64, 128, 64), (1, 128, 128), (5, 60, 2048), (130, 6144, 2048), (97, 200, 264),
                                   (512, 2048, 1408), (63, 512, 2048)])
def test_op_linear_tcgen05(B, T, N, K):
    x = _w((T, K), torch.float32, 11, 1.0)
    w = _w((N, K), torch.bfloat16, 12)
    xd, wd = x.cuda(), w.cuda()
    y = torch.full((T, N), float("nan"), device="cuda")
    rc = B.lib().promoe_op_linear(xd.data_ptr(), wd.data_ptr(), y.data_ptr(), T, N, K, 1, 3, None)
    assert rc == 0
    torch.cuda.synchronize()
    ref = x.double() @ w.double().T
    err = (y.cpu().double() - ref).abs().max().item()
    # hi/lo split: |x - hi - lo| <= 2^-17 |x| per element → ~1e-5 relative on the dot product
    assert err <= 1e-4 * max(1.0, ref.abs().max().item()), err


@pytest.mark.parametrize("T,H,I", [(37, 256, 512), (130, 2048, 1408), (64, 4096, 14336), (1, 256, 512)])
def test_op_expert_ffn_tcgen05(B, T, H, I):
    from oracle.forward import swiglu_ffn
    x = _w((T, H), torch.float32, 7, 1.0)
    wg, wu, wdn = _w((I, H), torch.bfloat16, 8), _w((I, H), torch.bfloat16, 9), _w((H, I), torch.bfloat16, 10)
    xd, wgd, wud, wdd = x.cuda(), wg.cuda(), wu.cuda(), wdn.cuda()
    act = torch.empty((T, I), device="cuda"); y = torch.full((T, H), float("nan"), device="cuda")
    ws = torch.zeros(64, dtype=torch.uint8, device="cuda")
    rc = B.lib().promoe_op_expert_ffn(xd.data_ptr(), wgd.data_ptr(), wud.data_ptr(), wdd.data_ptr(), act.data_ptr(),
                                      y.data_ptr(), ws.data_ptr(), T, H, I, 1, 3, 0, None)
    assert rc == 0
    torch.cuda.synchronize()
    ref = swiglu_ffn(x.double(), wg, wu, wdn)
    err = (y.cpu().double() - ref).abs().max().item()
    assert err <= 2e-4 * max(1.0, ref.abs().max().item()), err


# ---- A2 + A3: RoPE + KV append + attention, op level, against OracleModel._attention -------------------------------
@pytest.mark.parametrize("nq,nkv,d,T0,n_dec", [(4, 4, 64, 70, 3),          # c1 head shape, two query tiles
                                               (16, 16, 128, 900, 4),      # c2/c3 heads; decode beyond 768 positions (multi-round key loop)
                                               (8, 2, 128, 2110, 3),       # GQA (c4 ratio); decode at positions 2110+ (c5's longest prompts)
                                               (4, 4, 128, 1, 2)])         # T0 = 1: a one-token prefill, then decode at positions 1, 2
def test_op_attention(B, nq, nkv, d, T0, n_dec):
    """promoe_op_attention against the oracle's attention block: a T0-token causal prefill (several 64-row query tiles, a
    ragged tail), then n_dec single-token steps through the fused decode kernel at positions T0, T0+1, ... — the paths
    bench.py's prompt lengths reach (position > 768: the carried-(m, l) multi-round loop of the decode kernel)."""
    import types
    from oracle.forward import OracleModel
    H = nq * d
    qkv_w = (nq + 2 * nkv) * d
    max_seq = T0 + n_dec
    wqkv = _w((qkv_w, H), torch.float32, 31)
    shape = types.SimpleNamespace(n_q_heads=nq, n_kv_heads=nkv, head_dim=d, n_layers=1, n_experts=1, rope_theta=10000.0)
    weights = types.SimpleNamespace(shape=shape, dense={"l0.wqkv": wqkv, "l0.wo": torch.eye(H)})
    ora = OracleModel(weights)
    half = d // 2
    ang = torch.arange(max_seq, dtype=torch.float64)[:, None] * (10000.0 ** (-2.0 * torch.arange(half, dtype=torch.float64) / d))[None, :]
    cos_t, sin_t = torch.cos(ang).float().cuda(), torch.sin(ang).float().cuda()
    kc = torch.zeros(nkv, max_seq, d, device="cuda"); vc = torch.zeros(nkv, max_seq, d, device="cuda")
    ws = torch.zeros(nq * 16 * (d + 2), device="cuda"); cnt = torch.zeros(nq, dtype=torch.int32, device="cuda")
    L = B.lib()
    pos = 0
    for step, T in enumerate([T0] + [1] * n_dec):
        u1 = _w((T, H), torch.float32, 40 + step, 1.0)
        qkv = (u1.double() @ wqkv.double().T).float().cuda()        # the projection is not under test here
        out = torch.full((T, H), float("nan"), device="cuda")
        rc = L.promoe_op_attention(qkv.data_ptr(), cos_t.data_ptr(), sin_t.data_ptr(), kc.data_ptr(), vc.data_ptr(),
                                   out.data_ptr(), ws.data_ptr(), cnt.data_ptr(), T, pos, nq, nkv, d, max_seq, None)
        assert rc == 0
        torch.cuda.synchronize()
        ref = ora._attention(0, u1.double())
        ora.pos += T
        pos += T
        err = (out.cpu().double() - ref).abs().max().item()
        assert err <= 2e-5 * max(1.0, ref.abs().max().item()), (step, err)
        assert int(cnt.abs().sum()) == 0                             # the arrival counters are left zero
    # the cache holds the rotated keys / raw values of every position
    kref = torch.stack([ora.kcache[0][:, g, :] for g in range(nkv)])
    assert (kc[:, :pos].cpu().double() - kref).abs().max().item() <= 1e-5 * max(1.0, kref.abs().max().item())
    assert L.promoe_op_attention(qkv.data_ptr(), cos_t.data_ptr(), sin_t.data_ptr(), kc.data_ptr(), vc.data_ptr(), out.data_ptr(),
                                 ws.data_ptr(), cnt.data_ptr(), 1, max_seq, nq, nkv, d, max_seq, None) == B.PROMOE_EINVAL


# ---- A9 with INT4 group-quantised experts (format DESIGN.md G18) ---------------------------------------
@pytest.mark.parametrize("H,I", [(256, 512), (2048, 1408), (4096, 14336), (128, 128)])
def test_op_expert_ffn_int4(B, H, I):
    """promoe_op_expert_ffn with wdtype 2 (decode GEMVs that dequantise in registers) against the oracle's
    dequantise-then-fp64 FFN on the same packed image; K = 1408 has a ragged last pass, K = 14336 many passes."""
    from oracle.forward import swiglu_ffn
    from oracle.quant import dequant_expert
    from synth.weights import pack_int4
    mats = [_w((I, H), torch.float32, 8), _w((I, H), torch.float32, 9), _w((H, I), torch.float32, 10)]
    packed = [pack_int4(m) for m in mats]
    img = torch.cat([c.reshape(-1) for c, _ in packed] + [s.contiguous().view(torch.uint8).reshape(-1) for _, s in packed])
    assert img.numel() == 3 * H * I * 33 // 64
    x = _w((1, H), torch.float32, 7, 1.0)
    xd, imgd = x.cuda(), img.cuda()
    act = torch.empty((1, I), device="cuda"); y = torch.full((1, H), float("nan"), device="cuda")
    ws = torch.zeros(64, dtype=torch.uint8, device="cuda")
    rc = B.lib().promoe_op_expert_ffn(xd.data_ptr(), imgd.data_ptr(), None, None, act.data_ptr(), y.data_ptr(), ws.data_ptr(),
                                      1, H, I, 2, 1, 0, None)
    assert rc == 0
    torch.cuda.synchronize()
    wg, wu, wd = dequant_expert(img, H, I)
    ref = swiglu_ffn(x.double(), wg, wu, wd)
    err = (y.cpu().double() - ref).abs().max().item()
    assert err <= 2e-4 * max(1.0, ref.abs().max().item()), err
    assert B.lib().promoe_op_expert_ffn(xd.data_ptr(), imgd.data_ptr(), None, None, act.data_ptr(), y.data_ptr(), ws.data_ptr(),
                                        1, H + 64, I, 2, 1, 0, None) == B.PROMOE_EINVAL       # not a multiple of the group
