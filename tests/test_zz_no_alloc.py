"""-m gpu: promoe_op_expert_ffn_static — the batch-1 expert FFN for callers that may not allocate (scratch in a
file-scope device array of libpromoe.so, csrc/op_static.cu) — against the existing caller-scratch entry point
promoe_op_expert_ffn (path 1) and the CPU oracle, on two calls in a row (the array keeps the previous call's contents).

Collected last (file name): the suite runs with pytest -x.
"""
from __future__ import annotations

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
    t = torch.randn(shape, generator=g, dtype=torch.float32)
    return (t * (std if std is not None else shape[-1] ** -0.5)).to(dtype)


def _existing(B, x, wg, wu, wd, H, I, wdtype):
    act = torch.empty(I, device="cuda")
    y = torch.full((H,), float("nan"), device="cuda")
    ws = torch.zeros(64, dtype=torch.uint8, device="cuda")
    assert B.lib().promoe_op_expert_ffn(x.data_ptr(), wg.data_ptr(), wu.data_ptr(), wd.data_ptr(), act.data_ptr(),
                                        y.data_ptr(), ws.data_ptr(), 1, H, I, wdtype, 1, 0, None) == 0
    torch.cuda.synchronize()
    return y


@pytest.mark.parametrize("wdtype", [0, 1])
def test_static_scratch_matches_existing_path_twice(B, wdtype):
    from oracle.forward import swiglu_ffn
    L = B.lib()
    dt = torch.float32 if wdtype == 0 else torch.bfloat16
    # two calls in a row with DIFFERENT shapes and inputs: the second one finds the first one's activations (a longer
    # vector) and record in the shared array
    cases = [(2048, 1408, 21), (256, 512, 33)]
    for H, I, seed in cases:
        x = _w((H,), torch.float32, seed, 1.0)
        wg, wu, wdn = _w((I, H), dt, seed + 1), _w((I, H), dt, seed + 2), _w((H, I), dt, seed + 3)
        xd, wgd, wud, wdd = x.cuda(), wg.cuda(), wu.cuda(), wdn.cuda()
        y = torch.full((H,), float("nan"), device="cuda")
        rc = L.promoe_op_expert_ffn_static(xd.data_ptr(), wgd.data_ptr(), wud.data_ptr(), wdd.data_ptr(), y.data_ptr(),
                                           H, I, wdtype, None)
        assert rc == 0
        torch.cuda.synchronize()
        ref_gpu = _existing(B, xd, wgd, wud, wdd, H, I, wdtype)
        assert torch.equal(y, ref_gpu)                          # same kernels, same order: bit-identical
        ref = swiglu_ffn(x.double().view(1, H), wg, wu, wdn).view(H)
        err = (y.cpu().double() - ref).abs().max().item()
        assert err <= 2e-4 * max(1.0, ref.abs().max().item()), err


def test_static_scratch_limits(B):
    L = B.lib()
    mx = L.promoe_op_expert_ffn_static_max_inter()
    assert mx == 16384
    d = torch.zeros(16, device="cuda")
    p = d.data_ptr()
    assert L.promoe_op_expert_ffn_static(p, p, p, p, p, 256, mx + 16, 1, None) == B.PROMOE_EINVAL   # beyond the static scratch
    assert L.promoe_op_expert_ffn_static(None, p, p, p, p, 256, 512, 1, None) == B.PROMOE_EINVAL
    assert L.promoe_op_expert_ffn_static(p, p, p, p, p, 250, 512, 1, None) == B.PROMOE_EINVAL
    # the largest size the array admits (c4's expert is I = 14336 < 16384)
    H, I = 256, mx
    x = _w((H,), torch.float32, 5, 1.0).cuda()
    wg, wu, wdn = (_w((I, H), torch.bfloat16, 6).cuda(), _w((I, H), torch.bfloat16, 7).cuda(), _w((H, I), torch.bfloat16, 8).cuda())
    y = torch.full((H,), float("nan"), device="cuda")
    assert L.promoe_op_expert_ffn_static(x.data_ptr(), wg.data_ptr(), wu.data_ptr(), wdn.data_ptr(), y.data_ptr(), H, I, 1, None) == 0
    torch.cuda.synchronize()
    assert torch.equal(y, _existing(B, x, wg, wu, wdn, H, I, 1))
