"""ctypes binding of include/promoe.h — argument marshalling only; every step of the path runs in libpromoe.so.

Same names as the C-ABI (promoe_create, promoe_load_dense, promoe_load_experts, promoe_prefill, promoe_decode,
promoe_stats, ...).  The library is built in-tree by `python -m paper_2410_22134_b200.build`; if it is missing the
import fails loudly — there is no CPU fallback.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpromoe.so")

PROMOE_OK, PROMOE_EINVAL, PROMOE_ENOMEM, PROMOE_ECUDA, PROMOE_ESTATE, PROMOE_ETIMEOUT = 0, -1, -2, -3, -4, -5
PRED_NONE, PRED_MLP, PRED_TRACE = 0, 1, 2
F_PREEMPT, F_REORDER, F_WARM, F_TRACE, F_TENSOR, F_NOFUSE = 1, 2, 4, 8, 16, 32
F_UNCHUNKED, F_DEMOTE, F_TRACE_U = 64, 128, 256
TRACE_SEL, TRACE_GATES, TRACE_MARGIN, TRACE_PERM, TRACE_PRECISE, TRACE_PRED, TRACE_HIDDEN, TRACE_PREDLIST, TRACE_ZLOGITS, TRACE_U = range(10)

EXPORTS = [
    "promoe_create", "promoe_destroy", "promoe_last_error", "promoe_load_dense", "promoe_load_experts",
    "promoe_prefill", "promoe_decode", "promoe_set_prediction_trace", "promoe_stats", "promoe_get_trace",
    "promoe_reset", "promoe_get_slots", "promoe_op_linear", "promoe_op_route",
    "promoe_op_permute", "promoe_op_expert_ffn", "promoe_op_expert_ffn_static", "promoe_op_expert_ffn_static_max_inter",
    "promoe_op_attention", "promoe_prefill_seq", "promoe_decode_batch",
]
BENCH_EXPORTS = ["promoe_bench_h2d", "promoe_bench_kernel_time"]   # include/promoe_bench.h (bench.py only)


class promoe_shape_t(C.Structure):
    _fields_ = [(n, C.c_int32) for n in (
        "n_layers", "hidden", "n_q_heads", "n_kv_heads", "head_dim", "vocab", "max_seq", "n_experts", "top_k",
        "expert_inter", "n_shared_inter", "shared_gate", "n_dense_layers", "dense_inter", "router_bias",
        "pred_hidden", "wdtype")] + [("rope_theta", C.c_float), ("rms_eps", C.c_float)]


class promoe_opts_t(C.Structure):
    _fields_ = [("cache_slots", C.c_int32), ("stride", C.c_int32), ("chunk_bytes", C.c_uint64),
                ("predictor_mode", C.c_int32), ("flags", C.c_int32), ("max_inflight", C.c_int32),
                ("high_group", C.c_int32), ("max_spec_decode", C.c_int32), ("max_spec_prefill", C.c_int32),
                ("low_cap_chunks", C.c_int32), ("fetch_ctas", C.c_int32),
                ("compute_stream", C.c_void_p), ("max_batch", C.c_int32), ("static_slots", C.c_int32)]


class promoe_dense_t(C.Structure):
    _fields_ = [("emb", C.c_void_p), ("lm_head", C.c_void_p), ("final_norm", C.c_void_p)] + [
        (n, C.POINTER(C.c_void_p)) for n in (
            "ln1", "ln2", "wqkv", "wo", "router", "router_bias", "pred_w1", "pred_w2", "ffn_gate", "ffn_up",
            "ffn_down", "shared_gate_w")]


class promoe_stats_t(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in (
        "steps", "tokens", "accesses", "hits_resident", "hits_prefetch", "misses", "evictions", "predicted",
        "predicted_correct", "pred_allocs", "need_experts", "chunks_issued", "chunks_cancelled", "chunks_high",
        "chunks_low", "h2d_bytes", "fetched_at_gate", "fetched_at_gate_of", "registered_host_bytes",
        "kernel_launches", "high_bytes", "low_bytes", "low_bytes_useful", "hits_landed", "owed_bytes_at_gate",
        "landed_chunks_at_gate", "landed_chunks_of")] + [
        ("copy_busy_ms", C.c_double), ("step_ms", C.c_double), ("last_step_ms", C.c_double),
        ("timeouts", C.c_int32), ("reserved", C.c_int32)]

    def as_dict(self) -> Dict[str, float]:
        return {n: getattr(self, n) for n, _ in self._fields_ if n != "reserved"}


class PromoeError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"promoe error {code}: {msg}")
        self.code = code


_lib: Optional[C.CDLL] = None


def lib() -> C.CDLL:
    """Load libpromoe.so (fails loudly when the CUDA extension has not been built)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2410_22134_b200.build` (no CPU fallback exists)")
    L = C.CDLL(LIB_PATH)
    vp, i32, u64, sz = C.c_void_p, C.c_int32, C.c_uint64, C.c_size_t
    L.promoe_create.argtypes = [C.POINTER(promoe_shape_t), C.POINTER(promoe_opts_t), C.POINTER(vp)]
    L.promoe_destroy.argtypes = [vp]; L.promoe_destroy.restype = None
    L.promoe_last_error.argtypes = [vp]; L.promoe_last_error.restype = C.c_char_p
    L.promoe_load_dense.argtypes = [vp, C.POINTER(promoe_dense_t)]
    L.promoe_load_experts.argtypes = [vp, C.POINTER(vp), sz]
    L.promoe_prefill.argtypes = [vp, vp, i32, vp]
    L.promoe_decode.argtypes = [vp, i32, vp]
    L.promoe_prefill_seq.argtypes = [vp, i32, vp, i32, vp]
    L.promoe_decode_batch.argtypes = [vp, i32, vp, vp, vp]
    L.promoe_set_prediction_trace.argtypes = [vp, vp, sz]
    L.promoe_stats.argtypes = [vp, C.POINTER(promoe_stats_t)]
    L.promoe_get_trace.argtypes = [vp, C.c_int, C.POINTER(vp), C.POINTER(sz)]
    L.promoe_reset.argtypes = [vp]
    L.promoe_get_slots.argtypes = [vp, i32, vp]
    L.promoe_bench_h2d.argtypes = [sz, i32, i32, C.POINTER(C.c_double)]
    L.promoe_op_linear.argtypes = [vp, vp, vp, i32, i32, i32, i32, i32, vp]
    L.promoe_op_route.argtypes = [vp, vp, vp, i32, i32, i32, i32, i32, vp, vp, vp, vp, vp]
    L.promoe_op_permute.argtypes = [vp, i32, i32, i32, vp, vp, vp, vp, vp]
    L.promoe_op_expert_ffn.argtypes = [vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, i32, vp]
    L.promoe_op_attention.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, i32, vp]
    L.promoe_op_expert_ffn_static.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, vp]
    L.promoe_op_expert_ffn_static_max_inter.argtypes = []
    L.promoe_bench_kernel_time.argtypes = [vp, i32, i32, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    for n in EXPORTS + BENCH_EXPORTS:
        f = getattr(L, n)
        if n not in ("promoe_destroy", "promoe_last_error"):
            f.restype = C.c_int
    _lib = L
    return L


def _check(rc: int, h=None) -> None:
    if rc != PROMOE_OK:
        msg = lib().promoe_last_error(h)
        raise PromoeError(rc, msg.decode() if msg else "")


# ---- thin wrappers, same names as the C-ABI ------------------------------------------------------------------
def promoe_create(shape: promoe_shape_t, opts: promoe_opts_t) -> C.c_void_p:
    h = C.c_void_p()
    _check(lib().promoe_create(C.byref(shape), C.byref(opts), C.byref(h)))
    return h


def promoe_destroy(h) -> None:
    lib().promoe_destroy(h)


def promoe_load_dense(h, dense: promoe_dense_t) -> None:
    _check(lib().promoe_load_dense(h, C.byref(dense)), h)


def promoe_load_experts(h, host_ptrs: Sequence[int], expert_bytes: int) -> None:
    arr = (C.c_void_p * len(host_ptrs))(*host_ptrs)
    _check(lib().promoe_load_experts(h, arr, expert_bytes), h)


def promoe_prefill(h, ids: np.ndarray, logits_out: Optional[np.ndarray]) -> None:
    ids = np.ascontiguousarray(ids, dtype=np.int32)
    _check(lib().promoe_prefill(h, ids.ctypes.data, ids.size, logits_out.ctypes.data if logits_out is not None else None), h)


def promoe_decode(h, token_id: int, logits_out: Optional[np.ndarray]) -> None:
    _check(lib().promoe_decode(h, int(token_id), logits_out.ctypes.data if logits_out is not None else None), h)


def promoe_prefill_seq(h, seq: int, ids: np.ndarray, logits_out: Optional[np.ndarray]) -> None:
    ids = np.ascontiguousarray(ids, dtype=np.int32)
    _check(lib().promoe_prefill_seq(h, int(seq), ids.ctypes.data, ids.size, logits_out.ctypes.data if logits_out is not None else None), h)


def promoe_decode_batch(h, seqs: np.ndarray, token_ids: np.ndarray, logits_out: Optional[np.ndarray]) -> None:
    seqs = np.ascontiguousarray(seqs, dtype=np.int32)
    token_ids = np.ascontiguousarray(token_ids, dtype=np.int32)
    assert seqs.size == token_ids.size
    _check(lib().promoe_decode_batch(h, seqs.size, seqs.ctypes.data, token_ids.ctypes.data,
                                     logits_out.ctypes.data if logits_out is not None else None), h)


def promoe_set_prediction_trace(h, pred: np.ndarray) -> None:
    pred = np.ascontiguousarray(pred, dtype=np.int32)
    _check(lib().promoe_set_prediction_trace(h, pred.ctypes.data, pred.size), h)


def promoe_stats(h) -> promoe_stats_t:
    st = promoe_stats_t()
    _check(lib().promoe_stats(h, C.byref(st)), h)
    return st


def promoe_get_trace(h, which: int, dtype) -> np.ndarray:
    data, nbytes = C.c_void_p(), C.c_size_t()
    _check(lib().promoe_get_trace(h, which, C.byref(data), C.byref(nbytes)), h)
    buf = (C.c_char * nbytes.value).from_address(data.value)
    return np.frombuffer(buf, dtype=dtype).copy()


def promoe_reset(h) -> None:
    _check(lib().promoe_reset(h), h)


def promoe_get_slots(h, moe_layer: int, n_slots: int) -> np.ndarray:
    out = np.empty(n_slots, dtype=np.int32)
    _check(lib().promoe_get_slots(h, moe_layer, out.ctypes.data), h)
    return out


def promoe_bench_h2d(nbytes: int, depth: int = 2, reps: int = 5) -> float:
    g = C.c_double()
    _check(lib().promoe_bench_h2d(nbytes, depth, reps, C.byref(g)))
    return g.value


def promoe_bench_kernel_time(h, which: int, reps: int = 200):
    """(average launch ms, algorithmic bytes per launch) of decode kernel `which` over resident slots."""
    ms, nb = C.c_double(), C.c_double()
    _check(lib().promoe_bench_kernel_time(h, which, reps, C.byref(ms), C.byref(nb)), h)
    return ms.value, nb.value
