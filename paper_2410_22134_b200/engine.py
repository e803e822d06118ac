"""`ProMoE` — a thin handle around the C-ABI for a model whose weights come from `synth.make_weights`.

PyTorch is used for device memory only (dense tensors are moved to the GPU with `.cuda()`, the routed experts stay
in the pinned host tensor); every step of the path runs inside libpromoe.so.
"""
from __future__ import annotations

import ctypes as C
from typing import Dict, List, Optional

import numpy as np
import torch

from . import binding as B


def shape_struct(s) -> B.promoe_shape_t:
    """synth.Shape → promoe_shape_t (field names are identical)."""
    st = B.promoe_shape_t()
    for name, _ in B.promoe_shape_t._fields_:
        setattr(st, name, getattr(s, name))
    return st


class ProMoE:
    def __init__(self, weights, cache_slots: int, stride: int = 1, chunk_bytes: int = 0,
                 predictor_mode: int = B.PRED_MLP, flags: int = B.F_PREEMPT | B.F_REORDER | B.F_WARM | B.F_TRACE,
                 max_inflight: int = 0, high_group: int = 0, max_spec_decode: int = 0, max_spec_prefill: int = 0,
                 low_cap_chunks: int = 0, fetch_ctas: int = 0, max_batch: int = 1, static_slots: int = 0, device: str = "cuda:0"):
        if not torch.cuda.is_available():
            raise RuntimeError("ProMoE needs a CUDA device (there is no CPU fallback)")
        B.lib()
        self.w = weights
        self.s = weights.shape
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        s = self.s
        self.n_moe = s.n_layers - s.n_dense_layers
        self.slots_per_layer = cache_slots // self.n_moe
        self.stride = stride
        opts = B.promoe_opts_t(cache_slots=cache_slots, stride=stride, chunk_bytes=chunk_bytes,
                               predictor_mode=predictor_mode, flags=flags, max_inflight=max_inflight, high_group=high_group,
                               max_spec_decode=max_spec_decode, max_spec_prefill=max_spec_prefill,
                               low_cap_chunks=low_cap_chunks, fetch_ctas=fetch_ctas,
                               compute_stream=None, max_batch=max_batch, static_slots=static_slots)
        self.max_batch = max_batch
        self.h = B.promoe_create(shape_struct(s), opts)
        # dense parameters → device (borrowed by the library; kept alive here)
        self._dev: Dict[str, torch.Tensor] = {k: v.to(self.device).contiguous() for k, v in weights.dense.items()}
        self._keep: List[object] = []
        d = B.promoe_dense_t()
        d.emb = self._dev["emb"].data_ptr()
        d.lm_head = self._dev["lm_head"].data_ptr()
        d.final_norm = self._dev["final_norm"].data_ptr()

        def per_layer(name: str):
            arr = (C.c_void_p * s.n_layers)()
            for l in range(s.n_layers):
                t = self._dev.get(f"l{l}.{name}")
                arr[l] = t.data_ptr() if t is not None else None
            self._keep.append(arr)
            return C.cast(arr, C.POINTER(C.c_void_p))

        for name in ("ln1", "ln2", "wqkv", "wo", "router", "router_bias", "pred_w1", "pred_w2", "ffn_gate", "ffn_up",
                     "ffn_down", "shared_gate_w"):
            setattr(d, name, per_layer(name))
        B.promoe_load_dense(self.h, d)
        ex = weights.experts
        assert ex.is_contiguous() and ex.device.type == "cpu"
        self.expert_bytes = ex.shape[2] * ex.element_size()
        base = ex.data_ptr()
        ptrs = [base + (m * s.n_experts + e) * self.expert_bytes for m in range(self.n_moe) for e in range(s.n_experts)]
        B.promoe_load_experts(self.h, ptrs, self.expert_bytes)
        self._logits = np.empty(s.vocab, dtype=np.float32)
        self._blogits = np.empty((max(1, max_batch), s.vocab), dtype=np.float32)

    # ---- steps ----------------------------------------------------------------------------------------------
    def prefill(self, ids, want_logits: bool = True) -> Optional[np.ndarray]:
        ids = np.ascontiguousarray(np.asarray(ids, dtype=np.int32))
        B.promoe_prefill(self.h, ids, self._logits if want_logits else None)
        return self._logits.copy() if want_logits else None

    def decode(self, token_id: int, want_logits: bool = True) -> Optional[np.ndarray]:
        B.promoe_decode(self.h, int(token_id), self._logits if want_logits else None)
        return self._logits.copy() if want_logits else None

    def prefill_seq(self, seq: int, ids, want_logits: bool = True) -> Optional[np.ndarray]:
        ids = np.ascontiguousarray(np.asarray(ids, dtype=np.int32))
        B.promoe_prefill_seq(self.h, seq, ids, self._logits if want_logits else None)
        return self._logits.copy() if want_logits else None

    def decode_batch(self, seqs, token_ids, want_logits: bool = True) -> Optional[np.ndarray]:
        """One new token for each sequence in `seqs`; returns logits [len(seqs), vocab]."""
        n = len(seqs)
        out = self._blogits[:n]
        B.promoe_decode_batch(self.h, np.asarray(seqs, dtype=np.int32), np.asarray(token_ids, dtype=np.int32), out if want_logits else None)
        return out.copy() if want_logits else None

    def set_prediction_trace(self, lists: List[Optional[List[int]]]) -> None:
        E = self.s.n_experts
        buf = np.zeros((self.n_moe, 1 + E), dtype=np.int32)
        for m, lst in enumerate(lists):
            if lst:
                buf[m, 0] = len(lst)
                buf[m, 1:1 + len(lst)] = lst
        B.promoe_set_prediction_trace(self.h, buf)

    def reset(self) -> None:
        B.promoe_reset(self.h)

    def stats(self) -> Dict[str, float]:
        return B.promoe_stats(self.h).as_dict()

    def slots(self, m: int) -> np.ndarray:
        return B.promoe_get_slots(self.h, m, self.slots_per_layer)

    # ---- traces of the last step --------------------------------------------------------------------------
    def trace(self, T: int) -> Dict[str, np.ndarray]:
        s, Lm, k, E = self.s, self.n_moe, self.s.top_k, self.s.n_experts
        out = {
            "sel": B.promoe_get_trace(self.h, B.TRACE_SEL, np.int32).reshape(Lm, T, k),
            "gates": B.promoe_get_trace(self.h, B.TRACE_GATES, np.float32).reshape(Lm, T, k),
            "margin": B.promoe_get_trace(self.h, B.TRACE_MARGIN, np.float32).reshape(Lm, T),
            "z": B.promoe_get_trace(self.h, B.TRACE_ZLOGITS, np.float32).reshape(Lm, T, E),
            "precise": B.promoe_get_trace(self.h, B.TRACE_PRECISE, np.int32).reshape(Lm, 1 + 5 * E),
            "pred": B.promoe_get_trace(self.h, B.TRACE_PRED, np.int32).reshape(Lm, 1 + 4 * E),
            "predlist": B.promoe_get_trace(self.h, B.TRACE_PREDLIST, np.int32).reshape(Lm, 1 + E),
            "hidden": B.promoe_get_trace(self.h, B.TRACE_HIDDEN, np.float32).reshape(T, s.hidden),
        }
        if T > 1:
            out["perm"] = B.promoe_get_trace(self.h, B.TRACE_PERM, np.int32).reshape(Lm, 2 * E + 1 + 2 * T * k)
        return out

    def close(self) -> None:
        if self.h is not None:
            B.promoe_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
