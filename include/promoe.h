/* promoe.h — C-ABI of the B200-native ProMoE hot path (expert-offloaded MoE decoder step).
 *
 * Paper: arxiv 2410.22134 "ProMoE" (PAPER.md; P:NNN = its line NNN).  The five core calls follow
 * BASELINE.json `north_star`: promoe_create(model shape, cache_slots, stride), promoe_load_experts(host
 * ptrs), promoe_prefill, promoe_decode, promoe_stats.  The remaining calls hand over the always-resident
 * non-expert parameters ("non-expert parameters are always kept on the GPU"), expose traces for
 * parity tests, and micro-entry points for single hot-path steps.  Measurement hooks used only by bench.py live in
 * include/promoe_bench.h, not here.
 *
 * Conventions
 *  - every call returns 0 (PROMOE_OK) or a negative PROMOE_E* code; no exception or abort crosses the ABI;
 *    promoe_last_error() returns a static/handle-owned message for the last failing call.
 *  - one handle = one model instance on the CUDA device that is current at promoe_create; calls on one
 *    handle are not thread-safe.
 *  - "device ptr" = CUDA device memory, "host ptr" = ordinary host memory, "pinned host ptr" = page-locked
 *    host memory (the library cudaHostRegister()s unpinned expert buffers and counts that in the stats).
 *  - borrowed pointers (dense weights, expert host images) must outlive the handle; the library owns the
 *    slot region (ONE contiguous allocation), KV cache, traces, streams and events.
 *  - weights are row-major [out_features, in_features]; bf16 (wdtype 1) or fp32 (wdtype 0); all
 *    activations, the KV cache and accumulators are fp32 (reading G1).
 */
#ifndef PROMOE_H
#define PROMOE_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define PROMOE_API __attribute__((visibility("default")))
#else
#define PROMOE_API
#endif

#define PROMOE_OK 0
#define PROMOE_EINVAL (-1)   /* bad argument / unsupported shape */
#define PROMOE_ENOMEM (-2)   /* device or host allocation failed */
#define PROMOE_ECUDA (-3)    /* a CUDA call or kernel failed; see promoe_last_error */
#define PROMOE_ESTATE (-4)   /* call out of order (e.g. decode before load) or sequence overflow */
#define PROMOE_ETIMEOUT (-5) /* an expert kernel gave up waiting for a chunk-ready flag */

typedef struct promoe promoe_t;

/* "model shape" (BASELINE.json configs; Table 1 P:39-48 names the families). */
typedef struct {
  int32_t n_layers, hidden, n_q_heads, n_kv_heads, head_dim, vocab, max_seq;
  int32_t n_experts, top_k, expert_inter;
  int32_t n_shared_inter;  /* 0 = no shared expert; c2 5632; c3 2816 (two always-on experts = one MLP) */
  int32_t shared_gate;     /* 1 = sigmoid scalar gate on the shared expert (c2) */
  int32_t n_dense_layers;  /* leading layers with a dense FFN (c3: 1) */
  int32_t dense_inter;
  int32_t router_bias;     /* 1 = per-expert logit bias (c3) */
  int32_t pred_hidden;     /* predictor MLP hidden width ("2-layer MLP") */
  int32_t wdtype;          /* 0 fp32 (c1), 1 bf16, 2 = bf16 dense weights + INT4 group-quantised routed experts:
                              per matrix 4-bit codes (two per byte, even element in the low nibble) then, behind the three code
                              blocks, one bf16 scale per 128 consecutive elements of a row; value = (code - 8) * scale; image =
                              [gate codes | up codes | down codes | gate scales | up scales | down scales] (G18) */
  float rope_theta, rms_eps;
} promoe_shape_t;

/* predictor_mode */
#define PROMOE_PRED_NONE 0   /* reactive cache, no prefetch (BASELINE.json config 5 baseline) */
#define PROMOE_PRED_MLP 1    /* learned stride predictor */
#define PROMOE_PRED_TRACE 2  /* injected prediction lists (oracle-routing upper bound) */
/* flags */
#define PROMOE_F_PREEMPT 1   /* early preemption: drop un-issued LOW chunks of a layer at its gate */
#define PROMOE_F_REORDER 2   /* reordered inference: cached -> being prefetched -> missing.  Clear = the ID-order baseline of
                                the ablation (Fig. 12 "Base"): experts in ascending id, classified at their turn, plain
                                LRU victim over all slots — a needed expert may be evicted before its turn (G16) */
#define PROMOE_F_WARM 4      /* warm start: experts 0..C-1 resident in every layer (G4) */
#define PROMOE_F_TRACE 8     /* record routing / permutation / cache traces for promoe_get_trace */
#define PROMOE_F_NOFUSE 32   /* decode with the unfused per-op kernels and copy-engine fills (19 launches per layer, host in the layer
                                loop) instead of the fused step on the device-side fetch worker */
#define PROMOE_F_TENSOR 16   /* prefill GEMMs on tcgen05 tensor cores (bf16 weights; INT4 experts through exact bf16 hi/lo staging
                                images); else SIMT fp32 */
#define PROMOE_F_DEMOTE 128  /* a predicted (PRED) slot whose expert its gate did not select gets the oldest LRU stamp at that gate: a
                                misprediction costs one LRU victim instead of a most-recently-used slot (G17; not in the
                                paper, which keeps mispredicted prefetches as ordinary cache entries) */
#define PROMOE_F_TRACE_U 256  /* also record u_l, the post-attention RMSNorm output the router and the predictor of every MoE layer
                                read (G6): PROMOE_TRACE_U — the input side of the predictor's offline training set */
#define PROMOE_F_UNCHUNKED 64 /* ablation (Fig. 12 "+chunk" off): an expert image is copied all or nothing — one LOW
                                 copy per predicted expert, and a gate that finds a partial image fetches it again from byte 0 */

typedef struct {
  int32_t cache_slots;     /* TOTAL slots; per MoE layer = cache_slots / n_moe_layers (must divide), G14 */
  int32_t stride;          /* predictor at MoE layer m targets MoE layer m+stride; >= 1 */
  uint64_t chunk_bytes;    /* chunk size: granularity of the per-chunk ready flags, of the LOW (predicted) copies and
                              of preemption.  0 = default 256 KiB (decode fetches on the device, where a chunk costs no host
                              call: DESIGN.md §6); multiple of 256.  Prefill (copy engines): a HIGH (precise) fill covers
                              high_group chunks per copy operation */
  int32_t predictor_mode;
  int32_t flags;
  int32_t max_inflight;    /* LOW (predicted) chunks in flight (P:191 bounded preemption delay).  Prefill / unfused decode (copy
                              engines): chunks kept on the copy stream, 0 = default 2.  Fused decode (device-side worker): the number
                              of fetch CTAs that copy LOW chunks, one chunk each at a time, 0 = default 1 */
  int32_t high_group;      /* chunks per HIGH (precise) copy operation; 0 = the whole remaining fill in ONE copy (measured
                              fastest); ready flags are written behind every operation */
  int32_t max_spec_decode; /* experts of one PushPredicted that may ALLOCATE a slot in a decode step (listed order = most
                              confident first); 0 = default top_k (all, as Alg. 2), < 0 = none (touch only) */
  int32_t max_spec_prefill;/* same for a prefill step (T > 1); <= 0 = default none: with 50-100 % of the experts needed
                               an allocation only swaps one needed expert for another (G7) */
  int32_t low_cap_chunks;  /* a LOW (predicted) fill stops after this many chunks; the rest is fetched only if the gate needs
                              the expert (then as HIGH).  0 = no cap.  Physical only: never changes a trace or an output */
  int32_t fetch_ctas;      /* CTAs (one warp each, TMA bulk copies) of the device-side fetch worker of the fused decode step;
                              0 = default 4 (three reach the SM-side link limit at any chunk size: profiles/r02_fill_probe.md).
                              < 0 = no worker: legal only when nothing is ever fetched (every expert resident) — for runs under
                              a profiler that serialises kernels; a needed fetch then ends in PROMOE_ETIMEOUT.  Physical only */
  void* compute_stream;    /* cudaStream_t owned by the caller (torch); NULL = library creates one */
  int32_t max_batch;       /* sequences the handle can hold (each with its own KV cache and position) for batched decode, P:381-413;
                              0 = 1.  promoe_prefill / promoe_decode work on sequence 0 */
  int32_t static_slots;    /* > 0: the "static" baseline of P:317 — slots [0, static_slots) of every layer never take an allocation
                              (with PROMOE_F_WARM they hold experts 0..static_slots-1 for good); the remaining slots are the staging
                              buffers (the paper uses two; here at least top_k must remain, so that one decode step never recycles a buffer:
                              static_slots <= slots per layer - top_k).  0 = an ordinary LRU cache */
} promoe_opts_t;

/* Device pointers to the always-resident parameters.  Per-layer arrays are HOST arrays of n_layers DEVICE
 * pointers (entries for layers that lack the tensor are NULL).  Norm gains and router bias are fp32; every
 * other tensor has the model's wdtype. */
typedef struct {
  const void* emb;         /* [vocab, hidden] */
  const void* lm_head;     /* [vocab, hidden] */
  const float* final_norm; /* [hidden] */
  const float* const* ln1; /* [hidden] pre-attention RMSNorm gain */
  const float* const* ln2; /* [hidden] pre-FFN RMSNorm gain */
  const void* const* wqkv; /* [(nq+2nkv)*d, hidden], rows: q heads | k heads | v heads */
  const void* const* wo;   /* [hidden, nq*d] */
  const void* const* router;        /* [E, hidden]  (MoE layers) */
  const float* const* router_bias;  /* [E] or NULL */
  const void* const* pred_w1;       /* [pred_hidden, hidden] (MoE layers) */
  const void* const* pred_w2;       /* [E, pred_hidden] */
  const void* const* ffn_gate;      /* shared expert (MoE layers) or dense FFN (dense layers): [I', hidden] */
  const void* const* ffn_up;        /* [I', hidden] */
  const void* const* ffn_down;      /* [hidden, I'] */
  const void* const* shared_gate_w; /* [1, hidden] or NULL */
} promoe_dense_t;

/* Cumulative since create / reset.  Logical counters follow DESIGN.md "logical-time cache"; physical
 * ones are measured on the copy stream. */
typedef struct {
  uint64_t steps, tokens;
  uint64_t accesses, hits_resident, hits_prefetch, misses;   /* class A / B / C at the gate */
  uint64_t evictions, predicted, predicted_correct, pred_allocs;
  uint64_t need_experts;        /* sum |needed \ resident at step start| (B_need / expert_bytes) */
  uint64_t chunks_issued, chunks_cancelled, chunks_high, chunks_low;
  uint64_t h2d_bytes;           /* bytes physically copied */
  uint64_t fetched_at_gate, fetched_at_gate_of;  /* FetchRate numerator / denominator */
  uint64_t registered_host_bytes; /* expert host bytes the library had to cudaHostRegister */
  uint64_t kernel_launches;     /* kernels launched by the library in this process so far (all handles) */
  /* byte-accurate (physical) view — the logical counters above follow the slot TABLE, these follow the BYTES */
  uint64_t high_bytes, low_bytes;     /* bytes moved by HIGH (precise) / LOW (predicted) copies; sum = h2d_bytes */
  uint64_t low_bytes_useful;          /* LOW bytes of fills whose expert was needed at its gate (class B) */
  uint64_t hits_landed;               /* class A / B accesses whose image had completely landed when the gate was processed */
  uint64_t owed_bytes_at_gate;        /* bytes the HIGH fills still had to move for the needed experts, summed over gates */
  uint64_t landed_chunks_at_gate, landed_chunks_of;   /* class-B experts: chunks landed at the gate / chunks per image
                                         (the partial-fetch form of FetchRate) */
  double copy_busy_ms;          /* copy-stream busy time, from per-chunk events */
  double step_ms;               /* sum of step times (compute-stream events) */
  double last_step_ms;
  int32_t timeouts;             /* kernels that gave up on a ready flag */
  int32_t reserved;
} promoe_stats_t;

/* trace kinds for promoe_get_trace (valid until the next step call; library-owned HOST memory) */
#define PROMOE_TRACE_SEL 0       /* int32 [n_moe, T, k]   selected experts, descending logit */
#define PROMOE_TRACE_GATES 1     /* float [n_moe, T, k]   renormalised gate weights */
#define PROMOE_TRACE_MARGIN 2    /* float [n_moe, T]      z_(k) - z_(k+1) */
#define PROMOE_TRACE_PERM 3      /* int32 [n_moe, E + (E+1) + 2*T*k]  count | offset | perm | inv */
#define PROMOE_TRACE_PRECISE 4   /* int32 [n_moe, 1 + 5*E]  n, then (expert, class, slot, victim, dep) in launch order */
#define PROMOE_TRACE_PRED 5      /* int32 [n_moe, 1 + 4*E]  n, then (expert, action, slot, victim) in listed order; row m = push INTO layer m */
#define PROMOE_TRACE_HIDDEN 6    /* float [T, hidden]     residual stream after the full stack */
#define PROMOE_TRACE_PREDLIST 7  /* int32 [n_moe, 1 + E]  n, list predicted BY the predictor at layer m (uncapped by G5) */
#define PROMOE_TRACE_ZLOGITS 8   /* float [n_moe, T, E]   router logits */
#define PROMOE_TRACE_U 9         /* float [n_moe, T, hidden]  u_l per MoE layer (needs PROMOE_F_TRACE_U) */

PROMOE_API int promoe_create(const promoe_shape_t* shape, const promoe_opts_t* opts, promoe_t** out);
PROMOE_API void promoe_destroy(promoe_t* h);
PROMOE_API const char* promoe_last_error(const promoe_t* h); /* h may be NULL: last create error */

/* Hand over the non-expert parameters (device pointers, borrowed). */
PROMOE_API int promoe_load_dense(promoe_t* h, const promoe_dense_t* w);

/* host_ptrs[m*E + e] = host image of routed expert e of MoE layer m: [Wgate (I x H) | Wup (I x H) | Wdown
 * (H x I)] contiguous, expert_bytes = 3*H*I*sizeof(w) (three linears).  Borrowed until destroy.
 * With PROMOE_F_WARM the first C experts of every layer are copied into their slots here. */
PROMOE_API int promoe_load_experts(promoe_t* h, const void* const* host_ptrs, size_t expert_bytes);

/* Prefill: ids_host = host ptr to n_tokens int32 ids; positions continue from the current sequence length.
 * logits_out = HOST ptr to vocab floats (last token) or NULL.  Synchronous: returns when logits are valid. */
PROMOE_API int promoe_prefill(promoe_t* h, const int32_t* ids_host, int32_t n_tokens, float* logits_out);
/* Decode one token (caller samples; tests teacher-force).  logits_out as above. */
PROMOE_API int promoe_decode(promoe_t* h, int32_t token_id, float* logits_out);

/* Batched decode (§7.5: batch sizes 1-4).  The handle holds opts.max_batch independent sequences.
 * promoe_prefill_seq = promoe_prefill on sequence `seq` (its own KV cache and position).  promoe_decode_batch decodes ONE new
 * token for each of the n_seq DISTINCT sequences seqs[0..n_seq): the layers run once over the n_seq rows — one gate per layer
 * (needed experts = the union over the rows), one slot-table step, the stride predictor voting over the rows (G7),
 * grouped expert FFNs over the permuted rows — while every row attends to its own sequence.  logits_out = HOST ptr to
 * n_seq * vocab floats (row b = sequence seqs[b]) or NULL.  Traces of the step have T = n_seq rows. */
PROMOE_API int promoe_prefill_seq(promoe_t* h, int32_t seq, const int32_t* ids_host, int32_t n_tokens, float* logits_out);
PROMOE_API int promoe_decode_batch(promoe_t* h, int32_t n_seq, const int32_t* seqs, const int32_t* token_ids, float* logits_out);

/* predictor_mode TRACE: lists for the NEXT step call; pred[m*(1+E)] = n, then n expert ids = the list the
 * predictor at MoE layer m would emit for layer m+stride.  Host ptr, copied. */
PROMOE_API int promoe_set_prediction_trace(promoe_t* h, const int32_t* pred, size_t n_int32);

PROMOE_API int promoe_stats(promoe_t* h, promoe_stats_t* out);
PROMOE_API int promoe_get_trace(promoe_t* h, int which, const void** data, size_t* bytes);
PROMOE_API int promoe_reset(promoe_t* h);   /* clears KV cache, cache state (re-warms if F_WARM) and stats */

/* Current logical slot table of MoE layer m: slot_expert_out = host ptr to C int32 (-1 = empty). */
PROMOE_API int promoe_get_slots(promoe_t* h, int32_t moe_layer, int32_t* slot_expert_out);

/* Micro entry points: single hot-path steps on caller-provided DEVICE buffers (used by kernel-level parity
 * tests).  stream = cudaStream_t or NULL (default stream).
 * All are asynchronous on `stream`. */
/* y[T,N] = x[T,K] . W[N,K]^T ; x,y fp32; W wdtype (0 fp32 / 1 bf16). path: 0 auto, 1 gemv, 2 simt gemm, 3 tcgen05 */
PROMOE_API int promoe_op_linear(const float* x, const void* w, float* y, int32_t T, int32_t N, int32_t K, int32_t wdtype,
                     int32_t path, void* stream);
/* router row A4: z = u.R^T (+b); top-k (ties -> lower index); gates = softmax over selected. */
PROMOE_API int promoe_op_route(const float* u, const void* router, const float* bias, int32_t T, int32_t H, int32_t E,
                    int32_t k, int32_t wdtype, float* z_out, int32_t* sel_out, float* gates_out,
                    float* margin_out, void* stream);
/* permutation row A8: sel [T,k] -> count[E], offset[E+1], perm[T*k], inv[T*k] */
PROMOE_API int promoe_op_permute(const int32_t* sel, int32_t T, int32_t k, int32_t E, int32_t* count, int32_t* offset,
                      int32_t* perm, int32_t* inv, void* stream);

/* attention rows A2 + A3 on caller-provided DEVICE buffers: rotate-half RoPE on q and k (tables cos_t / sin_t
 * [max_seq, d/2] fp32, angle = pos * theta^(-2i/d), G11), KV append at positions pos0 .. pos0+T-1, then causal attention of
 * the T new rows over cache positions 0 .. pos0+t.  qkv [T, (nq + 2 nkv) d] fp32 (rows: q heads | k heads | v heads; q and k
 * are rotated in place when T > 1); kcache / vcache [nkv, max_seq, d] fp32; out [T, nq d].  T == 1 runs the fused decode
 * kernel of the step and needs ws (nq * 16 * (d + 2) floats) and counters (nq int32, zero on entry, left zero); T > 1 runs the
 * prefill kernels (ws / counters may be NULL).  d in {64, 128}; nq a multiple of nkv (GQA). */
PROMOE_API int promoe_op_attention(float* qkv, const float* cos_t, const float* sin_t, float* kcache, float* vcache,
                                   float* out, float* ws, int32_t* counters, int32_t T, int32_t pos0, int32_t nq,
                                   int32_t nkv, int32_t d, int32_t max_seq, void* stream);

/* expert FFN row A9 on one resident weight set: y[T,H] = Wd.(silu(Wg.x) * (Wu.x)); x [T,H], act_ws [T,I] scratch,
 * prob_ws >= 64 bytes of device scratch (problem record).  path: 0 auto, 1 HBM-streaming GEMV (T == 1),
 * 2 SIMT grouped GEMM, 3 tcgen05 grouped GEMM (bf16 weights).  wdtype 2: wg = DEVICE ptr to one INT4 expert image (format at
 * promoe_shape_t.wdtype; wu / wd ignored), T == 1 and path 0 / 1 only. */
PROMOE_API int promoe_op_expert_ffn(const float* x, const void* wg, const void* wu, const void* wd, float* act_ws,
                                    float* y, void* prob_ws, int32_t T, int32_t H, int32_t I, int32_t wdtype,
                                    int32_t path, int32_t reserved, void* stream);

/* The same batch-1 expert FFN (A9 decode path, T == 1: y[H] = Wd.(silu(Wg.x) * (Wu.x))) for callers that may NOT allocate —
 * code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The [I] activation vector and the
 * problem record live in ONE file-scope device array of the library (64.25 KiB per GPU that loads the library, held until
 * the process exits); the call itself performs no cudaMalloc / cudaFree and calls no allocating library routine.
 * x [H], y [H] fp32 DEVICE ptrs, weights as above (DEVICE, borrowed for the call).  Limit: I <= 16384
 * (promoe_op_expert_ffn_static_max_inter()); larger I, H or I not a multiple of 16, or a NULL pointer → PROMOE_EINVAL.
 * Asynchronous on `stream`.  Every call on a device SHARES the array: calls that overlap on the GPU (different streams,
 * no ordering between them) race on it; calls on one stream are ordered.  Nothing in it must start at zero (each call
 * overwrites what it reads), so the previous call's contents never matter.  Same kernels as promoe_op_expert_ffn path 1:
 * the result is bit-identical. */
PROMOE_API int promoe_op_expert_ffn_static(const float* x, const void* wg, const void* wu, const void* wd, float* y,
                                           int32_t H, int32_t I, int32_t wdtype, void* stream);
PROMOE_API int promoe_op_expert_ffn_static_max_inter(void);

#ifdef __cplusplus
}
#endif
#endif /* PROMOE_H */
