// step.cu — the step scheduler: promoe_prefill / promoe_decode.  One host call per step; every arithmetic step
// of the path runs in the kernels of kernels_*.cu on the compute stream `cs`, copies on the copy stream `ps`.
//
// Per layer:
//   A1 rmsnorm → A2 qkv + rope + kv append → A3 attention + o-proj + residual → A1 rmsnorm
//   dense layer: SwiGLU FFN + residual
//   MoE layer m: A4 router + top-k + gates ‖ A5 predictor scores → list ‖ A8 permutation (T > 1)
//                A6 slot-table kernel: PushPrecise(m) then PushPredicted(m+stride) (Alg. 2) → problem
//                   table in launch order (cached → being prefetched → missing) + host command
//                shared expert (always resident) is launched BEFORE the host looks at the command: it covers the
//                   device→host hand-over and the first copy
//                A7 host: cancel stale LOW chunks, enqueue HIGH fills, queue LOW fills
//                A9 routed experts in launch order; decode: GEMV kernels gating on chunk flags; prefill: grouped
//                   GEMMs, ready groups first, slots recycled in launch order when |needed| > C
//                A10 combine in fixed j order + shared + residual
//   final norm + lm_head on the last token.
#include "engine.h"
#include "gemm_tc.h"

#include <cstdio>
#include <cstring>

using namespace pmk;

int ce_retire(promoe_t* h, bool all);
int ce_pump_low(promoe_t* h);
int ce_wait_cmd(promoe_t* h, int m, uint32_t seq, int part);
int ce_process_cmd(promoe_t* h, int m, std::vector<int>* deferred, int parts);
int ce_issue_deferred(promoe_t* h, int m, int i, cudaEvent_t after);
void ce_account_cmd(promoe_t* h, int m);
int ce_sync_phys_from_device(promoe_t* h);
int ce_flush_flags(promoe_t* h);

#define CKS(call)                                                                                  \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess) {                                                                       \
      h->err = std::string(#call) + ": " + cudaGetErrorString(e_);                                 \
      return PROMOE_ECUDA;                                                                         \
    }                                                                                              \
  } while (0)

static bool use_tc(const promoe_t* h, int T) { return T > 1 && h->tc != nullptr && h->wdd == 1; }

// fp32 rows of x → bf16 hi/lo planes in xsA (the activation operand of the tcgen05 GEMMs, reading G1)
static void split_A(promoe_t* h, const float* x, int T, int K) {
  launch_split_rows(x, nullptr, 1, T, K, h->xsA, h->xsA_half, h->cs);
}

// y[T,N] (+)= x[T,K]·W^T on the compute stream: GEMV for one token; T > 1: tcgen05 GEMM (bf16 weights) or SIMT.
// presplit: xsA already holds the hi/lo split of x.
static int linear(promoe_t* h, const float* x, const void* w, float* y, int T, int N, int K, int flags, bool presplit = false) {
  if (T == 1) { launch_gemv(x, w, y, N, K, h->wdd, flags, h->cs); return PROMOE_OK; }
  if (N <= 4) { launch_linear_small_n(x, w, y, T, N, K, h->wdd, flags, h->cs); return PROMOE_OK; }
  if (!use_tc(h, T) || N < 16) { launch_gemm_simt(x, w, y, T, N, K, h->wdd, flags, h->cs); return PROMOE_OK; }
  if (!presplit) split_A(h, x, T, K);
  TcGemm g;
  g.a0 = w; g.a_rows = N; g.b_hi = h->xsA; g.b_lo_off = h->xsA_half; g.b_rows_cap = (int)(h->xsA_half / K);
  g.K = K; g.N = N; g.rows = T; g.y = y; g.ldy = N; g.flags = flags;
  return tc_launch(h->tc, g, h->cs, &h->err) ? PROMOE_OK : PROMOE_ECUDA;
}

// SwiGLU FFN of an always-resident MLP (shared expert / dense layer) for all T rows of u → h->sy.
// T > 1 with tensor cores: expects the split of u in xsA.
static int resident_ffn(promoe_t* h, int l, int inter, int T) {
  const int H = h->s.hidden, wd = h->wdd;
  if (T == 1) {
    launch_ffn_gateup_gemv(h->u, h->shared_prob + l, 1, inter, H, h->sact, h->ffn_w, wd, h->chunk_bytes, h->err_dev, h->cs);
    launch_ffn_down_gemv(h->sact, h->ffn_w, h->shared_prob + l, 1, inter, H, h->sy, wd, h->chunk_bytes, h->err_dev, h->cs);
  } else if (!use_tc(h, T)) {
    launch_ffn_gateup_gemm_simt(h->u, nullptr, 1, h->shared_prob, l, 1, T, T, inter, H, h->sact, h->ffn_w, wd, h->cs);
    launch_ffn_down_gemm_simt(h->sact, h->ffn_w, h->shared_prob, l, 1, T, T, inter, H, h->sy, wd, h->cs);
  } else {
    TcGemm g;
    g.a0 = h->ffn_gate[l]; g.a1 = h->ffn_up[l]; g.a_rows = inter;
    g.b_hi = h->xsA; g.b_lo_off = h->xsA_half; g.b_rows_cap = (int)(h->xsA_half / H);
    g.K = H; g.N = inter; g.rows = T; g.swiglu = true;
    g.o_hi = h->xsB; g.o_lo_off = h->xsB_half; g.ldo = inter;
    TcGemm d;
    d.a0 = h->ffn_down[l]; d.a_rows = H; d.b_hi = h->xsB; d.b_lo_off = h->xsB_half; d.b_rows_cap = (int)(h->xsB_half / inter);
    d.K = inter; d.N = H; d.rows = T; d.y = h->sy; d.ldy = H;
    if (!tc_launch(h->tc, g, h->cs, &h->err) || !tc_launch(h->tc, d, h->cs, &h->err)) return PROMOE_ECUDA;
  }
  return PROMOE_OK;
}

// Routed experts [i, j) of the problem table (prefill): grouped SwiGLU FFN over their row ranges → yexp.
static int expert_batch(promoe_t* h, const int32_t* perm, int i, int j, int max_rows) {
  const promoe_shape_t& s = h->s;
  const int H = s.hidden, I = s.expert_inter, k = s.top_k, E = s.n_experts;
  if (h->q4 && use_tc(h, 2)) {
    // INT4 experts on the tensor cores: bf16 hi/lo staging images (exact), ONE [gate | up] GEMM of N = 2·I per image with the
    // second accumulating onto the first, SwiGLU + split, then the down GEMM the same way (kernels_q4.cu)
    const size_t stride = (size_t)3 * H * I;
    launch_dequant_q4_bf16(h->problems, i, j - i, H, I, h->q4_stage_bf, h->q4_lo_off, stride, h->problems_deq, h->cs);
    for (int pass = 0; pass < 2; ++pass) {
      TcGemm g;
      g.a0 = h->q4_stage_bf + (pass ? h->q4_lo_off : 0); g.a_rows = 2 * I; g.a_batches = E; g.a_batch_stride = stride * 2;
      g.b_hi = h->xsG; g.b_lo_off = h->xsG_half; g.b_rows_cap = (int)(h->xsG_half / H);
      g.K = H; g.N = 2 * I; g.probs = h->problems_deq; g.p0 = i; g.np = j - i; g.max_rows = max_rows;
      g.slot_base = (const uint8_t*)h->q4_stage_bf; g.y = h->q4_gu; g.ldy = 2 * I; g.flags = pass ? LIN_ACC : 0;
      if (!tc_launch(h->tc, g, h->cs, &h->err)) return PROMOE_ECUDA;
    }
    launch_swiglu_split(h->q4_gu, h->problems_deq, i, j - i, max_rows, I, h->xsB, h->xsB_half, h->cs);
    for (int pass = 0; pass < 2; ++pass) {
      TcGemm d;
      d.a0 = h->q4_stage_bf + (pass ? h->q4_lo_off : 0) + (size_t)2 * H * I; d.a_rows = H; d.a_batches = E; d.a_batch_stride = stride * 2;
      d.b_hi = h->xsB; d.b_lo_off = h->xsB_half; d.b_rows_cap = (int)(h->xsB_half / I);
      d.K = I; d.N = H; d.probs = h->problems_deq; d.p0 = i; d.np = j - i; d.max_rows = max_rows;
      d.slot_base = (const uint8_t*)h->q4_stage_bf; d.y = h->yexp; d.ldy = H; d.flags = pass ? LIN_ACC : 0;
      if (!tc_launch(h->tc, d, h->cs, &h->err)) return PROMOE_ECUDA;
    }
    return PROMOE_OK;
  }
  if (h->q4) {     // INT4 experts: exact fp32 staging images, then the fp32 SIMT grouped GEMM (kernels_q4.cu)
    launch_dequant_q4(h->problems, i, j - i, H, I, h->q4_stage, (size_t)3 * H * I, h->problems_deq, h->cs);
    launch_ffn_gateup_gemm_simt(h->u, perm, k, h->problems_deq, i, j - i, max_rows, 0, I, H, h->act, I, 0, h->cs);
    launch_ffn_down_gemm_simt(h->act, I, h->problems_deq, i, j - i, max_rows, 0, I, H, h->yexp, 0, h->cs);
    return PROMOE_OK;
  }
  if (!use_tc(h, 2)) {
    launch_ffn_gateup_gemm_simt(h->u, perm, k, h->problems, i, j - i, max_rows, 0, I, H, h->act, I, s.wdtype, h->cs);
    launch_ffn_down_gemm_simt(h->act, I, h->problems, i, j - i, max_rows, 0, I, H, h->yexp, s.wdtype, h->cs);
    return PROMOE_OK;
  }
  const int n_slots = h->Lm * h->C;
  TcGemm g;   // gate | up rows of the slot images: one 3-D tensor map over the whole slot region
  g.a0 = h->slots; g.a1 = h->slots; g.a_rows = 2 * I; g.a1_row_off = I; g.a_batches = n_slots; g.a_batch_stride = h->Be;
  g.b_hi = h->xsG; g.b_lo_off = h->xsG_half; g.b_rows_cap = (int)(h->xsG_half / H);
  g.K = H; g.N = I; g.probs = h->problems; g.p0 = i; g.np = j - i; g.max_rows = max_rows; g.slot_base = h->slots;
  g.swiglu = true; g.o_hi = h->xsB; g.o_lo_off = h->xsB_half; g.ldo = I;
  TcGemm d;   // down rows
  d.a0 = h->slots + (size_t)2 * H * I * h->wb; d.a_rows = H; d.a_batches = n_slots; d.a_batch_stride = h->Be;
  d.b_hi = h->xsB; d.b_lo_off = h->xsB_half; d.b_rows_cap = (int)(h->xsB_half / I);
  d.K = I; d.N = H; d.probs = h->problems; d.p0 = i; d.np = j - i; d.max_rows = max_rows; d.slot_base = h->slots;
  d.y = h->yexp; d.ldy = H;
  if (!tc_launch(h->tc, g, h->cs, &h->err) || !tc_launch(h->tc, d, h->cs, &h->err)) return PROMOE_ECUDA;
  return PROMOE_OK;
}

#define RC(expr) do { int rc_ = (expr); if (rc_ != PROMOE_OK) return rc_; } while (0)

// One layer of the batch-1 decode step with the fused kernels of kernels_decode.cu (7 launches instead of 19).
static int decode_layer_fused(promoe_t* h, int l, uint32_t step_seq, int pos0) {
  const promoe_shape_t& s = h->s;
  const int H = s.hidden, E = s.n_experts, k = s.top_k, C = h->C, Lm = h->Lm, I = s.expert_inter, wd = h->wdd;
  const int nq = s.n_q_heads, nkv = s.n_kv_heads, d = s.head_dim;
  cudaStream_t cs = h->cs;
  const size_t kv_layer = (size_t)nkv * s.max_seq * d;
  NormGemvArgs a{};                                                                      // K1
  a.x = h->x; a.gain = h->ln1[l]; a.eps = s.rms_eps; a.K = H;
  a.seg[0] = GemvSeg{h->wqkv[l], h->qkv, h->qkv_w, 0}; a.nseg = 1;
  launch_norm_multi_gemv(a, wd, cs);
  const size_t kv_seq = (size_t)h->cur_seq[0] * h->kv_seq_elems;
  launch_attn_decode_fused(h->qkv, h->cos_t, h->sin_t, h->kcache + kv_seq + (size_t)l * kv_layer, h->vcache + kv_seq + (size_t)l * kv_layer,   // K2
                           h->attn_ws, h->attn, h->attn_cnt, pos0, nq, nkv, d, s.max_seq, h->nsplit, cs);
  launch_gemv(h->attn, h->wo[l], h->x, H, nq * d, wd, LIN_ACC, cs);          // K3
  NormGemvArgs b{};                                                                      // K4
  b.x = h->x; b.gain = h->ln2[l]; b.eps = s.rms_eps; b.K = H; b.u_out = h->u;
  if (l < s.n_dense_layers) {
    b.wg = h->ffn_gate[l]; b.wu = h->ffn_up[l]; b.act = h->sact; b.n_sw = s.dense_inter;
    launch_norm_multi_gemv(b, wd, cs);
    launch_ffn_down_combine(nullptr, 0, nullptr, nullptr, nullptr, 0, h->shared_prob + l, h->sact, nullptr, nullptr, H, h->x, wd,
                            h->chunk_bytes, h->err_dev, cs);
    return PROMOE_OK;
  }
  const int m = l - s.n_dense_layers;
  const uint32_t seq = step_seq * 4096u + (uint32_t)m + 1u;
  int32_t* sel = h->sel + (size_t)m * h->maxT * k;
  float* gates = h->gates + (size_t)m * h->maxT * k;
  const bool mlp = h->o.predictor_mode == PROMOE_PRED_MLP;
  b.seg[b.nseg++] = GemvSeg{h->router[l], h->zraw, E, 0};
  if (mlp) b.seg[b.nseg++] = GemvSeg{h->pred_w1[l], h->p1, s.pred_hidden, LIN_RELU};
  if (s.n_shared_inter && s.shared_gate) b.seg[b.nseg++] = GemvSeg{h->shared_gate_w[l], h->sgate, 1, 0};
  launch_norm_multi_gemv(b, wd, cs);
  if (h->trace_u && cudaMemcpyAsync(h->trace_u + (size_t)m * h->maxT * H, h->u, (size_t)H * 4, cudaMemcpyDeviceToDevice, cs) != cudaSuccess) {
    h->err = "trace copy of u failed"; return PROMOE_ECUDA;
  }
  // The shared expert (resident weights, needs only u) runs on a side stream BESIDE the single-CTA slot-table kernel
  // and the host hand-over instead of behind them; K7 joins it.  (Ordering of sact / sy / u across layers: the fork
  // event of the next layer is recorded after this layer's K7, which has waited for the join event.)
  if (s.n_shared_inter) {
    if (cudaEventRecord(h->ev_fork, cs) != cudaSuccess || cudaStreamWaitEvent(h->cs2, h->ev_fork, 0) != cudaSuccess) {
      h->err = "fork of the shared-expert stream failed"; return PROMOE_ECUDA;
    }
    launch_ffn_gateup_gemv(h->u, h->shared_prob + l, 1, s.n_shared_inter, H, h->sact, h->ffn_w, wd, h->chunk_bytes, h->err_dev, h->cs2, 1);
    launch_ffn_down_gemv(h->sact, h->ffn_w, h->shared_prob + l, 1, s.n_shared_inter, H, h->sy, wd, h->chunk_bytes, h->err_dev, h->cs2, 1);
    if (cudaEventRecord(h->ev_join, h->cs2) != cudaSuccess) { h->err = "join event failed"; return PROMOE_ECUDA; }
  }
  int32_t* plist = (mlp || h->o.predictor_mode == PROMOE_PRED_TRACE) ? h->pred_list + (size_t)m * (1 + E) : nullptr;
  RouteFuse rf{};                                                                        // K5
  rf.zraw = h->zraw; rf.bias = s.router_bias ? h->router_bias[l] : nullptr; rf.z_out = h->z + (size_t)m * h->maxT * E;
  rf.sel = sel; rf.gates = gates; rf.margin = h->margin + (size_t)m * h->maxT;
  rf.p1 = h->p1; rf.pred_w2 = mlp ? h->pred_w2[l] : nullptr; rf.ph = s.pred_hidden; rf.wdtype = wd;
  rf.pred_out = mlp ? plist : nullptr; rf.k = k; rf.cap = C;
  launch_slot_table(h->tbl, m, h->o.stride, h->max_spec_decode, sel, 1, k, nullptr, plist,
                    ((h->o.flags & PROMOE_F_REORDER) ? 1 : 0) | ((h->o.flags & PROMOE_F_DEMOTE) ? 2 : 0) | (h->static_slots << 8), h->slots, h->Be, h->flags, h->n_chunks, H, I, h->q4 ? 0 : h->wb, h->problems,
                    h->n_prob, h->row_of, h->cmd_dev + m, seq, h->trace_precise + (size_t)m * (1 + 5 * E),
                    (m + h->o.stride < Lm) ? h->trace_pred + (size_t)(m + h->o.stride) * (1 + 4 * E) : nullptr, cs, &rf, h->cmd_fetch + m,
                    m > 0 ? h->cmd_fetch + (m - 1) : nullptr, h->err_dev);
  // A7 runs beside this stream: the fetch worker (kernels_fetch.cu, resident since the start of the step) sees the
  // command K5 publishes in device memory and pulls the missing chunks over the link; the flag-gated kernels K6/K7 are
  // enqueued right away and wait (ld.acquire.sys on the chunk flags, __nanosleep between polls) for exactly the bytes
  // they read.  The host is not in the layer loop at all.
  // K6 waits for the gate word K5 publishes behind the problem table (not for K5's predictor half)
  const uint32_t* gate_word = (const uint32_t*)&h->cmd_fetch[m].seq;
  if (h->q4) launch_ffn_gateup_gemv_q4(h->u, h->problems, k, I, H, h->act, I, h->chunk_bytes, h->err_dev, cs, gate_word, seq);      // K6 (INT4)
  else launch_ffn_gateup_gemv(h->u, h->problems, k, I, H, h->act, I, wd, h->chunk_bytes, h->err_dev, cs, 0, gate_word, seq);      // K6
  if (s.n_shared_inter && cudaStreamWaitEvent(cs, h->ev_join, 0) != cudaSuccess) { h->err = "join of the shared-expert stream failed"; return PROMOE_ECUDA; }
  if (h->q4) {                                                                                             // K7 (INT4)
    launch_ffn_down_combine_q4(h->act, I, h->problems, h->row_of, gates, k, (s.n_shared_inter && s.shared_gate) ? h->sgate : nullptr,
                               s.n_shared_inter ? h->sy : nullptr, H, h->x, h->chunk_bytes, h->err_dev, cs);
    return PROMOE_OK;
  }
  launch_ffn_down_combine(h->act, I, h->problems, h->row_of, gates, k, nullptr, nullptr,               // K7
                            (s.n_shared_inter && s.shared_gate) ? h->sgate : nullptr, s.n_shared_inter ? h->sy : nullptr, H, h->x,
                            wd, h->chunk_bytes, h->err_dev, cs);
  return PROMOE_OK;
}

static int run_layers(promoe_t* h, int T, uint32_t step_seq, int pos0, bool fused);

// One step.  seqs == nullptr: T tokens of ONE sequence `seq` (prefill, or decode with T = 1).  seqs != nullptr: a batched
// decode step — row b is the new token of sequence seqs[b] (T = n rows); it takes the T > 1 path of the layer loop
// with per-row attention, and returns the logits of every row.
static int run_step(promoe_t* h, const int32_t* ids_host, int T, float* logits_out, int seq = 0, const int32_t* seqs = nullptr) {
  const promoe_shape_t& s = h->s;
  const int H = s.hidden, E = s.n_experts, k = s.top_k, C = h->C, Lm = h->Lm, I = s.expert_inter;
  const int nq = s.n_q_heads, nkv = s.n_kv_heads, d = s.head_dim, wd = h->wdd;
  if (!h->dense_loaded || !h->experts_loaded) { h->err = "step before load_dense / load_experts"; return PROMOE_ESTATE; }
  if (T < 1 || !ids_host) { h->err = "step: no tokens"; return PROMOE_EINVAL; }
  const bool batch = seqs != nullptr;
  if (batch) {
    if (T > h->max_batch) { h->err = "decode_batch: more rows than max_batch"; return PROMOE_EINVAL; }
    for (int b = 0; b < T; ++b) {
      if (seqs[b] < 0 || seqs[b] >= h->max_batch) { h->err = "decode_batch: sequence index out of range"; return PROMOE_EINVAL; }
      for (int c = 0; c < b; ++c) if (seqs[c] == seqs[b]) { h->err = "decode_batch: a sequence appears twice"; return PROMOE_EINVAL; }
      if (h->seq_pos[seqs[b]] + 1 > s.max_seq) { h->err = "step: sequence exceeds max_seq"; return PROMOE_ESTATE; }
    }
  } else {
    if (seq < 0 || seq >= h->max_batch) { h->err = "step: sequence index out of range"; return PROMOE_EINVAL; }
    if (h->seq_pos[seq] + T > s.max_seq) { h->err = "step: sequence exceeds max_seq"; return PROMOE_ESTATE; }
  }
  for (int t = 0; t < T; ++t)
    if (ids_host[t] < 0 || ids_host[t] >= s.vocab) { h->err = "step: token id out of range"; return PROMOE_EINVAL; }
  cudaStream_t cs = h->cs;
  const uint32_t step_seq = ++h->step_seq;
  h->cur_batch = batch;
  h->cur_n_seq = batch ? T : 1;
  for (int b = 0; b < h->cur_n_seq; ++b) { h->cur_seq[b] = batch ? seqs[b] : seq; h->cur_pos[b] = h->seq_pos[h->cur_seq[b]]; }
  const int pos0 = h->cur_pos[0];
  // residency at step start, for B_need: needed \ resident-at-step-start
  std::fill(h->start_resident.begin(), h->start_resident.end(), 0);
  for (int m = 0; m < Lm; ++m)
    for (int i = 0; i < C; ++i) {
      const int e = h->mirror[(size_t)m * C + i];
      if (e >= 0) h->start_resident[(size_t)m * E + e] = 1;
    }
  for (auto& v : h->pending_pred) v.clear();

  const bool fused = T == 1 && !batch && !(h->o.flags & PROMOE_F_NOFUSE);
  h->want_done_events = T > 1;
  if (!fused) RC(ce_sync_phys_from_device(h));      // the copy-engine path tracks slots on the host
  if (T > 1) RC(ce_retire(h, true));   // prefill orders compute after fills with events: start from a drained copy stream
  memcpy(h->ids_pin, ids_host, (size_t)T * 4);
  CKS(cudaMemcpyAsync(h->ids, h->ids_pin, (size_t)T * 4, cudaMemcpyHostToDevice, cs));
  const bool worker = fused && h->fetch_ctas > 0;
  if (fused) CKS(cudaMemsetAsync(h->fetch_ctr, 0, sizeof(unsigned long long) * kFetchCounters, h->fs));
  if (worker) {    // A7 of this step: the device-side fetch worker, resident before anything that may wait for it
    FetchArgs fa{};
    fa.cmd = h->cmd_fetch; fa.src = h->src_dev; fa.slots = h->slots; fa.Be = h->Be; fa.chunk_bytes = h->chunk_bytes;
    fa.flags = h->flags; fa.claims = h->claims; fa.complete = h->complete; fa.ctr = h->fetch_ctr; fa.err = h->err_dev;
    fa.alive = h->alive; fa.step = step_seq; fa.Lm = Lm; fa.C = C; fa.E = E; fa.n_chunks = h->n_chunks;
    fa.preempt = (h->o.flags & PROMOE_F_PREEMPT) != 0; fa.unchunked = h->unchunked; fa.low_cap = h->low_cap;
    fa.low_ctas = h->unchunked ? 1 : std::max(1, std::min(h->o.max_inflight > 0 ? h->o.max_inflight : 1, h->fetch_ctas));
    // nothing may be queued BEHIND the worker on its stream, and no copy may be submitted behind a kernel that waits:
    // a pending operation behind a spinning kernel blocks later copy submissions (profiles/r02_spin_probe.md)
    CKS(launch_fetch(fa, h->fetch_ctas, h->fs));
  }
  cudaError_t e_end = cudaEventRecord(h->step_start, cs);
  if (e_end == cudaSuccess && (h->o.flags & PROMOE_F_TRACE)) {
    e_end = cudaMemsetAsync(h->trace_pred, 0, (size_t)Lm * (1 + 4 * E) * 4, cs);
    if (e_end == cudaSuccess && h->o.predictor_mode == PROMOE_PRED_NONE) e_end = cudaMemsetAsync(h->pred_list, 0, (size_t)Lm * (1 + E) * 4, cs);
  }
  int rc_layers = PROMOE_OK;
  if (e_end == cudaSuccess) {
    launch_embed(h->ids, h->emb, h->x, T, H, wd, cs, worker ? h->alive : nullptr, step_seq, h->err_dev);
    rc_layers = run_layers(h, T, step_seq, pos0, fused);
  }
  const int n_logit_rows = batch ? T : 1;
  if (rc_layers == PROMOE_OK && e_end == cudaSuccess) {   // ---- last token (batch: every row): final norm + lm_head
    for (int b = 0; b < n_logit_rows; ++b) {
      NormGemvArgs f{};
      f.x = h->x + (size_t)(batch ? b : T - 1) * H; f.gain = h->final_norm; f.eps = s.rms_eps; f.K = H;
      f.seg[0] = GemvSeg{h->lm_head, h->logits + (size_t)b * s.vocab, s.vocab, 0}; f.nseg = 1;
      launch_norm_multi_gemv(f, wd, cs);
    }
    e_end = cudaEventRecord(h->step_end, cs);
    if (e_end == cudaSuccess && logits_out) e_end = cudaMemcpyAsync(h->logits_pin, h->logits, (size_t)s.vocab * 4 * n_logit_rows, cudaMemcpyDeviceToHost, cs);
    if (e_end == cudaSuccess) e_end = cudaMemcpyAsync(h->err_pin, h->err_dev, 4, cudaMemcpyDeviceToHost, cs);
  }
  const bool failed = rc_layers != PROMOE_OK || e_end != cudaSuccess;
  if (fused) {
    // a step that could not be enqueued completely: raise the error word so that the worker (and any kernel waiting for
    // it) gives up at once instead of running into its time-out
    if (failed) { const int one = 1; cudaMemcpy(h->err_dev, &one, 4, cudaMemcpyHostToDevice); }
#ifdef PMK_FETCH_TRACE
    fprintf(stderr, "[host] step %u enqueued, sync cs\n", step_seq);
    cudaError_t e1 = cudaStreamSynchronize(cs);
    fprintf(stderr, "[host] cs done (%d), sync fs\n", (int)e1);
    cudaError_t e2 = cudaStreamSynchronize(h->fs);
    fprintf(stderr, "[host] fs done (%d)\n", (int)e2);
#else
    cudaError_t e1 = cudaStreamSynchronize(cs), e2 = cudaStreamSynchronize(h->fs);
#endif
    if (failed) cudaMemset(h->err_dev, 0, 4);
    if (!failed && e1 != cudaSuccess) e_end = e1;
    if (!failed && e_end == cudaSuccess && e2 != cudaSuccess) e_end = e2;
    if (!failed && e_end == cudaSuccess)
      e_end = cudaMemcpy(h->fetch_ctr_pin, h->fetch_ctr, sizeof(unsigned long long) * kFetchCounters, cudaMemcpyDeviceToHost);
    h->phys_dirty = true;
  } else if (!failed) {
    // keep feeding LOW chunks while the tail of the step drains (no-preempt mode may leave some queued)
    while (cudaStreamQuery(cs) == cudaErrorNotReady) {
      int rc = ce_pump_low(h);
      if (rc) return rc;
    }
    RC(ce_flush_flags(h));
  }
  if (rc_layers != PROMOE_OK) return rc_layers;
  if (e_end != cudaSuccess) { h->err = std::string("step: ") + cudaGetErrorString(e_end); return PROMOE_ECUDA; }
  CKS(cudaStreamSynchronize(cs));
  const int err_host = *h->err_pin;
  if (logits_out) memcpy(logits_out, h->logits_pin, (size_t)s.vocab * 4 * n_logit_rows);
  float ms = 0.f;
  CKS(cudaEventElapsedTime(&ms, h->step_start, h->step_end));
  if (fused) {     // statistics: logical from the command ring, physical from the worker's counters
    for (int m = 0; m < Lm; ++m) ce_account_cmd(h, m);
    const unsigned long long* c = h->fetch_ctr_pin;
    promoe_stats_t& st = h->st;
    st.high_bytes += c[0]; st.low_bytes += c[1]; st.h2d_bytes += c[0] + c[1]; st.low_bytes_useful += c[2]; st.hits_landed += c[3];
    st.owed_bytes_at_gate += c[4]; st.landed_chunks_at_gate += c[5]; st.landed_chunks_of += c[6];
    st.fetched_at_gate += c[7]; st.fetched_at_gate_of += c[8]; st.chunks_high += c[9]; st.chunks_low += c[10];
    st.chunks_issued += c[9] + c[10]; st.chunks_cancelled += c[11]; st.copy_busy_ms += (double)c[12] * 1e-6;
  } else {
    int rc = ce_retire(h, false);
    if (rc) return rc;
  }
  h->st.steps++; h->st.tokens += (uint64_t)T;
  h->st.step_ms += ms; h->st.last_step_ms = ms;
  if (batch) for (int b = 0; b < T; ++b) h->seq_pos[seqs[b]] += 1;
  else h->seq_pos[seq] += T;
  h->pos = h->seq_pos[0];
  h->last_T = T;
  if (err_host) {
    h->st.timeouts++;
    CKS(cudaMemsetAsync(h->err_dev, 0, 4, cs));
    h->err = "a kernel timed out waiting for a chunk-ready flag or for the fetch worker (device error word " + std::to_string(err_host) + ")";
    return PROMOE_ETIMEOUT;
  }
  return PROMOE_OK;
}

// The layer loop of one step on the compute stream.
static int run_layers(promoe_t* h, int T, uint32_t step_seq, int pos0, bool fused) {
  const promoe_shape_t& s = h->s;
  const int H = s.hidden, E = s.n_experts, k = s.top_k, C = h->C, Lm = h->Lm, I = s.expert_inter;
  const int nq = s.n_q_heads, nkv = s.n_kv_heads, d = s.head_dim, wd = h->wdd;
  cudaStream_t cs = h->cs;
  const size_t kv_layer = (size_t)nkv * s.max_seq * d;
  std::vector<int> deferred;
  for (int l = 0; l < s.n_layers; ++l) {
    if (fused) { RC(decode_layer_fused(h, l, step_seq, pos0)); continue; }
    // ---- attention block (A1-A3)
    launch_rmsnorm(h->x, h->ln1[l], h->u1, T, H, s.rms_eps, cs);
    RC(linear(h, h->u1, h->wqkv[l], h->qkv, T, h->qkv_w, H, 0));
    if (h->cur_batch) {
      // batched decode: row b attends to ITS sequence — the fused decode attention (RoPE + append + split attention + merge)
      // once per row on that sequence's cache, at that sequence's position
      for (int b = 0; b < T; ++b) {
        const size_t off = (size_t)h->cur_seq[b] * h->kv_seq_elems + (size_t)l * kv_layer;
        launch_attn_decode_fused(h->qkv + (size_t)b * h->qkv_w, h->cos_t, h->sin_t, h->kcache + off, h->vcache + off, h->attn_ws,
                                 h->attn + (size_t)b * nq * d, h->attn_cnt, h->cur_pos[b], nq, nkv, d, s.max_seq, h->nsplit, cs);
      }
    } else {
      float* kc = h->kcache + (size_t)h->cur_seq[0] * h->kv_seq_elems + (size_t)l * kv_layer;
      float* vc = h->vcache + (size_t)h->cur_seq[0] * h->kv_seq_elems + (size_t)l * kv_layer;
      launch_rope_append(h->qkv, h->cos_t, h->sin_t, kc, vc, T, pos0, nq, nkv, d, s.max_seq, cs);
      if (T == 1) launch_attn_decode(h->qkv, kc, vc, h->attn, h->attn_ws, pos0 + 1, nq, nkv, d, s.max_seq, h->nsplit, cs);
      else launch_attn_prefill(h->qkv, kc, vc, h->attn, T, pos0, nq, nkv, d, s.max_seq, cs);
    }
    RC(linear(h, h->attn, h->wo[l], h->x, T, H, nq * d, LIN_ACC));
    launch_rmsnorm(h->x, h->ln2[l], h->u, T, H, s.rms_eps, cs);
    const bool tc = use_tc(h, T);
    if (tc) split_A(h, h->u, T, H);   // u feeds the router, predictor, shared-expert and dense GEMMs
    if (l < s.n_dense_layers) {
      RC(resident_ffn(h, l, s.dense_inter, T));
      launch_add(h->x, h->sy, h->x, (size_t)T * H, cs);
      continue;
    }
    // ---- MoE block
    const int m = l - s.n_dense_layers;
    if (h->trace_u) CKS(cudaMemcpyAsync(h->trace_u + (size_t)m * h->maxT * H, h->u, (size_t)T * H * 4, cudaMemcpyDeviceToDevice, cs));
    const uint32_t seq = step_seq * 4096u + (uint32_t)m + 1u;
    int32_t* sel = h->sel + (size_t)m * h->maxT * k;
    float* gates = h->gates + (size_t)m * h->maxT * k;
    int32_t* perm = h->perm + (size_t)m * h->maxT * k;
    int32_t* inv = h->inv + (size_t)m * h->maxT * k;
    int32_t* offset = h->offset + (size_t)m * (E + 1);
    RC(linear(h, h->u, h->router[l], h->zraw, T, E, H, 0, tc));                             // A4
    launch_topk_gate(h->zraw, s.router_bias ? h->router_bias[l] : nullptr, T, E, k, h->z + (size_t)m * h->maxT * E, sel,
                     gates, h->margin + (size_t)m * h->maxT, cs);
    int32_t* plist = nullptr;
    if (h->o.predictor_mode == PROMOE_PRED_MLP) {                                      // A5
      RC(linear(h, h->u, h->pred_w1[l], h->p1, T, s.pred_hidden, H, LIN_RELU, tc));
      // the split of u must stay in xsA for the shared expert, so W2's input is split into another buffer
      if (T == 1) launch_gemv(h->p1, h->pred_w2[l], h->p2, E, s.pred_hidden, wd, 0, cs);
      else if (tc && E >= 16) {   // tcgen05 too, with xsG as the split buffer (it is refilled with the gathered rows later)
        launch_split_rows(h->p1, nullptr, 1, T, s.pred_hidden, h->xsG, h->xsG_half, cs);
        TcGemm g;
        g.a0 = h->pred_w2[l]; g.a_rows = E; g.b_hi = h->xsG; g.b_lo_off = h->xsG_half;
        g.b_rows_cap = (int)(h->xsG_half / s.pred_hidden); g.K = s.pred_hidden; g.N = E; g.rows = T; g.y = h->p2; g.ldy = E;
        if (!tc_launch(h->tc, g, cs, &h->err)) return PROMOE_ECUDA;
      } else launch_gemm_simt(h->p1, h->pred_w2[l], h->p2, T, E, s.pred_hidden, wd, 0, cs);
      plist = h->pred_list + (size_t)m * (1 + E);
      launch_pred_list(h->p2, T, E, k, C, plist, cs, h->votes_ws);
    } else if (h->o.predictor_mode == PROMOE_PRED_TRACE) {
      plist = h->pred_list + (size_t)m * (1 + E);
    }
    if (T > 1) launch_permute(sel, T, k, E, h->count + (size_t)m * E, offset, perm, inv, cs);   // A8
    launch_slot_table(h->tbl, m, h->o.stride, (T == 1 || h->cur_batch) ? h->max_spec_decode : h->max_spec_prefill, sel, T, k, T > 1 ? offset : nullptr, plist,     // A6
                      ((h->o.flags & PROMOE_F_REORDER) ? 1 : 0) | ((h->o.flags & PROMOE_F_DEMOTE) ? 2 : 0) | (h->static_slots << 8), h->slots, h->Be, h->flags, h->n_chunks, H, I, h->q4 ? 0 : h->wb,
                      h->problems, h->n_prob, h->row_of, h->cmd_dev + m, seq,
                      h->trace_precise + (size_t)m * (1 + 5 * E),
                      (m + h->o.stride < Lm) ? h->trace_pred + (size_t)(m + h->o.stride) * (1 + 4 * E) : nullptr, cs);
    const float* shared = nullptr;
    const float* sgate = nullptr;
    if (s.n_shared_inter) {                                                            // A10 shared expert first
      RC(resident_ffn(h, l, s.n_shared_inter, T));
      shared = h->sy;
      if (s.shared_gate) { RC(linear(h, h->u, h->shared_gate_w[l], h->sgate, T, 1, H, 0)); sgate = h->sgate; }
    }
    // ---- A7: hand-over to the copy engine
    int rc = ce_wait_cmd(h, m, seq, 1);
    if (rc == PROMOE_OK) rc = ce_wait_cmd(h, m, seq, 2);
    if (rc) return rc;
    deferred.clear();
    rc = ce_process_cmd(h, m, &deferred, 3);
    if (rc) return rc;
    const LayerCmd& cmd = h->cmd_host[m];
    const int n = cmd.n_needed;
    // ---- A9 routed experts, launch order
    if (T == 1) {
      if (h->q4) {
        launch_ffn_gateup_gemv_q4(h->u, h->problems, n, I, H, h->act, I, h->chunk_bytes, h->err_dev, cs);
        launch_ffn_down_gemv_q4(h->act, I, h->problems, n, H, h->yexp, h->chunk_bytes, h->err_dev, cs);
      } else {
        launch_ffn_gateup_gemv(h->u, h->problems, n, I, H, h->act, I, wd, h->chunk_bytes, h->err_dev, cs);
        launch_ffn_down_gemv(h->act, I, h->problems, n, I, H, h->yexp, wd, h->chunk_bytes, h->err_dev, cs);
      }
      launch_combine(h->x, h->yexp, h->row_of, gates, 1, k, H, shared, sgate, h->x, cs);
    } else {
      if (tc) launch_split_rows(h->u, perm, k, T * k, H, h->xsG, h->xsG_half, cs);   // gathered rows, permuted order
      // batches: [all class A] [all class B] then the class C experts as their fills land in copy order — one by one for bf16
      // images (311 us of copy per expert against ≈ 30 us of compute), in groups of up to 3 for INT4 images, whose 6 launches per
      // expert (dequantise, two [gate|up] passes, SwiGLU, two down passes: ≈ 120 us of 22-CTA launches, profiles/r02_int4.md)
      // out-last the 80 us copy of the next image; measured on c2 / c3: 2: 6231 / 8033 tok/s, 3: 6290 / 8235, 4: 6282 / 8152,
      // 8: 6184 / 7861, 16: 5919 / 7426 (a larger group waits longer for its last image and leaves a longer tail)
      const int c_group = h->q4 ? 3 : 1;
      int i = 0;
      size_t dnext = 0;
      while (i < n) {
        const int cls = cmd.need[7 * i + 1];
        int j = i + 1;
        // class A / B: one grouped launch — unless fills are waiting for their slots (prefill with |needed| > C: every
        // class-C fill recycles the slot of a resident expert that has been computed): then groups of 8, so that the first
        // copies start after 8 experts instead of after all of them (the link idled for the whole class-A batch: 0.3 ms per
        // layer with bf16 images, 0.75 ms with INT4 images and their dequantisation pass)
        if (cls != 2) while (j < n && cmd.need[7 * j + 1] == cls && (deferred.empty() || j - i < 8)) ++j;
        else   // class C: experts whose fill has been issued (no slot dependency, or one the loop below has already released:
               // `deferred` is in launch order, so those are the entries before `dnext`); a fill that is still held back
               // waits for an event recorded BEHIND this batch and must not be waited for inside it
          while (j < n && j - i < c_group && cmd.need[7 * j + 1] == 2 &&
                 (cmd.need[7 * j + 4] < 0 || (dnext > 0 && j <= deferred[dnext - 1]))) ++j;
        int max_rows = 0;
        for (int q = i; q < j; ++q) {
          max_rows = std::max(max_rows, (int)cmd.need[7 * q + 6]);
          SlotPhys& p = h->phys[(size_t)m * C + cmd.need[7 * q + 2]];
          if (p.done_valid) CKS(cudaStreamWaitEvent(cs, p.done, 0));      // dependency mechanism
        }
        RC(expert_batch(h, perm, i, j, max_rows));
        // slots recycled inside the layer: fills that wait for a launch position in [i, j)
        bool need_ev = false;
        for (size_t q = dnext; q < deferred.size(); ++q) {
          const int dep = cmd.need[7 * deferred[q] + 4];
          if (dep < j) need_ev = true;
        }
        if (need_ev) {
          cudaEvent_t ev = h->done_ev[i % h->done_ev.size()];
          CKS(cudaEventRecord(ev, cs));
          while (dnext < deferred.size() && cmd.need[7 * deferred[dnext] + 4] < j) {
            rc = ce_issue_deferred(h, m, deferred[dnext], ev);
            if (rc) return rc;
            ++dnext;
          }
        }
        i = j;
      }
      launch_combine(h->x, h->yexp, inv, gates, T, k, H, shared, sgate, h->x, cs);
    }
  }
  return PROMOE_OK;
}

extern "C" int promoe_prefill(promoe_t* h, const int32_t* ids_host, int32_t n_tokens, float* logits_out) {
  if (!h) return PROMOE_EINVAL;
  return run_step(h, ids_host, n_tokens, logits_out);
}
extern "C" int promoe_decode(promoe_t* h, int32_t token_id, float* logits_out) {
  if (!h) return PROMOE_EINVAL;
  return run_step(h, &token_id, 1, logits_out);
}
extern "C" int promoe_prefill_seq(promoe_t* h, int32_t seq, const int32_t* ids_host, int32_t n_tokens, float* logits_out) {
  if (!h) return PROMOE_EINVAL;
  return run_step(h, ids_host, n_tokens, logits_out, seq);
}
extern "C" int promoe_decode_batch(promoe_t* h, int32_t n_seq, const int32_t* seqs, const int32_t* token_ids, float* logits_out) {
  if (!h || !seqs || !token_ids || n_seq < 1) return PROMOE_EINVAL;
  if (n_seq == 1) return run_step(h, token_ids, 1, logits_out, seqs[0]);      // one row: the fused decode step of that sequence
  return run_step(h, token_ids, n_seq, logits_out, 0, seqs);
}
