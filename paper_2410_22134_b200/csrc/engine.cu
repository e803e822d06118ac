// engine.cu — promoe_create / load / reset / destroy: shapes, buffers, the contiguous slot region,
// slot-table state, streams.  The step scheduler is in step.cu, the copy engine in copy_engine.cu.
#include "engine.h"
#include "gemm_tc.h"

#include <cuda.h>

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstdio>
#include <cstring>

using namespace pmk;

static std::string g_create_err;
namespace pmk {
unsigned long long g_launches = 0;
bool g_use_pdl = true;
}

#define CK(call)                                                                                   \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess) {                                                                       \
      h->err = std::string(#call) + ": " + cudaGetErrorString(e_);                                 \
      return PROMOE_ECUDA;                                                                         \
    }                                                                                              \
  } while (0)

template <typename T>
static cudaError_t dalloc(T** p, size_t n) {
  cudaError_t e = cudaMalloc((void**)p, n * sizeof(T));
  if (e == cudaSuccess) e = cudaMemset(*p, 0, n * sizeof(T));
  return e;
}

int promoe_init_cache_state(promoe_t* h, bool copy_warm);  // below
int ce_retire(promoe_t* h, bool all);


extern "C" const char* promoe_last_error(const promoe_t* h) { return h ? h->err.c_str() : g_create_err.c_str(); }

extern "C" int promoe_create(const promoe_shape_t* sp, const promoe_opts_t* op, promoe_t** out) {
  if (!sp || !op || !out) { g_create_err = "null argument"; return PROMOE_EINVAL; }
  const promoe_shape_t& s = *sp;
  auto bad = [&](const char* m) { g_create_err = m; return PROMOE_EINVAL; };
  const int Lm = s.n_layers - s.n_dense_layers;
  if (s.n_layers <= 0 || Lm <= 0 || s.hidden % 16 || s.expert_inter % 16) return bad("hidden/expert_inter must be multiples of 16");
  if (s.head_dim != 64 && s.head_dim != 128) return bad("head_dim must be 64 or 128");
  if (s.n_q_heads % s.n_kv_heads) return bad("n_q_heads must be a multiple of n_kv_heads");
  if (s.n_experts > 256 || s.top_k > 16 || s.top_k > s.n_experts) return bad("n_experts <= 256, top_k <= 16");
  if (s.n_shared_inter % 16 || s.dense_inter % 16 || s.pred_hidden % 8) return bad("ffn widths must be multiples of 16");
  if (s.wdtype != 0 && s.wdtype != 1 && s.wdtype != 2) return bad("wdtype must be 0 (fp32), 1 (bf16) or 2 (bf16 + INT4 routed experts)");
  if (s.wdtype == 2 && (s.hidden % 128 || s.expert_inter % 128)) return bad("INT4 experts need hidden and expert_inter to be multiples of 128 (the quantisation group)");
  if (op->cache_slots <= 0 || op->cache_slots % Lm) return bad("cache_slots must be a positive multiple of n_moe_layers");
  const int C = op->cache_slots / Lm;
  if (C > s.n_experts) return bad("more slots per layer than experts");
  if (C < s.top_k) return bad("slots per layer must be >= top_k (a decode step pins top_k experts)");
  if (op->stride < 1) return bad("stride must be >= 1");
  if ((size_t)s.max_seq * s.top_k > 16384 * 4) return bad("max_seq*top_k too large for the single-CTA permutation");

  preload_all();      // no kernel of this library may be loaded lazily behind a spinning kernel
  (void)cudaGetLastError();
  promoe_t* h = new promoe();
  h->s = s; h->o = *op; h->Lm = Lm; h->C = C;
  h->wb = s.wdtype == 0 ? 4 : 2;
  h->wdd = s.wdtype == 0 ? 0 : 1;
  h->q4 = s.wdtype == 2;
  h->Be = (size_t)3 * s.hidden * s.expert_inter * h->wb;
  if (h->q4) h->Be = (size_t)3 * s.hidden * s.expert_inter / 2 + (size_t)3 * s.hidden * s.expert_inter / 128 * 2;   // codes + bf16 scales (G18)
  h->chunk_bytes = op->chunk_bytes ? (size_t)op->chunk_bytes : ((size_t)256 << 10);
  if (h->chunk_bytes % 256) { delete h; return bad("chunk_bytes must be a multiple of 256"); }
  h->n_chunks = (int)((h->Be + h->chunk_bytes - 1) / h->chunk_bytes);
  // the pinned ring the flag copies read from must hold the words of every fill that can be in flight (one layer's
  // HIGH fills) at least twice over
  if (h->n_chunks > kMaxChunks || (size_t)h->n_chunks * C * 2 > kFlagSrcRing) { delete h; return bad("chunk_bytes too small for this expert size (too many chunks per image)"); }
  // the fused down+combine kernel cuts (top_k + shared) dot products into pieces of 2048 elements: at most 192 pieces
  {
    const int pieces = s.top_k * ((s.expert_inter + 2047) / 2048) + (std::max(s.n_shared_inter, s.dense_inter) + 2047) / 2048;
    if (pieces > 192) { delete h; return bad("top_k * ceil(expert_inter / 2048) + ceil(shared_inter / 2048) must be <= 192"); }
  }
  h->unchunked = (op->flags & PROMOE_F_UNCHUNKED) != 0;
  cudaGetDevice(&h->dev);
  // < 0: no fetch worker at all — only for runs in which nothing is ever fetched (every expert resident), e.g. under a
  // profiler that serialises kernels: a persistent worker would never see the gates of kernels that cannot run beside it
  h->fetch_ctas = op->fetch_ctas > 0 ? std::min(op->fetch_ctas, 16) : (op->fetch_ctas < 0 ? 0 : 4);
  h->max_inflight = op->max_inflight > 0 ? op->max_inflight : 2;
  h->high_group = op->high_group > 0 ? op->high_group : 0;
  h->low_cap = op->low_cap_chunks > 0 ? op->low_cap_chunks : 0;
  h->max_spec_decode = op->max_spec_decode == 0 ? s.top_k : std::max(0, op->max_spec_decode);
  h->max_spec_prefill = op->max_spec_prefill <= 0 ? 0 : op->max_spec_prefill;
  h->maxT = s.max_seq;
  h->max_batch = op->max_batch > 0 ? op->max_batch : 1;
  if (h->max_batch > 8) { delete h; return bad("max_batch must be <= 8"); }
  h->seq_pos.assign(h->max_batch, 0);
  h->static_slots = op->static_slots > 0 ? op->static_slots : 0;
  // the fused decode step runs the k experts of a layer side by side: a staging buffer must never be recycled inside one step
  if (h->static_slots > C - s.top_k) { delete h; return bad("static_slots must leave at least top_k staging slots per layer"); }
  h->qkv_w = (s.n_q_heads + 2 * s.n_kv_heads) * s.head_dim;
  h->ffn_w = s.n_shared_inter > s.dense_inter ? s.n_shared_inter : s.dense_inter;
  h->nsplit = 16;
  int rc = [&]() -> int {
    const int H = s.hidden, E = s.n_experts, k = s.top_k, L = s.n_layers, T = h->maxT;
    if (op->compute_stream) h->cs = (cudaStream_t)op->compute_stream;
    else { CK(cudaStreamCreateWithFlags(&h->cs, cudaStreamNonBlocking)); h->own_cs = true; }
    CK(cudaStreamCreateWithFlags(&h->ps, cudaStreamNonBlocking));
    CK(cudaStreamCreateWithFlags(&h->cs2, cudaStreamNonBlocking));
    { int lo = 0, hi = 0; CK(cudaDeviceGetStreamPriorityRange(&lo, &hi)); CK(cudaStreamCreateWithPriority(&h->fs, cudaStreamNonBlocking, hi)); }
    CK(cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming)); CK(cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming));
    CK(dalloc(&h->x, (size_t)T * H)); CK(dalloc(&h->u1, (size_t)T * H)); CK(dalloc(&h->u, (size_t)T * H));
    CK(dalloc(&h->qkv, (size_t)T * h->qkv_w)); CK(dalloc(&h->attn, (size_t)T * s.n_q_heads * s.head_dim));
    CK(dalloc(&h->zraw, (size_t)T * E)); CK(dalloc(&h->p1, (size_t)T * s.pred_hidden)); CK(dalloc(&h->p2, (size_t)T * E));
    CK(dalloc(&h->act, (size_t)T * k * s.expert_inter)); CK(dalloc(&h->yexp, (size_t)T * k * H));
    if (h->ffn_w) { CK(dalloc(&h->sact, (size_t)T * h->ffn_w)); CK(dalloc(&h->sy, (size_t)T * H)); }
    CK(dalloc(&h->sgate, (size_t)T)); CK(dalloc(&h->attn_ws, (size_t)s.n_q_heads * h->nsplit * (s.head_dim + 2)));
    CK(dalloc(&h->xf, (size_t)H)); CK(dalloc(&h->logits, (size_t)s.vocab * h->max_batch));
    h->kv_seq_elems = (size_t)L * s.n_kv_heads * s.max_seq * s.head_dim;
    CK(dalloc(&h->kcache, h->kv_seq_elems * h->max_batch));
    CK(dalloc(&h->vcache, h->kv_seq_elems * h->max_batch));
    CK(dalloc(&h->ids, (size_t)T));
    CK(dalloc(&h->sel, (size_t)Lm * T * k)); CK(dalloc(&h->gates, (size_t)Lm * T * k)); CK(dalloc(&h->margin, (size_t)Lm * T));
    CK(dalloc(&h->z, (size_t)Lm * T * E));
    CK(dalloc(&h->votes_ws, (size_t)257)); CK(cudaMemset(h->votes_ws, 0, 257 * 4));
    if (op->flags & PROMOE_F_TRACE_U) CK(dalloc(&h->trace_u, (size_t)Lm * T * H));
    CK(dalloc(&h->count, (size_t)Lm * E)); CK(dalloc(&h->offset, (size_t)Lm * (E + 1)));
    CK(dalloc(&h->perm, (size_t)Lm * T * k)); CK(dalloc(&h->inv, (size_t)Lm * T * k));
    CK(dalloc(&h->pred_list, (size_t)Lm * (1 + E))); CK(dalloc(&h->trace_precise, (size_t)Lm * (1 + 5 * E)));
    CK(dalloc(&h->trace_pred, (size_t)Lm * (1 + 4 * E))); CK(dalloc(&h->row_of, (size_t)k)); CK(dalloc(&h->n_prob, (size_t)1));
    CK(dalloc(&h->problems, (size_t)E)); CK(dalloc(&h->shared_prob, (size_t)L)); CK(dalloc(&h->err_dev, (size_t)1)); CK(dalloc(&h->attn_cnt, (size_t)s.n_q_heads));
    if (h->q4) {
      CK(dalloc(&h->problems_deq, (size_t)E));
      if (op->flags & PROMOE_F_TENSOR) {
        h->q4_lo_off = (size_t)E * 3 * H * s.expert_inter;
        CK(dalloc(&h->q4_stage_bf, 2 * h->q4_lo_off)); CK(dalloc(&h->q4_gu, (size_t)T * k * 2 * s.expert_inter));
      } else CK(dalloc(&h->q4_stage, (size_t)E * 3 * H * s.expert_inter));
    }
    if ((op->flags & PROMOE_F_TENSOR) && s.wdtype >= 1) {
      h->tc = tc_create(&h->err);
      if (!h->tc) return PROMOE_ECUDA;
      auto up8 = [](size_t v) { return (v + 7) & ~(size_t)7; };
      const size_t ka = (size_t)std::max(std::max(H, s.n_q_heads * s.head_dim), s.pred_hidden);
      h->xsA_half = up8((size_t)T * ka);
      h->xsG_half = up8((size_t)T * k * H);
      h->xsB_half = up8(std::max((size_t)T * k * s.expert_inter, (size_t)T * h->ffn_w));
      CK(dalloc(&h->xsA, 2 * h->xsA_half)); CK(dalloc(&h->xsG, 2 * h->xsG_half)); CK(dalloc(&h->xsB, 2 * h->xsB_half));
    }
    // RoPE tables in double (reading G11): angle = pos * theta^(-2i/d)
    {
      const int half = s.head_dim / 2;
      std::vector<float> c((size_t)s.max_seq * half), sn((size_t)s.max_seq * half);
      for (int p = 0; p < s.max_seq; ++p)
        for (int i = 0; i < half; ++i) {
          const double a = (double)p * std::pow((double)s.rope_theta, -2.0 * i / s.head_dim);
          c[(size_t)p * half + i] = (float)std::cos(a); sn[(size_t)p * half + i] = (float)std::sin(a);
        }
      CK(dalloc(&h->cos_t, c.size())); CK(dalloc(&h->sin_t, sn.size()));
      CK(cudaMemcpy(h->cos_t, c.data(), c.size() * 4, cudaMemcpyHostToDevice));
      CK(cudaMemcpy(h->sin_t, sn.data(), sn.size() * 4, cudaMemcpyHostToDevice));
    }
    // expert cache: one contiguous slot region + chunk flags + logical table
    CK(cudaMalloc((void**)&h->slots, (size_t)Lm * C * h->Be));
    CK(dalloc(&h->flags, (size_t)Lm * C * h->n_chunks));
    CK(dalloc(&h->tbl.slot_expert, (size_t)Lm * C)); CK(dalloc(&h->tbl.expert_slot, (size_t)Lm * E));
    CK(dalloc(&h->tbl.stamp, (size_t)Lm * C)); CK(dalloc(&h->tbl.gen, (size_t)Lm * C));
    CK(dalloc(&h->tbl.origin, (size_t)Lm * C)); CK(dalloc(&h->tbl.clock, (size_t)1));
    h->tbl.Lm = Lm; h->tbl.C = C; h->tbl.E = E;
    CK(dalloc(&h->claims, (size_t)Lm * C * h->n_chunks)); CK(dalloc(&h->complete, (size_t)Lm * C)); CK(dalloc(&h->alive, (size_t)1));
    CK(dalloc(&h->fetch_ctr, (size_t)kFetchCounters)); CK(dalloc(&h->src_dev, (size_t)Lm * E));
    CK(cudaMalloc((void**)&h->cmd_fetch, sizeof(LayerCmd) * Lm)); CK(cudaMemset(h->cmd_fetch, 0, sizeof(LayerCmd) * Lm));
    CK(cudaHostAlloc((void**)&h->fetch_ctr_pin, sizeof(unsigned long long) * kFetchCounters, cudaHostAllocDefault));
    CK(cudaHostAlloc((void**)&h->cmd_host, sizeof(LayerCmd) * Lm, cudaHostAllocMapped));
    memset((void*)h->cmd_host, 0, sizeof(LayerCmd) * Lm);
    CK(cudaHostGetDevicePointer((void**)&h->cmd_dev, (void*)h->cmd_host, 0));
    CK(cudaHostAlloc((void**)&h->logits_pin, sizeof(float) * (size_t)s.vocab * h->max_batch, cudaHostAllocDefault));
    CK(cudaHostAlloc((void**)&h->ids_pin, sizeof(int32_t) * (size_t)T, cudaHostAllocDefault));
    CK(cudaHostAlloc((void**)&h->err_pin, sizeof(int), cudaHostAllocDefault));
    CK(cudaHostAlloc((void**)&h->flagsrc_host, sizeof(uint32_t) * kFlagSrcRing, cudaHostAllocDefault));
    h->phys.resize((size_t)Lm * C);
    for (auto& p : h->phys) CK(cudaEventCreateWithFlags(&p.done, cudaEventDisableTiming));
    const int ring = 8192;
    h->ev_ring.resize(ring); h->ev_ring_start.resize(ring); h->ev_is_low.assign(ring, 0);
    for (int i = 0; i < ring; ++i) { CK(cudaEventCreate(&h->ev_ring[i])); CK(cudaEventCreate(&h->ev_ring_start[i])); }
    h->done_ev.resize(E);
    for (auto& e : h->done_ev) CK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    CK(cudaEventCreate(&h->step_start)); CK(cudaEventCreate(&h->step_end));
    h->mirror.assign((size_t)Lm * C, -1);
    h->start_resident.assign((size_t)Lm * E, 0);
    h->pending_pred.resize(Lm);
    return PROMOE_OK;
  }();
  if (rc != PROMOE_OK) { g_create_err = h->err; promoe_destroy(h); return rc; }
  *out = h;
  return PROMOE_OK;
}

extern "C" void promoe_destroy(promoe_t* h) {
  if (!h) return;
  cudaDeviceSynchronize();
  for (void* p : h->registered) cudaHostUnregister(p);
  void* bufs[] = {h->x, h->u1, h->u, h->qkv, h->attn, h->zraw, h->p1, h->p2, h->act, h->yexp, h->sact, h->sy,
                  h->sgate, h->attn_ws, h->xf, h->logits, h->kcache, h->vcache, h->cos_t, h->sin_t, h->ids, h->sel,
                  h->count, h->offset, h->perm, h->inv, h->gates, h->margin, h->z, h->pred_list, h->trace_precise,
                  h->trace_pred, h->row_of, h->n_prob, h->problems, h->shared_prob, h->err_dev, h->attn_cnt, h->slots, h->flags,
                  h->tbl.slot_expert, h->tbl.expert_slot, h->tbl.stamp, h->tbl.gen, h->tbl.origin, h->tbl.clock,
                  h->claims, h->complete, h->alive, h->fetch_ctr, h->src_dev, h->cmd_fetch, h->trace_u, h->q4_stage, h->problems_deq, h->q4_stage_bf, h->q4_gu, h->votes_ws};
  for (void* b : bufs) if (b) cudaFree(b);
  if (h->xsA) cudaFree(h->xsA);
  if (h->xsG) cudaFree(h->xsG);
  if (h->xsB) cudaFree(h->xsB);
  if (h->tc) tc_destroy(h->tc);
  if (h->cmd_host) cudaFreeHost((void*)h->cmd_host);
  if (h->flagsrc_host) cudaFreeHost(h->flagsrc_host);
  if (h->logits_pin) cudaFreeHost(h->logits_pin);
  if (h->ids_pin) cudaFreeHost(h->ids_pin);
  if (h->err_pin) cudaFreeHost(h->err_pin);
  for (auto& p : h->phys) if (p.done) cudaEventDestroy(p.done);
  for (auto e : h->ev_ring) if (e) cudaEventDestroy(e);
  for (auto e : h->ev_ring_start) if (e) cudaEventDestroy(e);
  for (auto e : h->done_ev) if (e) cudaEventDestroy(e);
  if (h->step_start) cudaEventDestroy(h->step_start);
  if (h->step_end) cudaEventDestroy(h->step_end);
  if (h->ps) cudaStreamDestroy(h->ps);
  if (h->cs2) cudaStreamDestroy(h->cs2);
  if (h->fs) cudaStreamDestroy(h->fs);
  if (h->fetch_ctr_pin) cudaFreeHost(h->fetch_ctr_pin);
  if (h->ev_fork) cudaEventDestroy(h->ev_fork);
  if (h->ev_join) cudaEventDestroy(h->ev_join);
  if (h->own_cs && h->cs) cudaStreamDestroy(h->cs);
  delete h;
}

// ---------------------------------------------------------------------------------------------------------
extern "C" int promoe_load_dense(promoe_t* h, const promoe_dense_t* w) {
  if (!h || !w) return PROMOE_EINVAL;
  const promoe_shape_t& s = h->s;
  const int L = s.n_layers;
  if (!w->emb || !w->lm_head || !w->final_norm || !w->ln1 || !w->ln2 || !w->wqkv || !w->wo) {
    h->err = "load_dense: missing tensor"; return PROMOE_EINVAL;
  }
  h->emb = w->emb; h->lm_head = w->lm_head; h->final_norm = w->final_norm;
  auto cp = [&](auto& dst, auto src) { dst.assign(L, nullptr); if (src) for (int l = 0; l < L; ++l) dst[l] = src[l]; };
  cp(h->ln1, w->ln1); cp(h->ln2, w->ln2); cp(h->wqkv, w->wqkv); cp(h->wo, w->wo); cp(h->router, w->router);
  cp(h->router_bias, w->router_bias); cp(h->pred_w1, w->pred_w1); cp(h->pred_w2, w->pred_w2);
  cp(h->ffn_gate, w->ffn_gate); cp(h->ffn_up, w->ffn_up); cp(h->ffn_down, w->ffn_down);
  cp(h->shared_gate_w, w->shared_gate_w);
  std::vector<FfnProblem> sp(L);
  for (int l = 0; l < L; ++l) {
    const bool dense = l < s.n_dense_layers;
    if (!h->ln1[l] || !h->ln2[l] || !h->wqkv[l] || !h->wo[l]) { h->err = "load_dense: missing attention tensor"; return PROMOE_EINVAL; }
    if (!dense && !h->router[l]) { h->err = "load_dense: missing router"; return PROMOE_EINVAL; }
    if (!dense && s.router_bias && !h->router_bias[l]) { h->err = "load_dense: missing router bias"; return PROMOE_EINVAL; }
    if (!dense && h->o.predictor_mode == PROMOE_PRED_MLP && (!h->pred_w1[l] || !h->pred_w2[l])) {
      h->err = "load_dense: missing predictor weights"; return PROMOE_EINVAL;
    }
    const int inter = dense ? s.dense_inter : s.n_shared_inter;
    if (inter && (!h->ffn_gate[l] || !h->ffn_up[l] || !h->ffn_down[l])) { h->err = "load_dense: missing ffn tensor"; return PROMOE_EINVAL; }
    if (!dense && s.shared_gate && !h->shared_gate_w[l]) { h->err = "load_dense: missing shared gate"; return PROMOE_EINVAL; }
    FfnProblem pb{};
    pb.wg = h->ffn_gate[l]; pb.wu = h->ffn_up[l]; pb.wd = h->ffn_down[l];
    pb.flags = nullptr; pb.gen = 0; pb.inter = inter; pb.row0 = 0; pb.nrows = 1; pb.expert = -1;
    sp[l] = pb;
  }
  CK(cudaMemcpy(h->shared_prob, sp.data(), sizeof(FfnProblem) * L, cudaMemcpyHostToDevice));
  h->dense_loaded = true;
  return PROMOE_OK;
}

// (Re)initialise the logical table, the flags and the host mirrors; optionally copy the warm set.
int promoe_init_cache_state(promoe_t* h, bool copy_warm) {
  const int Lm = h->Lm, C = h->C, E = h->s.n_experts;
  const bool warm = (h->o.flags & PROMOE_F_WARM) != 0;
  std::vector<int32_t> se((size_t)Lm * C, -1), es((size_t)Lm * E, -1);
  std::vector<unsigned long long> stamp((size_t)Lm * C, 0);
  unsigned long long clock = 0;
  if (warm) {   // reading G4: experts 0..C-1 resident, expert 0 oldest, clock = Lm*C
    for (int m = 0; m < Lm; ++m)
      for (int i = 0; i < C; ++i) { se[(size_t)m * C + i] = i; es[(size_t)m * E + i] = i; stamp[(size_t)m * C + i] = (unsigned long long)m * C + i + 1; }
    clock = (unsigned long long)Lm * C;
  }
  CK(cudaStreamSynchronize(h->cs)); CK(cudaStreamSynchronize(h->ps)); CK(cudaStreamSynchronize(h->cs2)); CK(cudaStreamSynchronize(h->fs));
  CK(cudaMemset(h->claims, 0, (size_t)Lm * C * h->n_chunks * 4));
  CK(cudaMemset(h->complete, 0, (size_t)Lm * C * 4));
  CK(cudaMemset(h->cmd_fetch, 0, sizeof(LayerCmd) * Lm));
  h->phys_dirty = false;
  CK(cudaMemcpy(h->tbl.slot_expert, se.data(), se.size() * 4, cudaMemcpyHostToDevice));
  CK(cudaMemcpy(h->tbl.expert_slot, es.data(), es.size() * 4, cudaMemcpyHostToDevice));
  CK(cudaMemcpy(h->tbl.stamp, stamp.data(), stamp.size() * 8, cudaMemcpyHostToDevice));
  CK(cudaMemcpy(h->tbl.clock, &clock, 8, cudaMemcpyHostToDevice));
  CK(cudaMemset(h->tbl.gen, 0, (size_t)Lm * C * 4));
  CK(cudaMemset(h->tbl.origin, 0, (size_t)Lm * C));
  CK(cudaMemset(h->flags, 0, (size_t)Lm * C * h->n_chunks * 4));
  CK(cudaMemset(h->err_dev, 0, 4));
  CK(cudaMemset(h->votes_ws, 0, 257 * 4));
  CK(cudaMemset(h->attn_cnt, 0, (size_t)h->s.n_q_heads * 4));
  h->mirror = se;
  h->low.clear();
  h->batch_open = false;
  if (ce_retire(h, true)) return PROMOE_ECUDA;
  for (size_t i = 0; i < h->phys.size(); ++i) {
    SlotPhys& p = h->phys[i];
    p.gen = 0; p.expert = se[i]; p.issued = warm ? h->n_chunks : 0; p.flagged = p.issued; p.fill_seq = 0; p.done_valid = false;
    p.low_chunks = 0; p.low_bytes = 0; p.low_ring.clear();
  }

  if (warm && copy_warm && h->experts_loaded)
    for (int m = 0; m < Lm; ++m)
      for (int i = 0; i < C; ++i)
        CK(cudaMemcpy(h->slots + ((size_t)m * C + i) * h->Be, h->expert_host[(size_t)m * E + i], h->Be, cudaMemcpyHostToDevice));
  for (auto& v : h->pending_pred) v.clear();
  return PROMOE_OK;
}

extern "C" int promoe_load_experts(promoe_t* h, const void* const* host_ptrs, size_t expert_bytes) {
  if (!h || !host_ptrs) return PROMOE_EINVAL;
  if (expert_bytes != h->Be) { h->err = "load_experts: expert_bytes != 3*H*I*sizeof(w)"; return PROMOE_EINVAL; }
  const size_t n = (size_t)h->Lm * h->s.n_experts;
  h->expert_host.assign(host_ptrs, host_ptrs + n);
  bool contiguous = true;
  for (size_t i = 0; i < n; ++i) {
    if (!host_ptrs[i]) { h->err = "load_experts: null expert pointer"; return PROMOE_EINVAL; }
    if (i && (const char*)host_ptrs[i] != (const char*)host_ptrs[i - 1] + expert_bytes) contiguous = false;
  }
  auto unregistered = [](const void* p) {
    cudaPointerAttributes at{};
    cudaError_t e = cudaPointerGetAttributes(&at, p);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return true; }
    return at.type == cudaMemoryTypeUnregistered;
  };
  if (contiguous && unregistered(host_ptrs[0])) {      // one mapping (e.g. a shared-memory file shared by all ranks)
    CK(cudaHostRegister((void*)host_ptrs[0], n * expert_bytes, cudaHostRegisterPortable | cudaHostRegisterMapped));
    h->registered.push_back((void*)host_ptrs[0]);
    h->st.registered_host_bytes += n * expert_bytes;
  } else {
    for (size_t i = 0; i < n; ++i)
      if (unregistered(host_ptrs[i])) {
        CK(cudaHostRegister((void*)host_ptrs[i], expert_bytes, cudaHostRegisterMapped));
        h->registered.push_back((void*)host_ptrs[i]);
        h->st.registered_host_bytes += expert_bytes;
      }
  }
  // the device-side fetch worker reads the images through their device-visible addresses (pinned host memory is mapped
  // into the unified address space); TMA bulk copies need 16-byte alignment
  {
    std::vector<unsigned long long> sd(n);
    for (size_t i = 0; i < n; ++i) {
      void* dp = nullptr;
      cudaError_t e = cudaHostGetDevicePointer(&dp, (void*)host_ptrs[i], 0);
      if (e != cudaSuccess || !dp) { (void)cudaGetLastError(); h->err = "load_experts: expert image is not device-accessible pinned host memory"; return PROMOE_EINVAL; }
      if (((uintptr_t)dp & 15) || ((uintptr_t)host_ptrs[i] & 15)) { h->err = "load_experts: expert images must be 16-byte aligned"; return PROMOE_EINVAL; }
      sd[i] = (unsigned long long)(uintptr_t)dp;
    }
    CK(cudaMemcpy(h->src_dev, sd.data(), n * 8, cudaMemcpyHostToDevice));
  }
  h->experts_loaded = true;
  return promoe_init_cache_state(h, true);
}

extern "C" int promoe_reset(promoe_t* h) {
  if (!h) return PROMOE_EINVAL;
  const uint64_t reg = h->st.registered_host_bytes;
  h->st = promoe_stats_t{};
  h->st.registered_host_bytes = reg;
  h->pos = 0;
  std::fill(h->seq_pos.begin(), h->seq_pos.end(), 0);
  h->last_T = 0;
  return promoe_init_cache_state(h, true);
}

extern "C" int promoe_get_slots(promoe_t* h, int32_t m, int32_t* out) {
  if (!h || !out || m < 0 || m >= h->Lm) return PROMOE_EINVAL;
  CK(cudaStreamSynchronize(h->cs));
  CK(cudaMemcpy(out, h->tbl.slot_expert + (size_t)m * h->C, (size_t)h->C * 4, cudaMemcpyDeviceToHost));
  return PROMOE_OK;
}

extern "C" int promoe_stats(promoe_t* h, promoe_stats_t* out) {
  if (!h || !out) return PROMOE_EINVAL;
  *out = h->st;
  out->kernel_launches = pmk::g_launches;
  return PROMOE_OK;
}

