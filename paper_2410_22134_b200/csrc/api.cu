// api.cu — trace getters, injected prediction lists and the micro entry points of include/promoe.h.
#include "engine.h"
#include "gemm_tc.h"

#include <cstring>

using namespace pmk;

#define CKA(call)                                                                                  \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess) {                                                                       \
      if (h) h->err = std::string(#call) + ": " + cudaGetErrorString(e_);                          \
      return PROMOE_ECUDA;                                                                         \
    }                                                                                              \
  } while (0)

extern "C" int promoe_set_prediction_trace(promoe_t* h, const int32_t* pred, size_t n_int32) {
  if (!h || !pred) return PROMOE_EINVAL;
  const size_t want = (size_t)h->Lm * (1 + h->s.n_experts);
  if (n_int32 != want) { h->err = "set_prediction_trace: expected n_moe_layers*(1+E) int32"; return PROMOE_EINVAL; }
  if (h->o.predictor_mode != PROMOE_PRED_TRACE) { h->err = "set_prediction_trace: predictor_mode is not TRACE"; return PROMOE_ESTATE; }
  for (int m = 0; m < h->Lm; ++m) {
    const int32_t* row = pred + (size_t)m * (1 + h->s.n_experts);
    if (row[0] < 0 || row[0] > h->s.n_experts) { h->err = "set_prediction_trace: bad list length"; return PROMOE_EINVAL; }
    for (int i = 0; i < row[0]; ++i)
      if (row[1 + i] < 0 || row[1 + i] >= h->s.n_experts) { h->err = "set_prediction_trace: bad expert id"; return PROMOE_EINVAL; }
  }
  CKA(cudaStreamSynchronize(h->cs));
  CKA(cudaMemcpy(h->pred_list, pred, want * 4, cudaMemcpyHostToDevice));
  return PROMOE_OK;
}

// Copy `rows` rows of `row_bytes` from a device buffer whose rows are `stride_bytes` apart into trace_buf.
static int gather_rows(promoe_t* h, const void* dev, size_t rows, size_t row_bytes, size_t stride_bytes, size_t dst_off) {
  CKA(cudaMemcpy2D(h->trace_buf.data() + dst_off, row_bytes, dev, stride_bytes, row_bytes, rows, cudaMemcpyDeviceToHost));
  return PROMOE_OK;
}

extern "C" int promoe_get_trace(promoe_t* h, int which, const void** data, size_t* bytes) {
  if (!h || !data || !bytes) return PROMOE_EINVAL;
  const int T = h->last_T, k = h->s.top_k, E = h->s.n_experts, Lm = h->Lm, H = h->s.hidden;
  if (T <= 0) { h->err = "get_trace: no step has run"; return PROMOE_ESTATE; }
  CKA(cudaStreamSynchronize(h->cs));
  const size_t mT = (size_t)h->maxT;
  int rc = PROMOE_OK;
  size_t n = 0;
  switch (which) {
    case PROMOE_TRACE_SEL:
      n = (size_t)Lm * T * k * 4; h->trace_buf.resize(n);
      rc = gather_rows(h, h->sel, Lm, (size_t)T * k * 4, mT * k * 4, 0); break;
    case PROMOE_TRACE_GATES:
      n = (size_t)Lm * T * k * 4; h->trace_buf.resize(n);
      rc = gather_rows(h, h->gates, Lm, (size_t)T * k * 4, mT * k * 4, 0); break;
    case PROMOE_TRACE_MARGIN:
      n = (size_t)Lm * T * 4; h->trace_buf.resize(n);
      rc = gather_rows(h, h->margin, Lm, (size_t)T * 4, mT * 4, 0); break;
    case PROMOE_TRACE_ZLOGITS:
      n = (size_t)Lm * T * E * 4; h->trace_buf.resize(n);
      rc = gather_rows(h, h->z, Lm, (size_t)T * E * 4, mT * E * 4, 0); break;
    case PROMOE_TRACE_PERM: {
      if (T == 1) { h->err = "get_trace: no permutation in a decode step"; return PROMOE_ESTATE; }
      const size_t row = (size_t)(E + (E + 1) + 2 * T * k) * 4;
      n = (size_t)Lm * row; h->trace_buf.resize(n);
      // per layer: count | offset | perm | inv
      CKA(cudaMemcpy2D(h->trace_buf.data(), row, h->count, (size_t)E * 4, (size_t)E * 4, Lm, cudaMemcpyDeviceToHost));
      CKA(cudaMemcpy2D(h->trace_buf.data() + (size_t)E * 4, row, h->offset, (size_t)(E + 1) * 4, (size_t)(E + 1) * 4, Lm, cudaMemcpyDeviceToHost));
      CKA(cudaMemcpy2D(h->trace_buf.data() + (size_t)(2 * E + 1) * 4, row, h->perm, mT * k * 4, (size_t)T * k * 4, Lm, cudaMemcpyDeviceToHost));
      CKA(cudaMemcpy2D(h->trace_buf.data() + (size_t)(2 * E + 1 + T * k) * 4, row, h->inv, mT * k * 4, (size_t)T * k * 4, Lm, cudaMemcpyDeviceToHost));
      break;
    }
    case PROMOE_TRACE_PRECISE:
      n = (size_t)Lm * (1 + 5 * E) * 4; h->trace_buf.resize(n);
      CKA(cudaMemcpy(h->trace_buf.data(), h->trace_precise, n, cudaMemcpyDeviceToHost)); break;
    case PROMOE_TRACE_PRED:
      n = (size_t)Lm * (1 + 4 * E) * 4; h->trace_buf.resize(n);
      CKA(cudaMemcpy(h->trace_buf.data(), h->trace_pred, n, cudaMemcpyDeviceToHost)); break;
    case PROMOE_TRACE_PREDLIST:
      n = (size_t)Lm * (1 + E) * 4; h->trace_buf.resize(n);
      CKA(cudaMemcpy(h->trace_buf.data(), h->pred_list, n, cudaMemcpyDeviceToHost)); break;
    case PROMOE_TRACE_U:
      if (!h->trace_u) { h->err = "get_trace: PROMOE_TRACE_U needs PROMOE_F_TRACE_U at create"; return PROMOE_ESTATE; }
      n = (size_t)Lm * T * H * 4; h->trace_buf.resize(n);
      rc = gather_rows(h, h->trace_u, Lm, (size_t)T * H * 4, mT * H * 4, 0); break;
    case PROMOE_TRACE_HIDDEN:
      n = (size_t)T * H * 4; h->trace_buf.resize(n);
      CKA(cudaMemcpy(h->trace_buf.data(), h->x, n, cudaMemcpyDeviceToHost)); break;
    default:
      h->err = "get_trace: unknown trace kind"; return PROMOE_EINVAL;
  }
  if (rc) return rc;
  *data = h->trace_buf.data();
  *bytes = n;
  return PROMOE_OK;
}

// ---- micro entry points (device buffers; asynchronous on `stream`) -------------------------------------------
static int launch_status() { return cudaGetLastError() == cudaSuccess ? PROMOE_OK : PROMOE_ECUDA; }

extern "C" int promoe_op_linear(const float* x, const void* w, float* y, int32_t T, int32_t N, int32_t K,
                                int32_t wdtype, int32_t path, void* stream) {
  if (!x || !w || !y || T < 1 || N < 1 || K < 1 || (wdtype != 0 && wdtype != 1)) return PROMOE_EINVAL;
  if (K % (wdtype == 0 ? 4 : 8)) return PROMOE_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  if (path == 0) path = (T == 1) ? 1 : 2;
  if (path == 1) {
    for (int t = 0; t < T; ++t) launch_gemv(x + (size_t)t * K, w, y + (size_t)t * N, N, K, wdtype, 0, st);
  } else if (path == 2) {
    launch_gemm_simt(x, w, y, T, N, K, wdtype, 0, st);
  } else if (path == 3) {   // tcgen05 (test entry: allocates scratch and synchronises)
    if (wdtype != 1) return PROMOE_EINVAL;
    TcContext* tc = tc_create(nullptr);
    if (!tc) return PROMOE_ECUDA;
    __nv_bfloat16* sp = nullptr;
    int rc = PROMOE_ECUDA;
    if (cudaMalloc((void**)&sp, (size_t)2 * T * K * 2) == cudaSuccess) {
      launch_split_rows(x, nullptr, 1, T, K, sp, (size_t)T * K, st);
      TcGemm g;
      g.a0 = w; g.a_rows = N; g.b_hi = sp; g.b_lo_off = (size_t)T * K; g.b_rows_cap = T; g.K = K; g.N = N; g.rows = T;
      g.y = y; g.ldy = N;
      if (tc_launch(tc, g, st, nullptr) && cudaStreamSynchronize(st) == cudaSuccess) rc = PROMOE_OK;
      cudaFree(sp);
    }
    tc_destroy(tc);
    return rc == PROMOE_OK ? launch_status() : rc;
  } else return PROMOE_EINVAL;
  return launch_status();
}

extern "C" int promoe_op_route(const float* u, const void* router, const float* bias, int32_t T, int32_t H, int32_t E,
                               int32_t k, int32_t wdtype, float* z_out, int32_t* sel_out, float* gates_out,
                               float* margin_out, void* stream) {
  if (!u || !router || !z_out || !sel_out || !gates_out || T < 1 || E < 1 || E > 256 || k < 1 || k > 16 || k > E) return PROMOE_EINVAL;
  if (H % (wdtype == 0 ? 4 : 8)) return PROMOE_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  // raw logits go to z_out first, then top-k adds the bias in place
  if (T == 1) launch_gemv(u, router, z_out, E, H, wdtype, 0, st);
  else launch_gemm_simt(u, router, z_out, T, E, H, wdtype, 0, st);
  launch_topk_gate(z_out, bias, T, E, k, z_out, sel_out, gates_out, margin_out, st);
  return launch_status();
}

extern "C" int promoe_op_permute(const int32_t* sel, int32_t T, int32_t k, int32_t E, int32_t* count, int32_t* offset,
                                 int32_t* perm, int32_t* inv, void* stream) {
  if (!sel || !count || !offset || !perm || !inv || T < 0 || k < 1 || E < 1 || E > 256) return PROMOE_EINVAL;
  if ((size_t)T * k > 65536) return PROMOE_EINVAL;
  launch_permute(sel, T, k, E, count, offset, perm, inv, (cudaStream_t)stream);
  return launch_status();
}

extern "C" int promoe_op_expert_ffn(const float* x, const void* wg, const void* wu, const void* wd, float* act_ws,
                                    float* y, void* prob_ws, int32_t T, int32_t H, int32_t I, int32_t wdtype,
                                    int32_t path, int32_t reserved, void* stream) {
  (void)reserved;
  cudaStream_t st = (cudaStream_t)stream;
  if (wdtype == 2) {     // INT4 image [gate codes | up codes | down codes | scales] at wg (wu / wd ignored); GEMV path only
    if (!x || !wg || !act_ws || !y || !prob_ws || T != 1 || path > 1 || H % 128 || I % 128) return PROMOE_EINVAL;
    FfnProblem q{};
    q.wg = wg; q.wu = nullptr; q.wd = nullptr; q.flags = nullptr; q.gen = 0; q.inter = I; q.row0 = 0; q.nrows = 1; q.expert = -1;
    if (cudaMemcpyAsync(prob_ws, &q, sizeof(q), cudaMemcpyHostToDevice, st) != cudaSuccess) return PROMOE_ECUDA;
    launch_ffn_gateup_gemv_q4(x, (const FfnProblem*)prob_ws, 1, I, H, act_ws, I, (size_t)1 << 20, nullptr, st);
    launch_ffn_down_gemv_q4(act_ws, I, (const FfnProblem*)prob_ws, 1, H, y, (size_t)1 << 20, nullptr, st);
    return launch_status();
  }
  if (!x || !wg || !wu || !wd || !act_ws || !y || !prob_ws || T < 1 || H % 16 || I % 16 || (wdtype != 0 && wdtype != 1)) return PROMOE_EINVAL;
  FfnProblem pb{};
  pb.wg = wg; pb.wu = wu; pb.wd = wd; pb.flags = nullptr; pb.gen = 0; pb.inter = I; pb.row0 = 0; pb.nrows = T; pb.expert = -1;
  if (cudaMemcpyAsync(prob_ws, &pb, sizeof(pb), cudaMemcpyHostToDevice, st) != cudaSuccess) return PROMOE_ECUDA;
  const FfnProblem* dp = (const FfnProblem*)prob_ws;
  if (path == 0) path = (T == 1) ? 1 : 2;
  if (path == 1) {
    if (T != 1) return PROMOE_EINVAL;
    launch_ffn_gateup_gemv(x, dp, 1, I, H, act_ws, I, wdtype, (size_t)1 << 20, nullptr, st);
    launch_ffn_down_gemv(act_ws, I, dp, 1, I, H, y, wdtype, (size_t)1 << 20, nullptr, st);
  } else if (path == 2) {
    launch_ffn_gateup_gemm_simt(x, nullptr, 1, dp, 0, 1, T, 0, I, H, act_ws, I, wdtype, st);
    launch_ffn_down_gemm_simt(act_ws, I, dp, 0, 1, T, 0, I, H, y, wdtype, st);
  } else if (path == 3) {   // tcgen05 (test entry: allocates scratch and synchronises)
    if (wdtype != 1) return PROMOE_EINVAL;
    TcContext* tc = tc_create(nullptr);
    if (!tc) return PROMOE_ECUDA;
    __nv_bfloat16 *s1 = nullptr, *s2 = nullptr;
    int rc = PROMOE_ECUDA;
    if (cudaMalloc((void**)&s1, (size_t)2 * T * H * 2) == cudaSuccess && cudaMalloc((void**)&s2, (size_t)2 * T * I * 2) == cudaSuccess) {
      launch_split_rows(x, nullptr, 1, T, H, s1, (size_t)T * H, st);
      TcGemm g;
      g.a0 = wg; g.a1 = wu; g.a_rows = I; g.b_hi = s1; g.b_lo_off = (size_t)T * H; g.b_rows_cap = T; g.K = H; g.N = I; g.rows = T;
      g.swiglu = true; g.o_hi = s2; g.o_lo_off = (size_t)T * I; g.ldo = I;
      TcGemm d;
      d.a0 = wd; d.a_rows = H; d.b_hi = s2; d.b_lo_off = (size_t)T * I; d.b_rows_cap = T; d.K = I; d.N = H; d.rows = T;
      d.y = y; d.ldy = H;
      if (tc_launch(tc, g, st, nullptr) && tc_launch(tc, d, st, nullptr) && cudaStreamSynchronize(st) == cudaSuccess) rc = PROMOE_OK;
    }
    if (s1) cudaFree(s1);
    if (s2) cudaFree(s2);
    tc_destroy(tc);
    return rc == PROMOE_OK ? launch_status() : rc;
  } else return PROMOE_EINVAL;
  return launch_status();
}


// A2 + A3 on caller buffers: RoPE on q and k (rotate-half), KV append at positions pos0 .. pos0+T-1, attention over the
// cache.  T == 1 runs the fused decode kernel of the step (split over positions, last-CTA merge), T > 1 the prefill kernels.
extern "C" int promoe_op_attention(float* qkv, const float* cos_t, const float* sin_t, float* kcache, float* vcache,
                                   float* out, float* ws, int32_t* counters, int32_t T, int32_t pos0, int32_t nq,
                                   int32_t nkv, int32_t d, int32_t max_seq, void* stream) {
  if (!qkv || !cos_t || !sin_t || !kcache || !vcache || !out || T < 1 || pos0 < 0 || pos0 + T > max_seq) return PROMOE_EINVAL;
  if ((d != 64 && d != 128) || nq < 1 || nkv < 1 || nq % nkv) return PROMOE_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  if (T == 1) {
    if (!ws || !counters) return PROMOE_EINVAL;
    launch_attn_decode_fused(qkv, cos_t, sin_t, kcache, vcache, ws, out, counters, pos0, nq, nkv, d, max_seq, 16, st);
  } else {
    launch_rope_append(qkv, cos_t, sin_t, kcache, vcache, T, pos0, nq, nkv, d, max_seq, st);
    launch_attn_prefill(qkv, kcache, vcache, out, T, pos0, nq, nkv, d, max_seq, st);
  }
  return launch_status();
}
