// bench_hooks.cu — measurement hooks of include/promoe_bench.h: used by bench.py only, never by the step path.
#include "engine.h"
#include "../../include/promoe_bench.h"

#include <algorithm>
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

// Pinned H2D bandwidth for `bytes`-sized copies with `depth` copies kept in flight (chunk size choice).
extern "C" int promoe_bench_h2d(size_t bytes, int32_t depth, int32_t reps, double* gbs_out) {
  if (!bytes || depth < 1 || reps < 1 || !gbs_out) return PROMOE_EINVAL;
  void *hbuf = nullptr, *dbuf = nullptr;
  cudaStream_t st = nullptr;
  cudaEvent_t a = nullptr, b = nullptr;
  const size_t total = bytes * (size_t)depth;
  int rc = PROMOE_ECUDA;
  if (cudaHostAlloc(&hbuf, total, cudaHostAllocDefault) == cudaSuccess && cudaMalloc(&dbuf, total) == cudaSuccess &&
      cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking) == cudaSuccess && cudaEventCreate(&a) == cudaSuccess &&
      cudaEventCreate(&b) == cudaSuccess) {
    memset(hbuf, 1, total);
    double best = 0.0;
    for (int r = 0; r < reps + 1; ++r) {
      cudaEventRecord(a, st);
      for (int i = 0; i < depth; ++i)
        cudaMemcpyAsync((char*)dbuf + (size_t)i * bytes, (char*)hbuf + (size_t)i * bytes, bytes, cudaMemcpyHostToDevice, st);
      cudaEventRecord(b, st);
      if (cudaStreamSynchronize(st) != cudaSuccess) break;
      float ms = 0.f;
      cudaEventElapsedTime(&ms, a, b);
      if (r > 0 && ms > 0.f) best = std::max(best, (double)total / (ms * 1e6));
    }
    *gbs_out = best;
    rc = best > 0.0 ? PROMOE_OK : PROMOE_ECUDA;
  }
  if (a) cudaEventDestroy(a);
  if (b) cudaEventDestroy(b);
  if (st) cudaStreamDestroy(st);
  if (dbuf) cudaFree(dbuf);
  if (hbuf) cudaFreeHost(hbuf);
  return rc;
}


extern "C" int promoe_bench_kernel_time(promoe_t* h, int32_t which, int32_t reps, double* avg_ms_out, double* bytes_out) {
  if (!h || reps < 1 || !avg_ms_out || !bytes_out || (which != 0 && which != 1)) return PROMOE_EINVAL;
  if (!h->experts_loaded) { h->err = "kernel_time before load_experts"; return PROMOE_ESTATE; }
  const promoe_shape_t& s = h->s;
  const int k = s.top_k, H = s.hidden, I = s.expert_inter, Lm = h->Lm, C = h->C;
  const size_t hi = h->q4 ? (size_t)H * I / 2 : (size_t)H * I * h->wb;     // INT4: code bytes per matrix (scales follow the codes)
  // problem tables over resident slots, one per layer, so that consecutive launches stream different weights
  std::vector<FfnProblem> pb((size_t)Lm * k);
  for (int m = 0; m < Lm; ++m)
    for (int i = 0; i < k; ++i) {
      const uint8_t* img = h->slots + ((size_t)m * C + (i % C)) * h->Be;
      FfnProblem& p = pb[(size_t)m * k + i];
      p.wg = img; p.wu = img + hi; p.wd = img + 2 * hi; p.flags = nullptr; p.gen = 0; p.inter = I; p.row0 = i; p.nrows = 1;
      p.expert = -1; p.pad = 0;
    }
  FfnProblem* dp = nullptr;
  int32_t* row_of = nullptr;
  float* gates = nullptr;
  CKA(cudaMalloc((void**)&dp, pb.size() * sizeof(FfnProblem)));
  CKA(cudaMalloc((void**)&row_of, (size_t)k * 4));
  CKA(cudaMalloc((void**)&gates, (size_t)k * 4));
  std::vector<int32_t> ro(k);
  std::vector<float> g(k, 1.0f / (float)k);
  for (int i = 0; i < k; ++i) ro[i] = i;
  CKA(cudaMemcpy(dp, pb.data(), pb.size() * sizeof(FfnProblem), cudaMemcpyHostToDevice));
  CKA(cudaMemcpy(row_of, ro.data(), (size_t)k * 4, cudaMemcpyHostToDevice));
  CKA(cudaMemcpy(gates, g.data(), (size_t)k * 4, cudaMemcpyHostToDevice));
  cudaEvent_t a, b;
  CKA(cudaEventCreate(&a)); CKA(cudaEventCreate(&b));
  auto launch = [&](int r) {
    const FfnProblem* q = dp + (size_t)(r % Lm) * k;
    if (h->q4) {
      if (which == 0) launch_ffn_gateup_gemv_q4(h->u, q, k, I, H, h->act, I, h->chunk_bytes, h->err_dev, h->cs);
      else launch_ffn_down_combine_q4(h->act, I, q, row_of, gates, k, nullptr, nullptr, H, h->yexp, h->chunk_bytes, h->err_dev, h->cs);
    } else if (which == 0) launch_ffn_gateup_gemv(h->u, q, k, I, H, h->act, I, s.wdtype, h->chunk_bytes, h->err_dev, h->cs);
    else launch_ffn_down_combine(h->act, I, q, row_of, gates, k, nullptr, nullptr, nullptr, nullptr, H, h->yexp, s.wdtype,
                                 h->chunk_bytes, h->err_dev, h->cs);
  };
  for (int r = 0; r < 3; ++r) launch(r);
  CKA(cudaEventRecord(a, h->cs));
  for (int r = 0; r < reps; ++r) launch(r + 3);
  CKA(cudaEventRecord(b, h->cs));
  CKA(cudaStreamSynchronize(h->cs));
  float ms = 0.f;
  CKA(cudaEventElapsedTime(&ms, a, b));
  cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(dp); cudaFree(row_of); cudaFree(gates);
  *avg_ms_out = (double)ms / reps;
  *bytes_out = (double)k * (which == 0 ? 2.0 : 1.0) * (double)hi * (h->q4 ? 33.0 / 32.0 : 1.0);   // INT4: + one bf16 scale per 128 codes
  return PROMOE_OK;
}
