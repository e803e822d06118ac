// kernels.h — host-side launchers of the ProMoE sm_100a kernels (raw pointers + cudaStream_t).
// Row labels A1..A10 refer to DESIGN.md "hot path" (= SURVEY.md §8(a)).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "common.cuh"

namespace pmk {

// A0 embedding lookup: x[t,:] = Emb[ids[t],:] widened to fp32.
// alive != nullptr (fused decode): thread 0 first waits until *alive == alive_want, i.e. until the fetch kernel of this
// step (kernels_fetch.cu) is resident — every later kernel of the step is ordered behind this one, so no flag-gated
// kernel can occupy the GPU before the worker that feeds it runs.
void launch_embed(const int32_t* ids, const void* emb, float* x, int T, int H, int wdtype, cudaStream_t st,
                  const uint32_t* alive = nullptr, uint32_t alive_want = 0, int* err = nullptr);
// A1 RMSNorm: y = x * rsqrt(mean(x^2)+eps) * w   (one warp-group per row).
void launch_rmsnorm(const float* x, const float* w, float* y, int T, int H, float eps, cudaStream_t st);

// Linear y[T,N] (+)= x[T,K] . W[N,K]^T.  flags: bit0 add to y (residual), bit1 ReLU.
enum { LIN_ACC = 1, LIN_RELU = 2 };
// HBM-streaming GEMV (T == 1): one warp per output row, 16-byte loads.
void launch_gemv(const float* x, const void* w, float* y, int N, int K, int wdtype, int flags, cudaStream_t st);
// Small N, any T: one warp per output element (the N = 1 shared-expert gate in prefill).
void launch_linear_small_n(const float* x, const void* w, float* y, int T, int N, int K, int wdtype, int flags,
                           cudaStream_t st);
// SIMT fp32 tiled GEMM (any T).
void launch_gemm_simt(const float* x, const void* w, float* y, int T, int N, int K, int wdtype, int flags,
                      cudaStream_t st);

// A2 RoPE on q,k (rotate-half pairs (i, i+d/2)) + KV append.  qkv [T,(nq+2nkv)d] fp32; cos/sin tables
// [max_seq, d/2] fp32 (computed in double at create time, G11); kcache/vcache [nkv, max_seq, d] fp32.
void launch_rope_append(float* qkv, const float* cos_t, const float* sin_t, float* kcache, float* vcache, int T,
                        int pos0, int nq, int nkv, int d, int max_seq, cudaStream_t st);
// A3 decode attention (T == 1), split over positions; ws = workspace [nq, nsplit, d+2].
void launch_attn_decode(const float* qkv, const float* kcache, const float* vcache, float* out, float* ws,
                        int n_pos, int nq, int nkv, int d, int max_seq, int nsplit, cudaStream_t st);
// A3 prefill causal attention, fp32 flash-style.  q rows t=0..T-1 at positions pos0+t; keys 0..pos0+T-1.
void launch_attn_prefill(const float* qkv, const float* kcache, const float* vcache, float* out, int T, int pos0,
                         int nq, int nkv, int d, int max_seq, cudaStream_t st);

// A4 top-k + gate softmax over selected logits (+ margin); z [T,E] (+bias[E]).  One warp per token.
void launch_topk_gate(const float* z, const float* bias, int T, int E, int k, float* z_out, int32_t* sel,
                      float* gates, float* margin, cudaStream_t st);
// A5 predictor list: per-token top-k of scores p [T,E]; T==1: the top-k list; T>1: votes -> top-cap (G7).
// out list: pred[0] = n, pred[1..n] = experts.
void launch_pred_list(const float* p, int T, int E, int k, int cap, int32_t* pred, cudaStream_t st, int32_t* ws = nullptr);

// A8 permutation: histogram -> exclusive scan -> stable scatter (single CTA, atomics-free).
void launch_permute(const int32_t* sel, int T, int k, int E, int32_t* count, int32_t* offset, int32_t* perm,
                    int32_t* inv, cudaStream_t st);

struct RouteFuse;
// A6 slot table.  State of ONE model (all MoE layers) lives in device memory, laid out by SlotTable.
struct SlotTable {
  int32_t* slot_expert;      // [Lm, C]  expert in slot or -1
  int32_t* expert_slot;      // [Lm, E]  slot of expert or -1
  unsigned long long* stamp; // [Lm, C]  LRU stamp
  uint32_t* gen;             // [Lm, C]  allocation generation (flag value the slot's chunks must show)
  uint8_t* origin;           // [Lm, C]  0 RESIDENT, 1 PRED, 2 PRECISE
  unsigned long long* clock; // [1]
  int Lm, C, E;
};
// Command record written to mapped pinned host memory, one per (step, MoE layer).  `seq` is written last
// (release, system scope); the host issuer polls it.
struct LayerCmd {
  volatile uint32_t seq;     // step_seq * 4096 + layer + 1 once the NEEDED part (PushPrecise) is valid
  volatile uint32_t seq_pred;  // same value once the PREDICTED part (PushPredicted) is valid (published later)
  volatile uint32_t seq_done;  // same value once the kernel has written the table rows back (device copy only): the next
                               // layer's slot-table kernel waits for it, because the expert kernels no longer wait for the
                               // predictor half of this kernel (DESIGN.md §6 "gate word")
  uint32_t pad_;
  int32_t n_needed;
  int32_t n_pred;            // entries of the push INTO layer (m + stride), 0 if none
  int32_t pred_target;
  // needed experts in launch order: expert, class (0 A,1 B,2 C), slot, victim, dep, gen, nrows
  int32_t need[7 * 256];
  // predicted experts in listed order: expert, action (0 touch,1 alloc,2 skip), slot, victim, gen
  int32_t pred[5 * 256];
};
// One thread block (one warp) runs PushPrecise(m) then PushPredicted(m+stride) (Alg. 2) and writes:
//  problems[i] for the needed experts in launch order (row ranges from offset[] when T > 1),
//  dec_order[j] (decode: launch position -> j), the trace records and the host command.
// cmd_dev2: second copy of the command in DEVICE memory for the fetch kernel (fused decode), or nullptr.
void launch_slot_table(SlotTable tbl, int m, int stride, int max_spec, const int32_t* sel, int T, int k, const int32_t* offset,
                       const int32_t* pred_list, int reorder, const uint8_t* slot_base, size_t slot_bytes,
                       const uint32_t* flag_base, int flags_per_slot, int H, int inter, int wbytes,
                       FfnProblem* problems, int32_t* n_problems, int32_t* j_of_problem, LayerCmd* cmd,
                       uint32_t seq, int32_t* trace_precise, int32_t* trace_pred, cudaStream_t st,
                       const RouteFuse* fuse = nullptr, LayerCmd* cmd_dev2 = nullptr, const LayerCmd* cmd_prev = nullptr,
                       int* err = nullptr);

// A7 (fused decode): the device-side prefetch worker (kernels_fetch.cu).
struct FetchArgs {
  const LayerCmd* cmd;         // device ring [Lm] written by the slot-table kernel
  const unsigned long long* src;   // [Lm*E] device-visible addresses of the pinned host expert images
  uint8_t* slots;              // slot region [Lm, C, Be]
  unsigned long long Be, chunk_bytes;
  uint32_t* flags;             // [Lm, C, n_chunks]  generation whose chunk has landed (Alg. 1 l.10 ready_chunk)
  uint32_t* claims;            // [Lm, C, n_chunks]  (generation << 1 | by_LOW) of the copy that took the chunk
  uint32_t* complete;          // [Lm, C]            generation whose whole image is known to have landed
  unsigned long long* ctr;     // FC_N counters (kernels_fetch.cu), zeroed by the host before the launch
  int* err;                    // device error word (shared with the expert kernels)
  uint32_t* alive;             // ← step once the worker runs
  uint32_t step;
  int Lm, C, E, n_chunks, preempt, unchunked, low_cap;
  int low_ctas;                // CTAs that may copy LOW chunks (one chunk each at a time): bounds what a gate finds in its way
};
constexpr int kFetchCounters = 16;
cudaError_t launch_fetch(const FetchArgs& a, int ctas, cudaStream_t st);

// A9 decode expert FFN (GEMV, T == 1) over a problem list in launch order.
//  gateup: act[p, i] = silu(Wg_p[i,:].u) * (Wu_p[i,:].u)     down: y[p, h] = Wd_p[h,:].act[p,:]
// chunk geometry: image = [gate | up | down], chunk c covers bytes [c*chunk_bytes, (c+1)*chunk_bytes).
// gate_seq != nullptr (fused decode): the kernel does NOT wait for the kernel in front of it (the slot-table kernel, whose
// predictor half it does not need) but for *gate_seq == gate_want, the word that kernel publishes behind the problem table.
void launch_ffn_gateup_gemv(const float* u, const FfnProblem* probs, int n_probs, int max_inter, int H, float* act,
                            int act_stride, int wdtype, size_t chunk_bytes, int* err, cudaStream_t st,
                            int static_table = 0, const uint32_t* gate_seq = nullptr, uint32_t gate_want = 0);
void launch_ffn_down_gemv(const float* act, int act_stride, const FfnProblem* probs, int n_probs, int max_inter,
                          int H, float* y, int wdtype, size_t chunk_bytes, int* err, cudaStream_t st, int static_table = 0);
// A9 prefill grouped SwiGLU FFN, SIMT fp32: problems [p0, p0+np) each with its row range; x rows are gathered
// through row_src (permuted position -> row_src[pos] / src_div = token) or direct when row_src == nullptr.
void launch_ffn_gateup_gemm_simt(const float* x, const int32_t* row_src, int src_div, const FfnProblem* probs,
                                 int p0, int np, int max_rows, int rows_override, int max_inter, int H, float* act,
                                 int act_stride, int wdtype, cudaStream_t st);
void launch_ffn_down_gemm_simt(const float* act, int act_stride, const FfnProblem* probs, int p0, int np,
                               int max_rows, int rows_override, int max_inter, int H, float* y, int wdtype, cudaStream_t st);

// A9 with INT4 group-quantised expert images (kernels_q4.cu; G18).  Problem records as above with wg = image base.
void launch_ffn_gateup_gemv_q4(const float* u, const FfnProblem* probs, int n_probs, int max_inter, int H, float* act,
                               int act_stride, size_t chunk_bytes, int* err, cudaStream_t st,
                               const uint32_t* gate_seq = nullptr, uint32_t gate_want = 0);
void launch_ffn_down_gemv_q4(const float* act, int act_stride, const FfnProblem* probs, int n_probs, int H, float* y,
                             size_t chunk_bytes, int* err, cudaStream_t st);
void launch_ffn_down_combine_q4(const float* act, int act_stride, const FfnProblem* probs, const int32_t* row_of,
                                const float* gates, int k, const float* sgate_logit, const float* shared_y, int H, float* x,
                                size_t chunk_bytes, int* err, cudaStream_t st);
// prefill: INT4 images of problems [p0, p0+np) → fp32 staging images + records pointing at them (out_probs[p0 ..])
void launch_dequant_q4(const FfnProblem* probs, int p0, int np, int H, int max_inter, float* stage,
                       size_t stage_stride_elems, FfnProblem* out_probs, cudaStream_t st);

// tensor-core prefill: INT4 images → bf16 hi/lo staging images (lo plane lo_off elements behind the hi plane) + records;
// then silu(g)·u of the [gate | up] GEMM output as the hi/lo activation operand of the down GEMM
void launch_dequant_q4_bf16(const FfnProblem* probs, int p0, int np, int H, int max_inter, __nv_bfloat16* stage, size_t lo_off,
                            size_t stage_stride_elems, FfnProblem* out_probs, cudaStream_t st);
void launch_swiglu_split(const float* gu, const FfnProblem* probs, int p0, int np, int max_rows, int inter, __nv_bfloat16* o_hi,
                         size_t o_lo_off, cudaStream_t st);

// ---- fused decode kernels (kernels_decode.cu) ---------------------------------------------------------------
struct GemvSeg { const void* w; float* out; int n; int flags; };
struct NormGemvArgs {
  const float* x; const float* gain; float eps; int K;
  float* u_out;                       // normalised vector (written by CTA 0) or nullptr
  GemvSeg seg[4]; int nseg;           // plain row segments (router | predictor W1 | shared gate ...)
  const void* wg; const void* wu; float* act; int n_sw;   // SwiGLU pairs of the resident FFN (n_sw = 0: none)
  int n_rows_total;                   // filled by the launcher
};
void launch_norm_multi_gemv(const NormGemvArgs& a, int wdtype, cudaStream_t st);
void launch_attn_decode_fused(const float* qkv, const float* cos_t, const float* sin_t, float* kcache, float* vcache,
                              float* ws, float* out, int* counters, int pos, int nq, int nkv, int d, int max_seq,
                              int nsplit, cudaStream_t st);
void launch_ffn_down_combine(const float* act, int act_stride, const FfnProblem* probs, const int32_t* row_of,
                             const float* gates, int k, const FfnProblem* shared, const float* sact,
                             const float* sgate_logit, const float* shared_y, int H, float* x, int wdtype,
                             size_t chunk_bytes, int* err, cudaStream_t st);
// fused front end of the slot-table kernel for T == 1: top-k + gates on (zraw + bias), predictor W2 GEMV + list
struct RouteFuse {
  const float* zraw; const float* bias; float* z_out; int32_t* sel; float* gates; float* margin;
  const float* p1; const void* pred_w2; int ph; int wdtype; int32_t* pred_out; int k; int cap;
};

// A10 combine: out[t,:] = hres[t,:] + sum_j (fixed j order) g[t,j] * yexp[row(t,j),:] (+ sgate[t]*shared[t,:]).
//  row(t,j) = inv[t*k+j] (prefill) or pos_of_j[j] (decode).  shared may be nullptr; sgate nullptr => 1.
void launch_combine(const float* hres, const float* yexp, const int32_t* row_of, const float* gates, int T, int k,
                    int H, const float* shared, const float* sgate_logit, float* out, cudaStream_t st);
// out[t,:] = a[t,:] + b[t,:]  (dense layer residual)
void launch_add(const float* a, const float* b, float* out, size_t n, cudaStream_t st);

}  // namespace pmk
