// engine.h — the promoe handle: device buffers, slot region, copy engine state.  Internal to the library.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <deque>
#include <string>
#include <vector>

#include "../../include/promoe.h"
#include "kernels.h"

namespace pmk {
struct TcContext;

// One expert fill = all chunks of one expert image into one slot (Alg. 1: tasks of one expert, in chunk order).
struct FillJob {
  int layer, slot, expert;
  uint32_t gen;
  int prio;  // 0 HIGH, 1 LOW
  int low_issued = 0;   // chunks this LOW job has put on the copy stream (capped by low_cap_chunks)
};
// Physical state of a slot (what the copy stream has been asked to do), as opposed to the logical table on
// the device.  issued = chunks of generation `gen` already enqueued on the copy stream, in chunk order.
struct SlotPhys {
  uint32_t gen = 0;
  int expert = -1;
  int issued = 0;
  int flagged = 0;              // chunks whose ready flag write has been enqueued (<= issued)
  size_t fill_seq = 0;          // ring sequence of the last copy operation of this slot
  cudaEvent_t done = nullptr;   // recorded after the last chunk of the current generation
  bool done_valid = false;
  int low_chunks = 0;           // chunks of the current generation that were moved by LOW (predicted) copies
  size_t low_bytes = 0;         // their bytes, not yet attributed to useful / wasted
  std::vector<size_t> low_ring; // ring sequence of each of them (landed once the ring tail has passed it)
};
constexpr size_t kFlagSrcRing = 1u << 20;   // words in the pinned ring the flag copies read their generation values from
constexpr int kMaxChunks = 8192;            // chunks per expert image (promoe_create rejects smaller chunk sizes)

}  // namespace pmk

struct promoe {
  promoe_shape_t s{};
  promoe_opts_t o{};
  int Lm = 0, C = 0, wb = 2, n_chunks = 0, max_inflight = 2;
  int wdd = 1;                 // dtype of the DENSE weights (0 fp32, 1 bf16); wdtype 2 = bf16 dense + INT4 routed experts
  bool q4 = false;             // routed experts are INT4 group-quantised images (kernels_q4.cu)
  float* q4_stage = nullptr;   // prefill (SIMT): fp32 staging images of the needed experts [E, 3*H*I]
  __nv_bfloat16* q4_stage_bf = nullptr;   // prefill (tcgen05): bf16 hi plane [E, 3*H*I], lo plane q4_lo_off elements later
  size_t q4_lo_off = 0;
  float* q4_gu = nullptr;      // [maxT*k, 2*I] fp32 [gate | up] pre-activations of the INT4 tensor-core prefill
  pmk::FfnProblem* problems_deq = nullptr;   // records pointing into q4_stage
  size_t Be = 0, chunk_bytes = 0;
  int max_spec_decode = 0, max_spec_prefill = 0;   // allocations allowed per PushPredicted (knob G3)
  int maxT = 0, qkv_w = 0, ffn_w = 0, nsplit = 1;
  cudaStream_t cs = nullptr, ps = nullptr;
  cudaStream_t cs2 = nullptr;                 // side compute stream: the shared expert runs beside the slot-table kernel
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  bool own_cs = false, dense_loaded = false, experts_loaded = false;
  std::string err;

  // dense weights: host copies of the per-layer device-pointer arrays
  const void *emb = nullptr, *lm_head = nullptr;
  const float* final_norm = nullptr;
  std::vector<const float*> ln1, ln2, router_bias;
  std::vector<const void*> wqkv, wo, router, pred_w1, pred_w2, ffn_gate, ffn_up, ffn_down, shared_gate_w;
  std::vector<const void*> expert_host;   // [Lm*E] pinned host images
  std::vector<void*> registered;          // buffers we had to cudaHostRegister

  // activations (fp32)
  float *x = nullptr, *u1 = nullptr, *u = nullptr, *qkv = nullptr, *attn = nullptr, *zraw = nullptr;
  float *p1 = nullptr, *p2 = nullptr, *act = nullptr, *yexp = nullptr, *sact = nullptr, *sy = nullptr;
  float *sgate = nullptr, *attn_ws = nullptr, *xf = nullptr, *logits = nullptr;
  float *kcache = nullptr, *vcache = nullptr, *cos_t = nullptr, *sin_t = nullptr;
  int32_t* ids = nullptr;
  // per-MoE-layer routing / permutation buffers (double as traces)
  int32_t *sel = nullptr, *count = nullptr, *offset = nullptr, *perm = nullptr, *inv = nullptr;
  float *gates = nullptr, *margin = nullptr, *z = nullptr;
  int32_t* votes_ws = nullptr;            // [257] zeroed: vote histogram + arrival counter of the multi-CTA predictor list kernel
  float* trace_u = nullptr;               // [Lm, maxT, H] with PROMOE_F_TRACE_U, else nullptr
  int32_t *pred_list = nullptr, *trace_precise = nullptr, *trace_pred = nullptr, *row_of = nullptr,
          *n_prob = nullptr;
  pmk::FfnProblem *problems = nullptr, *shared_prob = nullptr;
  int* err_dev = nullptr;
  // pinned host staging: no pageable buffer is ever handed to an async copy (a pageable D2H above the driver's
  // staging threshold was seen to stall the copy stream for seconds while a flag-gated kernel was resident)
  float* logits_pin = nullptr;
  int32_t* ids_pin = nullptr;
  int* err_pin = nullptr;
  int* attn_cnt = nullptr;       // [n_q_heads] arrival counters of the fused decode attention (zero between launches)
  // tcgen05 path (PROMOE_F_TENSOR, bf16 weights): activation operands as bf16 hi/lo planes; the lo plane of each
  // buffer starts *_half elements after the hi plane
  pmk::TcContext* tc = nullptr;
  __nv_bfloat16 *xsA = nullptr, *xsG = nullptr, *xsB = nullptr;   // direct rows | gathered rows | SwiGLU outputs
  size_t xsA_half = 0, xsG_half = 0, xsB_half = 0;

  // expert cache
  uint8_t* slots = nullptr;       // ONE contiguous region [Lm, C, Be]
  uint32_t* flags = nullptr;      // [Lm, C, n_chunks]
  pmk::SlotTable tbl{};
  pmk::LayerCmd* cmd_host = nullptr;   // mapped pinned, [Lm]
  pmk::LayerCmd* cmd_dev = nullptr;
  uint32_t* flagsrc_host = nullptr;       // pinned ring holding the generation values the flag copies read
  size_t flagsrc_pos = 0;

  // copy engine (host)
  std::vector<pmk::SlotPhys> phys;     // [Lm*C]
  std::deque<pmk::FillJob> low;
  std::vector<cudaEvent_t> ev_ring;       // per-chunk end events (timing enabled)
  std::vector<cudaEvent_t> ev_ring_start;
  size_t ev_head = 0, ev_tail = 0;        // in flight = [tail, head)
  std::vector<int> ev_is_low;
  int low_inflight = 0, high_inflight = 0;
  bool batch_open = false, batch_used = false;   // HIGH fills of one command share one timing slot
  size_t batch_ri = 0;
  int low_cap = 0;                    // LOW fills stop after this many chunks (0 = no cap)
  int high_group = 0;                 // chunks per HIGH copy operation, 0 = whole remaining fill in one copy
  bool want_done_events = false;      // prefill: per-fill completion events for cudaStreamWaitEvent
  bool low_yields = true;             // LOW chunks wait while HIGH fills are outstanding
  std::vector<cudaEvent_t> done_ev;       // prefill: per launch position "expert finished" events
  cudaEvent_t step_start = nullptr, step_end = nullptr;

  // host mirror for statistics
  std::vector<int32_t> mirror;            // [Lm*C] slot -> expert
  std::vector<uint8_t> start_resident;    // [Lm*E]
  std::vector<std::vector<int32_t>> pending_pred;  // per target layer
  std::vector<int32_t> trace_pred_host_lists;      // predictor_mode TRACE input [Lm*(1+E)]
  promoe_stats_t st{};
  bool unchunked = false;             // ablation: a fill is all or nothing (no resume from ready_chunk, "without chunking")
  int dev = 0;
  // device-side fetch worker of the fused decode step (kernels_fetch.cu)
  cudaStream_t fs = nullptr;              // its stream (highest priority)
  pmk::LayerCmd* cmd_fetch = nullptr;     // device copy of the command ring [Lm]
  uint32_t *claims = nullptr, *complete = nullptr, *alive = nullptr;
  unsigned long long *fetch_ctr = nullptr, *fetch_ctr_pin = nullptr;   // device counters / pinned host copy
  unsigned long long* src_dev = nullptr;  // [Lm*E] device-visible addresses of the host expert images
  int fetch_ctas = 4;
  bool phys_dirty = false;                // the device path has moved bytes since the host's SlotPhys was last synced
  int pos = 0;                            // position of sequence 0 (= seq_pos[0]; kept for the single-sequence calls)
  int max_batch = 1;
  int static_slots = 0;                   // static-cache baseline (G21): slots [0, static_slots) of every layer never take an allocation
  std::vector<int> seq_pos;               // [max_batch] tokens held by each sequence
  size_t kv_seq_elems = 0;                // elements of one sequence's K (or V) cache: L * nkv * max_seq * d
  // the step being enqueued: which sequence(s) its rows belong to (run_step / run_batch_step set these)
  int cur_n_seq = 1; int cur_seq[8] = {0}; int cur_pos[8] = {0}; bool cur_batch = false;
  uint32_t step_seq = 0;
  int last_T = 0;
  std::vector<uint8_t> trace_buf;         // host staging for promoe_get_trace
};
