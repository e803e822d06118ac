// kernels_slot.cu — A6: the device-resident expert-cache slot table (lookup, hit/miss classes, LRU touch,
// eviction, launch order, copy commands).  Logical-time reading of PAPER.md Alg. 2 + Alg. 1 l.3-5
// + §5.3 + §6.1: every table transition happens here, in program order on
// the compute stream; wall-clock only decides how long a consumer waits for bytes.
#include "kernels.h"

namespace pmk {

constexpr int kMaxE = 256;

struct SlotView {
  int32_t* slot_expert; int32_t* expert_slot; unsigned long long* stamp; uint32_t* gen; uint8_t* origin;
  unsigned long long* clock; int C, E;   // all pointers: SHARED-memory copies of one layer's rows (+ a local clock)
  int s0;                                // first slot that may take an allocation (static-cache baseline G21: slots < s0 are fixed)
  __device__ void touch(int s) { stamp[s] = ++(*clock); }
  // Alg. 1 l.4 cache.replace_with: lowest EMPTY slot, else smallest stamp among unprotected slots; -1 if none.
  __device__ int victim(const uint8_t* prot) const {
    for (int s = s0; s < C; ++s) if (slot_expert[s] < 0) return s;
    int best = -1; unsigned long long bs = 0;
    for (int s = s0; s < C; ++s) {
      if (prot[slot_expert[s]]) continue;
      if (best < 0 || stamp[s] < bs) { best = s; bs = stamp[s]; }
    }
    return best;
  }
  __device__ int install(int s, int e, uint8_t org) {
    const int old = slot_expert[s];
    if (old >= 0) expert_slot[old] = -1;
    slot_expert[s] = e; expert_slot[e] = s; origin[s] = org;
    touch(s);
    gen[s] = (uint32_t)(*clock);
    return old;
  }
};

// Fused decode front end, instantiated per experts-per-lane count so that only a small piece of code is fetched
// (a single-CTA kernel runs from a cold instruction cache: code size is latency).
template <int NPL>
__device__ __noinline__ void front_route(const RouteFuse& rf, int E, int lane, int* f_sel, float* f_val) {
  float v[NPL];
#pragma unroll
  for (int q = 0; q < NPL; ++q) {
    const int e = lane + 32 * q;
    v[q] = -INFINITY;
    if (e < E) { v[q] = rf.zraw[e] + (rf.bias ? rf.bias[e] : 0.f); if (rf.z_out) rf.z_out[e] = v[q]; }
  }
  float nxt;
  warp_topk<NPL>(v, E, rf.k, lane, f_sel, f_val, &nxt);
  __syncwarp();
  const float zmax = f_val[0];
  const float ex = (lane < rf.k) ? expf(f_val[lane] - zmax) : 0.f;
  const float sum = warp_sum(ex);
  if (lane < rf.k) { rf.sel[lane] = f_sel[lane]; rf.gates[lane] = ex / sum; }
  if (lane == 0 && rf.margin) rf.margin[0] = (rf.k < E) ? f_val[rf.k - 1] - nxt : INFINITY;
}
template <int NPL>
__device__ __noinline__ void front_pred(const RouteFuse& rf, const float* s_p2, int E, int lane, int* f_sel, float* f_val) {
  float v[NPL];
#pragma unroll
  for (int q = 0; q < NPL; ++q) { const int e = lane + 32 * q; v[q] = (e < E) ? s_p2[e] : -INFINITY; }
  float nxt;
  warp_topk<NPL>(v, E, rf.k, lane, f_sel, f_val, &nxt);
  __syncwarp();
  const int np_ = min(rf.k, rf.cap);
  if (lane == 0) rf.pred_out[0] = np_;
  if (lane < np_) rf.pred_out[1 + lane] = f_sel[lane];
}

__global__ void __launch_bounds__(1024) slot_table_kernel(SlotTable tbl, int m, int stride, int max_spec,
                                                         const int32_t* sel, int T, int k,
                                                         const int32_t* __restrict__ offset,
                                                         const int32_t* pred_list,
                                                         const uint8_t* slot_base, size_t slot_bytes,
                                                         const uint32_t* flag_base, int flags_per_slot, int H,
                                                         int inter, int wbytes, FfnProblem* problems,
                                                         int32_t* n_problems, int32_t* row_of, LayerCmd* cmd,
                                                         uint32_t seq, int32_t* trace_precise,
                                                         int32_t* trace_pred, RouteFuse rf, LayerCmd* cmd2, int mode,
                                                         const LayerCmd* cmd_prev, int* err) {
  __shared__ uint8_t needed[kMaxE];
  __shared__ uint8_t prot[kMaxE];
  __shared__ int16_t order[kMaxE];
  __shared__ uint8_t cls[kMaxE];
  __shared__ int32_t rec[7 * kMaxE];    // staged command records (mapped host memory is write-only here)
  __shared__ int32_t prec[5 * kMaxE];
  __shared__ int s_n, s_np;
  // the table rows of layer m and of the prediction target are staged in shared memory (parallel loads), the
  // serial state machine runs on them, and they are written back in parallel: the kernel sits on the critical
  // path in front of every copy, so no dependent global load may be in the serial part
  __shared__ int32_t t_se[2][kMaxE], t_es[2][kMaxE];
  __shared__ unsigned long long t_stamp[2][kMaxE];
  __shared__ uint32_t t_gen[2][kMaxE];
  __shared__ uint8_t t_org[2][kMaxE];
  __shared__ unsigned long long t_clock;
  __shared__ int32_t s_pred[kMaxE + 1];
  const int E = tbl.E, C = tbl.C;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  pdl_enter();
  __shared__ float s_p2[kMaxE];
  __shared__ int f_sel[2][kMaxK];
  __shared__ float f_val[2][kMaxK];
  __shared__ int32_t s_sel1[kMaxK];
  __shared__ uint8_t prot2[kMaxE];       // membership of the predicted list (one push never evicts its own predictions)
  const int mt_ = m + stride;
  const bool have_t = pred_list != nullptr && mt_ < tbl.Lm;

  // ================= phase 1: route (fused decode only) + PushPrecise(m) → first publication =====================
  // The host needs only this part to issue the HIGH copies, so it is published BEFORE the predictor part runs.
  if (rf.zraw && warp == 0) {     // A4: top-k by logit (ties → lower index), gates = softmax over the selected
    if (E <= 32) front_route<1>(rf, E, lane, f_sel[0], f_val[0]);
    else if (E <= 64) front_route<2>(rf, E, lane, f_sel[0], f_val[0]);
    else if (E <= 128) front_route<4>(rf, E, lane, f_sel[0], f_val[0]);
    else front_route<8>(rf, E, lane, f_sel[0], f_val[0]);
  }
  // The expert kernels of the layer before this one did not wait for the END of that layer's slot-table kernel (gate word),
  // so nothing in the stream order says its table rows have been written back: wait for its `seq_done`.
  if (cmd_prev) {
    __shared__ int prev_ok;
    if (threadIdx.x == 0) prev_ok = wait_gate_word((const unsigned*)&cmd_prev->seq_done, seq - 1u, err);
    __syncthreads();
    (void)prev_ok;      // a time-out raises the error word: the step ends in PROMOE_ETIMEOUT
  }
  for (int i = threadIdx.x; i < C; i += blockDim.x) {
    t_se[0][i] = tbl.slot_expert[(size_t)m * C + i]; t_stamp[0][i] = tbl.stamp[(size_t)m * C + i];
    t_gen[0][i] = tbl.gen[(size_t)m * C + i]; t_org[0][i] = tbl.origin[(size_t)m * C + i];
  }
  for (int e = threadIdx.x; e < E; e += blockDim.x) t_es[0][e] = tbl.expert_slot[(size_t)m * E + e];
  if (threadIdx.x == 0) t_clock = *tbl.clock;
  __shared__ int32_t s_off[kMaxE + 1];    // prefill: group offsets staged in parallel (thread 0 reads them serially below)
  if (offset) for (int e = threadIdx.x; e <= E; e += blockDim.x) s_off[e] = offset[e];
  for (int e = threadIdx.x; e < kMaxE; e += blockDim.x) { needed[e] = 0; prot[e] = 0; prot2[e] = 0; }
  __syncthreads();                // sel (global, written by warp 0 in fused mode) is read below by this same block
  if (T == 1 && threadIdx.x < k) s_sel1[threadIdx.x] = sel[threadIdx.x];
  for (int i = threadIdx.x; i < T * k; i += blockDim.x) { const int e = sel[i]; needed[e] = 1; prot[e] = 1; }   // same-value writes
  __syncthreads();
  // G17 (mode bit 1): a PRED slot whose expert this gate did not select is a misprediction → stamp 0, the next victim
  if (mode & 2)
    for (int i = threadIdx.x; i < C; i += blockDim.x)
      if (t_org[0][i] == 1 && t_se[0][i] >= 0 && !needed[t_se[0][i]]) t_stamp[0][i] = 0;
  __syncthreads();
  int n_built = 0;
  if (threadIdx.x == 0 && !(mode & 1)) {
    // G16: ID-order baseline (Fig. 12 "Base"): ascending id, classified at its turn, plain LRU victim over ALL
    // slots — a needed expert may lose its slot before its turn and is then fetched again (§5.3)
    SlotView v{t_se[0], t_es[0], t_stamp[0], t_gen[0], t_org[0], &t_clock, C, E, mode >> 8};
    int n = 0;
    for (int e = 0; e < E; ++e) if (needed[e]) order[n++] = e;
    if (trace_precise) trace_precise[0] = n;
    for (int e = 0; e < E; ++e) prot[e] = 0;
    for (int i = 0; i < n; ++i) {
      const int e = order[i];
      int32_t* r = rec + 7 * i;
      int sl = v.expert_slot[e];
      if (sl >= 0) {
        cls[i] = v.origin[sl] == 1 ? 1 : 0;
        v.touch(sl);
        r[0] = e; r[1] = cls[i]; r[2] = sl; r[3] = -1; r[4] = -1; r[5] = (int32_t)v.gen[sl];
      } else {
        cls[i] = 2;
        sl = v.victim(prot);
        const int held = v.slot_expert[sl];
        int dep = -1;
        if (held >= 0) for (int q = 0; q < i; ++q) if (order[q] == held) dep = q;
        const int old = v.install(sl, e, 2);
        r[0] = e; r[1] = 2; r[2] = sl; r[3] = old; r[4] = dep; r[5] = (int32_t)v.gen[sl];
      }
    }
    n_built = n;        // hand-over to the common tail below
  }
  if (threadIdx.x == 0 && (mode & 1)) {
    SlotView v{t_se[0], t_es[0], t_stamp[0], t_gen[0], t_org[0], &t_clock, C, E, mode >> 8};
    // classes A (cached) → B (being prefetched) → C (not begun), ascending id inside
    int n = 0;
    if (T == 1) {      // decode: only the k selected experts — sort them by id instead of scanning all E
      int ids[kMaxK];
      for (int j = 0; j < k; ++j) {
        int e = s_sel1[j], q = j;
        while (q > 0 && ids[q - 1] > e) { ids[q] = ids[q - 1]; --q; }
        ids[q] = e;
      }
      for (int c = 0; c < 3; ++c)
        for (int j = 0; j < k; ++j) {
          const int e = ids[j], sl = v.expert_slot[e];
          const int ce = sl < 0 ? 2 : (v.origin[sl] == 1 ? 1 : 0);
          if (ce == c) { order[n] = e; cls[n++] = (uint8_t)c; }
        }
    } else {
      for (int e = 0; e < E; ++e)
        if (needed[e] && v.expert_slot[e] >= 0 && v.origin[v.expert_slot[e]] != 1) { order[n] = e; cls[n++] = 0; }
      for (int e = 0; e < E; ++e)
        if (needed[e] && v.expert_slot[e] >= 0 && v.origin[v.expert_slot[e]] == 1) { order[n] = e; cls[n++] = 1; }
      for (int e = 0; e < E; ++e)
        if (needed[e] && v.expert_slot[e] < 0) { order[n] = e; cls[n++] = 2; }
    }
    if (trace_precise) trace_precise[0] = n;
    // touch A then B (Alg. 2 l.15-17)
    for (int i = 0; i < n && cls[i] != 2; ++i) {
      const int e = order[i], sl = v.expert_slot[e];
      v.touch(sl);
      int32_t* r = rec + 7 * i;
      r[0] = e; r[1] = cls[i]; r[2] = sl; r[3] = -1; r[4] = -1; r[5] = (int32_t)v.gen[sl];
    }
    // class C: alloc; a needed expert not yet computed in launch order is pinned (G2); all pinned → wait for the
    // next finish in launch order.  prot[] == needed[] was prepared in parallel.
    int fin = 0;
    for (int i = 0; i < n; ++i) {
      if (cls[i] != 2) continue;
      const int e = order[i];
      int dep = -1;
      int sl = v.victim(prot);
      while (sl < 0) { prot[order[fin]] = 0; dep = fin; ++fin; sl = v.victim(prot); }
      const int old = v.install(sl, e, 2);
      int32_t* r = rec + 7 * i;
      r[0] = e; r[1] = 2; r[2] = sl; r[3] = old; r[4] = dep; r[5] = (int32_t)v.gen[sl];
    }
    n_built = n;
  }
  if (threadIdx.x == 0) {
    SlotView v{t_se[0], t_es[0], t_stamp[0], t_gen[0], t_org[0], &t_clock, C, E, mode >> 8};
    const int n = n_built;
    for (int sl = 0; sl < C; ++sl) v.origin[sl] = 0;
    // problem table + decode row map + trace
    const size_t hi = wbytes ? (size_t)H * inter * wbytes : (size_t)H * inter / 2;   // wbytes 0: INT4 codes (kernels_q4.cu)
    for (int i = 0; i < n; ++i) {
      const int32_t* r = rec + 7 * i;
      const int e = order[i];
      const int sl = r[2];   // the slot recorded at e's own alloc/touch (a later deferred alloc may recycle it)
      const uint8_t* img = slot_base + ((size_t)m * C + sl) * slot_bytes;
      FfnProblem pb;
      pb.wg = img; pb.wu = img + hi; pb.wd = img + 2 * hi;
      pb.flags = flag_base + ((size_t)m * C + sl) * flags_per_slot;
      pb.gen = (uint32_t)r[5];
      pb.inter = inter;
      pb.row0 = offset ? s_off[e] : i;
      pb.nrows = offset ? s_off[e + 1] - s_off[e] : 1;
      pb.expert = e; pb.pad = 0;
      problems[i] = pb;
      rec[7 * i + 6] = pb.nrows;
      if (trace_precise) for (int q = 0; q < 5; ++q) trace_precise[1 + 5 * i + q] = r[q];
    }
    *n_problems = n;
    if (row_of && T == 1)
      for (int j = 0; j < k; ++j)
        for (int i = 0; i < n; ++i) if (order[i] == s_sel1[j]) row_of[j] = i;
    s_n = n;
  }
  __syncthreads();
  // first publication (posted writes to mapped pinned memory; every writer fences its own stores; seq last)
  // (fused decode: a second copy in device memory feeds the fetch kernel, kernels_fetch.cu — the host copy is only read
  // after the step, for the statistics)
  if (cmd2) {
    // fused decode: the readers of this publication are on the DEVICE (fetch worker, K6's gate word) — device ring first, behind
    // a gpu-scope fence; the mapped host copy (read after the step, for the statistics) follows off the critical path, where the
    // system-scope fence and the posted PCIe writes cost nothing
    for (int i = threadIdx.x; i < 7 * s_n; i += blockDim.x) cmd2->need[i] = rec[i];
    if (threadIdx.x == 0) cmd2->n_needed = s_n;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(&cmd2->seq), "r"(seq) : "memory");
    pdl_done();      // the expert kernels may take their places while the host copy and the predictor half run
    for (int i = threadIdx.x; i < 7 * s_n; i += blockDim.x) cmd->need[i] = rec[i];
    if (threadIdx.x == 0) cmd->n_needed = s_n;
    __threadfence_system();
    __syncthreads();
    if (threadIdx.x == 0) { volatile uint32_t* sq = &cmd->seq; *sq = seq; }
  } else {
    for (int i = threadIdx.x; i < 7 * s_n; i += blockDim.x) cmd->need[i] = rec[i];
    if (threadIdx.x == 0) cmd->n_needed = s_n;
    __threadfence_system();
    __syncthreads();
    if (threadIdx.x == 0) { volatile uint32_t* sq = &cmd->seq; *sq = seq; }
  }

  if (!cmd2) pdl_done();      // the expert kernels may take their places while the predictor half runs
  // ================= phase 2: predictor W2 + list (fused decode only) + PushPredicted(m + stride) =================
  if (rf.zraw && rf.pred_out) {
    const int nwarps = blockDim.x >> 5;
    // compact loops (this single-CTA kernel runs from a cold instruction cache: code size is latency); two rows
    // per warp with both rows' loads issued before any FMA
    for (int e = warp; e < E; e += 2 * nwarps) {
      const int e1 = e + nwarps;
      const bool two = e1 < E;
      float a0 = 0.f, a1 = 0.f;
      if (rf.wdtype == 0) {
        const float* w0 = (const float*)rf.pred_w2 + (size_t)e * rf.ph;
        const float* w1 = (const float*)rf.pred_w2 + (size_t)(two ? e1 : e) * rf.ph;
#pragma unroll 2
        for (int kk = lane * 4; kk + 4 <= rf.ph; kk += 128) {
          float v0[4], v1[4];
          WVec<float>::load(w0 + kk, v0); WVec<float>::load(w1 + kk, v1);
          const float4 xv = *reinterpret_cast<const float4*>(rf.p1 + kk);
          a0 = fmaf(v0[0], xv.x, a0); a0 = fmaf(v0[1], xv.y, a0); a0 = fmaf(v0[2], xv.z, a0); a0 = fmaf(v0[3], xv.w, a0);
          a1 = fmaf(v1[0], xv.x, a1); a1 = fmaf(v1[1], xv.y, a1); a1 = fmaf(v1[2], xv.z, a1); a1 = fmaf(v1[3], xv.w, a1);
        }
      } else {
        const __nv_bfloat16* w0 = (const __nv_bfloat16*)rf.pred_w2 + (size_t)e * rf.ph;
        const __nv_bfloat16* w1 = (const __nv_bfloat16*)rf.pred_w2 + (size_t)(two ? e1 : e) * rf.ph;
#pragma unroll 2
        for (int kk = lane * 8; kk + 8 <= rf.ph; kk += 256) {
          float v0[8], v1[8];
          WVec<__nv_bfloat16>::load(w0 + kk, v0); WVec<__nv_bfloat16>::load(w1 + kk, v1);
          const float4 x0 = *reinterpret_cast<const float4*>(rf.p1 + kk), x1 = *reinterpret_cast<const float4*>(rf.p1 + kk + 4);
          const float xv[8] = {x0.x, x0.y, x0.z, x0.w, x1.x, x1.y, x1.z, x1.w};
#pragma unroll
          for (int q = 0; q < 8; ++q) { a0 = fmaf(v0[q], xv[q], a0); a1 = fmaf(v1[q], xv[q], a1); }
        }
      }
      a0 = warp_sum(a0); a1 = warp_sum(a1);
      if (lane == 0) { s_p2[e] = a0; if (two) s_p2[e1] = a1; }
    }
    __syncthreads();
    if (warp == 0) {              // A5: top-k of the predictor scores, listed by descending score
      if (E <= 32) front_pred<1>(rf, s_p2, E, lane, f_sel[1], f_val[1]);
      else if (E <= 64) front_pred<2>(rf, s_p2, E, lane, f_sel[1], f_val[1]);
      else if (E <= 128) front_pred<4>(rf, s_p2, E, lane, f_sel[1], f_val[1]);
      else front_pred<8>(rf, s_p2, E, lane, f_sel[1], f_val[1]);
    }
  }
  if (have_t) {
    for (int i = threadIdx.x; i < C; i += blockDim.x) {
      t_se[1][i] = tbl.slot_expert[(size_t)mt_ * C + i]; t_stamp[1][i] = tbl.stamp[(size_t)mt_ * C + i];
      t_gen[1][i] = tbl.gen[(size_t)mt_ * C + i]; t_org[1][i] = tbl.origin[(size_t)mt_ * C + i];
    }
    for (int e = threadIdx.x; e < E; e += blockDim.x) t_es[1][e] = tbl.expert_slot[(size_t)mt_ * E + e];
  }
  __syncthreads();                // pred_out (global, written above in fused mode) is read below by this same block
  if (have_t) for (int i = threadIdx.x; i <= E; i += blockDim.x) s_pred[i] = pred_list[i];
  __syncthreads();
  if (have_t) for (int i = threadIdx.x; i < s_pred[0]; i += blockDim.x) prot2[s_pred[1 + i]] = 1;
  __syncthreads();
  if (threadIdx.x == 0) {
    // PushPredicted(m + stride) (Alg. 2 l.1-10): touch cached, alloc missing as PRED; one push never evicts its own
    // predictions; no victim → skip; at most max_spec allocations (knob G3; most confident first)
    int np = 0;
    if (have_t) {
      SlotView t{t_se[1], t_es[1], t_stamp[1], t_gen[1], t_org[1], &t_clock, C, E, mode >> 8};
      np = s_pred[0];
      int allocs = 0;
      for (int i = 0; i < np; ++i) {
        const int e = s_pred[1 + i];
        int32_t* r = prec + 5 * i;
        int sl = t.expert_slot[e];
        if (sl >= 0) { t.touch(sl); r[0] = e; r[1] = 0; r[2] = sl; r[3] = -1; r[4] = (int32_t)t.gen[sl]; }
        else {
          sl = allocs < max_spec ? t.victim(prot2) : -1;
          if (sl >= 0) ++allocs;
          if (sl < 0) { r[0] = e; r[1] = 2; r[2] = -1; r[3] = -1; r[4] = 0; }
          else { const int old = t.install(sl, e, 1); r[0] = e; r[1] = 1; r[2] = sl; r[3] = old; r[4] = (int32_t)t.gen[sl]; }
        }
        if (trace_pred) for (int q = 0; q < 4; ++q) trace_pred[1 + 4 * i + q] = r[q];
      }
    }
    if (trace_pred) trace_pred[0] = np;
    s_np = np;
  }
  __syncthreads();
  // second publication
  for (int i = threadIdx.x; i < 5 * s_np; i += blockDim.x) { cmd->pred[i] = prec[i]; if (cmd2) cmd2->pred[i] = prec[i]; }
  if (threadIdx.x == 0) {
    cmd->n_pred = s_np; cmd->pred_target = m + stride;
    if (cmd2) { cmd2->n_pred = s_np; cmd2->pred_target = m + stride; }
  }
  __threadfence_system();
  __syncthreads();
  if (threadIdx.x == 0) {
    if (cmd2) { volatile uint32_t* s2 = &cmd2->seq_pred; *s2 = seq; }
    volatile uint32_t* sq = &cmd->seq_pred; *sq = seq;
  }
  // write the staged rows back
  for (int i = threadIdx.x; i < C; i += blockDim.x) {
    tbl.slot_expert[(size_t)m * C + i] = t_se[0][i]; tbl.stamp[(size_t)m * C + i] = t_stamp[0][i];
    tbl.gen[(size_t)m * C + i] = t_gen[0][i]; tbl.origin[(size_t)m * C + i] = t_org[0][i];
    if (have_t) {
      tbl.slot_expert[(size_t)mt_ * C + i] = t_se[1][i]; tbl.stamp[(size_t)mt_ * C + i] = t_stamp[1][i];
      tbl.gen[(size_t)mt_ * C + i] = t_gen[1][i]; tbl.origin[(size_t)mt_ * C + i] = t_org[1][i];
    }
  }
  for (int e = threadIdx.x; e < E; e += blockDim.x) {
    tbl.expert_slot[(size_t)m * E + e] = t_es[0][e];
    if (have_t) tbl.expert_slot[(size_t)mt_ * E + e] = t_es[1][e];
  }
  if (threadIdx.x == 0) *tbl.clock = t_clock;
  if (cmd2) {           // table rows are back in global memory: the next layer's kernel may read them
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(&cmd2->seq_done), "r"(seq) : "memory");
  }
}

void launch_slot_table(SlotTable tbl, int m, int stride, int max_spec, const int32_t* sel, int T, int k, const int32_t* offset,
                       const int32_t* pred_list, int reorder, const uint8_t* slot_base, size_t slot_bytes,
                       const uint32_t* flag_base, int flags_per_slot, int H, int inter, int wbytes,
                       FfnProblem* problems, int32_t* n_problems, int32_t* row_of, LayerCmd* cmd, uint32_t seq,
                       int32_t* trace_precise, int32_t* trace_pred, cudaStream_t st, const RouteFuse* rf, LayerCmd* cmd_dev2,
                       const LayerCmd* cmd_prev, int* err) {
  ++g_launches;
  const int mode = reorder;     // bit 0: reordered inference / 0 = ID order (G16); bit 1: demote mispredictions (G17);
                                // bits 8+: number of fixed slots of the static-cache baseline (G21)
  RouteFuse f{};
  if (rf) f = *rf;
  launch_pdl(slot_table_kernel, dim3(1), dim3((rf && T == 1) ? 1024 : 256), 0, st, tbl, m, stride, max_spec, sel, T, k, offset, pred_list,
             slot_base, slot_bytes, flag_base, flags_per_slot, H, inter, wbytes, problems, n_problems, row_of, cmd, seq,
             trace_precise, trace_pred, f, cmd_dev2, mode, cmd_prev, err);
}

// Load every kernel of this file NOW.  CUDA loads kernels lazily, on their first launch, and that load waits for every
// running kernel to finish: a first launch behind a kernel that spins on a flag (an expert kernel waiting for its bytes,
// the fetch worker waiting for a gate) would dead-lock until the spinner times out (profiles/r02_spin_probe.md).
void preload_slot() {
  preload_fn((const void*)slot_table_kernel);
}

}  // namespace pmk
