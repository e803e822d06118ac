// copy_engine.cu — A7, copy-engine path: chunked host→device prefetch on the dedicated copy stream (§5.1
// chunked prefetching P:185-193, §5.2 early preemption P:197-227, Alg. 1, two-priority queue P:179).
//
// Used by PREFILL (and by the unfused decode path kept for tests): there compute is ordered after the fills with
// stream events, the host is in the layer loop anyway, and the copy engines move 55.3 GB/s against 51.2 GB/s for
// SM-issued reads.  The fused decode step fetches with a device-side kernel instead (kernels_fetch.cu).
//
// The slot-table kernel (A6) publishes, per MoE layer, one command record in mapped pinned memory; the step thread
// reads it and
//   * HIGH (precise) fills: every missing chunk is enqueued on the copy stream at once, in launch order — nothing
//     may overtake them, so the stream itself is the queue;
//   * LOW (predicted) fills: kept in a host deque and fed to the stream only `max_inflight` chunks at a time, so a
//     HIGH chunk waits for at most that many (bounded preemption delay), only while no HIGH fill is
//     outstanding; the un-issued LOW chunks of a layer are dropped at that layer's gate (Alg. 2 l.12);
//   * readiness stays per chunk on the device: flags[slot][chunk] = generation, written from the copy stream behind
//     the data (Alg. 1 l.10 `ready_chunk`); the prefill GEMMs are ordered after their fills with stream events.
// Nothing here changes the logical slot table: it lives on the device and advances in program order.
#include "engine.h"

#include <cuda.h>

#include <atomic>
#include <chrono>
#include <cstring>

using namespace pmk;

#define CKC(call)                                                                                  \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess) {                                                                       \
      h->err = std::string(#call) + ": " + cudaGetErrorString(e_);                                 \
      return PROMOE_ECUDA;                                                                         \
    }                                                                                              \
  } while (0)

// retire finished timing slots of the ring; `all` = wait for every one (step end)
int ce_retire(promoe_t* h, bool all) {
  while (h->ev_tail != h->ev_head) {
    const size_t i = h->ev_tail % h->ev_ring.size();
    cudaError_t q = all ? cudaEventSynchronize(h->ev_ring[i]) : cudaEventQuery(h->ev_ring[i]);
    if (q == cudaErrorNotReady) break;
    if (q != cudaSuccess) { h->err = std::string("copy event: ") + cudaGetErrorString(q); return PROMOE_ECUDA; }
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, h->ev_ring_start[i], h->ev_ring[i]) == cudaSuccess) h->st.copy_busy_ms += ms;
    if (h->ev_is_low[i]) h->low_inflight--; else h->high_inflight--;
    h->ev_tail++;
  }
  return PROMOE_OK;
}

static int ring_slot(promoe_t* h, size_t* idx) {
  if (h->ev_head - h->ev_tail >= h->ev_ring.size()) {   // full: wait for the oldest
    const size_t i = h->ev_tail % h->ev_ring.size();
    CKC(cudaEventSynchronize(h->ev_ring[i]));
    int rc = ce_retire(h, false);
    if (rc) return rc;
  }
  *idx = h->ev_head % h->ev_ring.size();
  return PROMOE_OK;
}

// Flags of chunks [p.flagged, p.issued) ← generation, as ONE small copy behind the data copies (measured: a 32-bit
// stream write or a 4-byte copy behind EVERY chunk costs 8-30 % of the link, profiles/r01_fill_protocol.md).
// The source values live in a pinned ring of kFlagSrcRing words; promoe_create bounds n_chunks so that the words of
// every fill that can still be in flight on the copy stream (≤ one per slot of one layer + the LOW chunks) fit
// many times over before an entry is reused.
static int write_flags(promoe_t* h, int m, int s) {
  SlotPhys& p = h->phys[(size_t)m * h->C + s];
  const int n = p.issued - p.flagged;
  if (n <= 0) return PROMOE_OK;
  if (h->flagsrc_pos + (size_t)n > kFlagSrcRing) h->flagsrc_pos = 0;
  uint32_t* v = h->flagsrc_host + h->flagsrc_pos;
  h->flagsrc_pos += (size_t)n;
  for (int i = 0; i < n; ++i) v[i] = p.gen;
  uint32_t* fl = h->flags + ((size_t)m * h->C + s) * h->n_chunks + p.flagged;
  CKC(cudaMemcpyAsync(fl, v, (size_t)n * 4, cudaMemcpyHostToDevice, h->ps));
  p.flagged = p.issued;
  return PROMOE_OK;
}

// HIGH fills that the host issues back to back (all missing experts of one layer) share ONE timing slot: event
// records between the copies cost ≈ 2.5 % of the link (profiles/r01_fill_protocol.md, mode 3 vs plain copies).
static int batch_begin(promoe_t* h) {
  if (h->batch_open) return PROMOE_OK;
  int rc = ring_slot(h, &h->batch_ri);
  if (rc) return rc;
  CKC(cudaEventRecord(h->ev_ring_start[h->batch_ri], h->ps));
  h->batch_open = true; h->batch_used = false;
  return PROMOE_OK;
}
static int batch_end(promoe_t* h) {
  if (!h->batch_open) return PROMOE_OK;
  h->batch_open = false;
  if (!h->batch_used) return PROMOE_OK;        // nothing was copied: the start record is simply re-used later
  CKC(cudaEventRecord(h->ev_ring[h->batch_ri], h->ps));
  h->ev_is_low[h->batch_ri] = 0;
  h->high_inflight++;
  h->ev_head++;
  return PROMOE_OK;
}

// Enqueue chunks [c0, c1) of the fill (layer m, slot s) on the copy stream.  HIGH: `group` chunks per copy
// operation (0 = all of them in one; un-chunked mode: always the whole image), flags written behind every
// operation; LOW: one chunk per call, flags deferred until the fill completes or a HIGH operation takes it over.
static int issue_chunks(promoe_t* h, int m, int s, int c0, int c1, bool low) {
  SlotPhys& p = h->phys[(size_t)m * h->C + s];
  const uint8_t* src = (const uint8_t*)h->expert_host[(size_t)m * h->s.n_experts + p.expert];
  uint8_t* dst = h->slots + ((size_t)m * h->C + s) * h->Be;
  const bool own_slot = !h->batch_open;        // LOW chunks and stand-alone HIGH fills bracket themselves
  size_t ri = h->batch_ri;
  int rc;
  if (own_slot) {
    rc = ring_slot(h, &ri);
    if (rc) return rc;
    CKC(cudaEventRecord(h->ev_ring_start[ri], h->ps));
  } else h->batch_used = true;
  const int group = h->unchunked ? h->n_chunks : low ? 1 : (h->high_group > 0 ? h->high_group : h->n_chunks);
  for (int c = c0; c < c1; c += group) {
    const int ce = std::min(c1, c + group);
    const size_t off = (size_t)c * h->chunk_bytes;
    const size_t len = std::min((size_t)ce * h->chunk_bytes, h->Be) - off;
    CKC(cudaMemcpyAsync(dst + off, src + off, len, cudaMemcpyHostToDevice, h->ps));
    p.issued = ce;
    h->st.h2d_bytes += len;
    h->st.chunks_issued += (uint64_t)(ce - c);
    if (low) { h->st.chunks_low += (uint64_t)(ce - c); h->st.low_bytes += len; p.low_chunks += ce - c; p.low_bytes += len; }
    else { h->st.chunks_high += (uint64_t)(ce - c); h->st.high_bytes += len; }
    if (!low || ce == h->n_chunks) { rc = write_flags(h, m, s); if (rc) return rc; }
  }
  p.fill_seq = h->ev_head + 1;       // complete once the ring tail has passed this slot (the batch's, if batched)
  if (low) p.low_ring.push_back(h->ev_head + 1);
  if (own_slot) {
    CKC(cudaEventRecord(h->ev_ring[ri], h->ps));
    h->ev_is_low[ri] = low ? 1 : 0;
    if (low) h->low_inflight++; else h->high_inflight++;
    h->ev_head++;
  }
  if (c1 == h->n_chunks && h->want_done_events) { CKC(cudaEventRecord(p.done, h->ps)); p.done_valid = true; }
  return PROMOE_OK;
}

// LOW queue ("low-priority tasks are only executed when there are no high-priority tasks"): feed the copy
// stream only while no HIGH fill is outstanding on it, and keep at most max_inflight LOW chunks in flight so that a
// HIGH chunk arriving later waits for at most that many (bounded preemption delay).  On a B200 every bf16
// config is H2D-bound, so a LOW byte may only ever use link time that would otherwise idle.
int ce_pump_low(promoe_t* h) {
  int rc = ce_retire(h, false);
  if (rc) return rc;
  while (!h->low.empty() && h->low_inflight < h->max_inflight && (h->high_inflight == 0 || !h->low_yields)) {
    FillJob& j = h->low.front();
    SlotPhys& p = h->phys[(size_t)j.layer * h->C + j.slot];
    if (p.gen != j.gen || p.expert != j.expert || p.issued >= h->n_chunks ||
        (h->low_cap > 0 && j.low_issued >= h->low_cap)) { h->low.pop_front(); continue; }  // stale / done / capped
    rc = issue_chunks(h, j.layer, j.slot, p.issued, h->unchunked ? h->n_chunks : p.issued + 1, true);
    if (rc) return rc;
    j.low_issued++;
    if (p.issued >= h->n_chunks) h->low.pop_front();
  }
  return PROMOE_OK;
}

// Early preemption (Alg. 2 l.12): drop the un-issued LOW chunks that target layer m.
void ce_cancel_low(promoe_t* h, int m) {
  for (auto it = h->low.begin(); it != h->low.end();) {
    if (it->layer == m) {
      const SlotPhys& p = h->phys[(size_t)m * h->C + it->slot];
      if (p.gen == it->gen && p.issued < h->n_chunks) h->st.chunks_cancelled += (uint64_t)(h->n_chunks - p.issued);
      it = h->low.erase(it);
    } else ++it;
  }
}

// Wait (host) for the command of MoE layer m of step `seq`, pumping LOW chunks meanwhile.
// part 1 = the needed list (PushPrecise), 2 = the predicted list (PushPredicted, published later by the kernel)
int ce_wait_cmd(promoe_t* h, int m, uint32_t seq, int part) {
  volatile uint32_t* w = part == 2 ? &h->cmd_host[m].seq_pred : &h->cmd_host[m].seq;
  const auto t0 = std::chrono::steady_clock::now();
  unsigned spins = 0;
  while (*w != seq) {
    if (!h->low.empty() || h->ev_tail != h->ev_head) {
      int rc = ce_pump_low(h);
      if (rc) return rc;
    }
    if ((++spins & 0x3ff) == 0) {
      if (std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count() > 20.0) {
        cudaError_t e = cudaStreamQuery(h->cs);
        h->err = std::string("timeout waiting for the slot-table command: ") + cudaGetErrorString(e);
        return PROMOE_ETIMEOUT;
      }
    }
  }
  std::atomic_thread_fence(std::memory_order_acquire);
  return PROMOE_OK;
}

// Enqueue (HIGH) whatever is still missing of the fill behind needed record i of layer m; `after` = event the copy
// stream must wait for first (the compute that last read the slot's previous occupant, reading G2) or nullptr.
int ce_issue_needed(promoe_t* h, int m, int i, cudaEvent_t after) {
  const int32_t* r = (const int32_t*)h->cmd_host[m].need + 7 * i;
  SlotPhys& p = h->phys[(size_t)m * h->C + r[2]];
  if (p.issued >= h->n_chunks) return PROMOE_OK;
  if (after) CKC(cudaStreamWaitEvent(h->ps, after, 0));
  if (h->unchunked) { p.issued = 0; p.flagged = 0; }   // un-chunked prefetch (ablation): a partial image cannot be resumed
  // chunks a LOW fill has already put on the stream become visible first (their flags were deferred), so the expert
  // kernels can start on them while the rest of the image is still on the link
  if (p.issued > p.flagged) { int rc = write_flags(h, m, r[2]); if (rc) return rc; }
  return issue_chunks(h, m, r[2], p.issued, h->n_chunks, false);
}

static inline void new_generation(SlotPhys& p, uint32_t gen, int e) {
  p.gen = gen; p.expert = e; p.issued = 0; p.flagged = 0; p.done_valid = false;
  p.low_chunks = 0; p.low_bytes = 0; p.low_ring.clear();
}

// Process the command of MoE layer m: statistics, cancellation, HIGH fills (launch order), LOW jobs.
// Class-C fills whose slot is recycled inside the layer (dep >= 0: prefill with |needed| > C) are NOT
// issued here: their indices are appended to `deferred` and the step scheduler issues them with
// ce_issue_needed once the compute of launch position `dep` has been enqueued.
int ce_process_cmd(promoe_t* h, int m, std::vector<int>* deferred, int parts) {
  const LayerCmd& c = h->cmd_host[m];
  const int n = c.n_needed, E = h->s.n_experts, C = h->C;
  promoe_stats_t& st = h->st;
  { int rc0 = ce_retire(h, false); if (rc0) return rc0; }
  if (parts & 1) {
  if (h->o.flags & PROMOE_F_PREEMPT) ce_cancel_low(h, m);
  // prediction accuracy: |pred ∩ needed| / |pred| for the list pushed into this layer
  std::vector<int32_t>& pend = h->pending_pred[m];
  if (!pend.empty()) {
    st.predicted += pend.size();
    for (int32_t e : pend)
      for (int i = 0; i < n; ++i) if (c.need[7 * i] == e) { st.predicted_correct++; break; }
    pend.clear();
  }
  st.accesses += n;
  { int rcb = batch_begin(h); if (rcb) return rcb; }
  for (int i = 0; i < n; ++i) {
    const int32_t* r = (const int32_t*)c.need + 7 * i;
    const int e = r[0], cls = r[1], s = r[2], victim = r[3], dep = r[4];
    const uint32_t gen = (uint32_t)r[5];
    SlotPhys& p = h->phys[(size_t)m * C + s];
    if (!h->start_resident[(size_t)m * E + e]) st.need_experts++;
    if (cls == 0) st.hits_resident++;
    else if (cls == 1) {
      st.hits_prefetch++;
      st.fetched_at_gate_of++;
      if (p.gen == gen && p.issued >= h->n_chunks && h->ev_tail >= p.fill_seq) st.fetched_at_gate++;
    } else {
      st.misses++;
      if (victim >= 0) st.evictions++;
      h->mirror[(size_t)m * C + s] = e;
    }
    if (dep >= 0 && deferred) { st.owed_bytes_at_gate += h->Be; deferred->push_back(i); continue; }   // slot still in use by launch position dep
    if (p.gen != gen || p.expert != e) new_generation(p, gen, e);   // new allocation of this slot
    if (cls != 2) {       // byte-accurate view of a logical hit (a cancelled prefetch leaves a RESIDENT entry without its bytes)
      int landed = 0;
      for (size_t ri : p.low_ring) landed += h->ev_tail >= ri;
      const bool complete = p.issued >= h->n_chunks && h->ev_tail >= p.fill_seq;
      if (complete) st.hits_landed++;
      if (cls == 1) { st.landed_chunks_at_gate += complete ? h->n_chunks : landed; st.landed_chunks_of += h->n_chunks; st.low_bytes_useful += p.low_bytes; p.low_bytes = 0; }
    }
    if (p.issued < h->n_chunks)
      st.owed_bytes_at_gate += h->Be - std::min(h->Be, (size_t)(h->unchunked ? 0 : p.issued) * h->chunk_bytes);
    int rc = ce_issue_needed(h, m, i, nullptr);
    if (rc) return rc;
  }
  { int rce = batch_end(h); if (rce) return rce; }
  }   // parts & 1
  // PushPredicted(m + stride): LOW jobs (Alg. 2 l.1-10)
  const int mt = c.pred_target;
  if ((parts & 2) && c.n_pred > 0 && mt < h->Lm) {
    std::vector<int32_t>& pd = h->pending_pred[mt];
    pd.clear();
    for (int i = 0; i < c.n_pred; ++i) {
      const int32_t* r = (const int32_t*)c.pred + 5 * i;
      const int e = r[0], action = r[1], s = r[2], victim = r[3];
      const uint32_t gen = (uint32_t)r[4];
      pd.push_back(e);
      if (action == 2) continue;           // SKIP: no victim available
      SlotPhys& p = h->phys[(size_t)mt * C + s];
      if (action == 1) {
        st.pred_allocs++;
        if (victim >= 0) st.evictions++;
        h->mirror[(size_t)mt * C + s] = e;
        new_generation(p, gen, e);
      }
      if (p.issued < h->n_chunks) h->low.push_back(FillJob{mt, s, e, gen, 1, 0});   // alloc, or touch of a cancelled fill (G3)
    }
  }
  return ce_pump_low(h);
}

// Deferred class-C fill: take over the slot physically (the previous occupant's compute is ordered by `after`).
int ce_issue_deferred(promoe_t* h, int m, int i, cudaEvent_t after) {
  const int32_t* r = (const int32_t*)h->cmd_host[m].need + 7 * i;
  SlotPhys& p = h->phys[(size_t)m * h->C + r[2]];
  new_generation(p, (uint32_t)r[5], r[0]);
  return ce_issue_needed(h, m, i, after);
}


// ---- fused decode step: the bytes are moved by the device-side fetch worker (kernels_fetch.cu) --------------------
// Logical statistics of the command of MoE layer m, read from the host command ring AFTER the step (the same
// counters ce_process_cmd keeps on the copy-engine path).
void ce_account_cmd(promoe_t* h, int m) {
  const LayerCmd& c = h->cmd_host[m];
  const int n = c.n_needed, E = h->s.n_experts, C = h->C;
  promoe_stats_t& st = h->st;
  std::vector<int32_t>& pend = h->pending_pred[m];
  if (!pend.empty()) {     // prediction accuracy: |pred ∩ needed| / |pred| for the list pushed into this layer
    st.predicted += pend.size();
    for (int32_t e : pend)
      for (int i = 0; i < n; ++i) if (c.need[7 * i] == e) { st.predicted_correct++; break; }
    pend.clear();
  }
  st.accesses += n;
  for (int i = 0; i < n; ++i) {
    const int32_t* r = (const int32_t*)c.need + 7 * i;
    const int e = r[0], cls = r[1], s = r[2], victim = r[3];
    if (!h->start_resident[(size_t)m * E + e]) st.need_experts++;
    if (cls == 0) st.hits_resident++;
    else if (cls == 1) st.hits_prefetch++;
    else {
      st.misses++;
      if (victim >= 0) st.evictions++;
      h->mirror[(size_t)m * C + s] = e;
    }
  }
  const int mt = c.pred_target;
  if (c.n_pred > 0 && mt < h->Lm) {
    std::vector<int32_t>& pd = h->pending_pred[mt];
    pd.clear();
    for (int i = 0; i < c.n_pred; ++i) {
      const int32_t* r = (const int32_t*)c.pred + 5 * i;
      pd.push_back(r[0]);
      if (r[1] == 1) {
        st.pred_allocs++;
        if (r[3] >= 0) st.evictions++;
        h->mirror[(size_t)mt * C + r[2]] = r[0];
      }
    }
  }
}

// The copy-engine path keeps the physical state of every slot on the host (SlotPhys); the device path keeps it in
// flags[] / tbl.gen.  Before a copy-engine step that follows device-fetched steps: rebuild SlotPhys from the device.
int ce_sync_phys_from_device(promoe_t* h) {
  if (!h->phys_dirty) return PROMOE_OK;
  const int Lm = h->Lm, C = h->C, nc = h->n_chunks;
  std::vector<uint32_t> fl((size_t)Lm * C * nc), gen((size_t)Lm * C);
  std::vector<int32_t> se((size_t)Lm * C);
  CKC(cudaMemcpy(fl.data(), h->flags, fl.size() * 4, cudaMemcpyDeviceToHost));
  CKC(cudaMemcpy(gen.data(), h->tbl.gen, gen.size() * 4, cudaMemcpyDeviceToHost));
  CKC(cudaMemcpy(se.data(), h->tbl.slot_expert, se.size() * 4, cudaMemcpyDeviceToHost));
  for (size_t i = 0; i < h->phys.size(); ++i) {
    SlotPhys& p = h->phys[i];
    int pre = 0;
    while (pre < nc && fl[i * nc + pre] == gen[i]) ++pre;      // chunks are claimed in order: what has landed is a prefix
    p.gen = gen[i]; p.expert = se[i]; p.issued = pre; p.flagged = pre; p.fill_seq = 0; p.done_valid = false;
    p.low_chunks = 0; p.low_bytes = 0; p.low_ring.clear();
  }
  h->phys_dirty = false;
  return PROMOE_OK;
}

// End of a copy-engine step: flags of LOW chunks are deferred until their fill completes; make whatever has been put
// on the stream visible on the device, so that the device path (and a later gate) resumes from it.
int ce_flush_flags(promoe_t* h) {
  for (int m = 0; m < h->Lm; ++m)
    for (int s = 0; s < h->C; ++s) {
      const SlotPhys& p = h->phys[(size_t)m * h->C + s];
      if (p.issued > p.flagged) { int rc = write_flags(h, m, s); if (rc) return rc; }
    }
  return PROMOE_OK;
}
