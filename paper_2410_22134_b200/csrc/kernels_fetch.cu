// kernels_fetch.cu — A7 for the fused decode step: the DEVICE-SIDE prefetch worker.
//
// PAPER.md Alg. 1 is a worker thread that pops chunk tasks — HIGH (precise) before LOW (predicted), P:179 —
// copies `chunk_size` bytes into the expert's cache slot and bumps `ready_chunk`; Alg. 2 l.12 drops the LOW
// tasks of a layer at its gate (early preemption).  On a B200 that worker is this persistent kernel, launched
// once per decode step on its own high-priority stream: `fetch_ctas` CTAs of two warps — a SCOUT warp that finds out
// what has to be copied (polls the gates, scans flags, claims chunks) and an ENGINE thread that moves the bytes with the
// TMA unit (cp.async.bulk: pinned mapped host memory → shared-memory ring → HBM slot).  It costs no registers to speak
// of, no issue slots and no host round trip.
// Why not the copy engines (profiles/r02_fill_probe.md): SM-issued reads of host memory reach 51.2 GB/s
// against 55.3 GB/s for a cudaMemcpyAsync, but they buy per-chunk readiness for free (a flag copy per chunk costs the
// copy engine 8-30 % of the link, profiles/r01_fill_protocol.md), a gate-to-first-byte latency of ≈ 2 µs instead of a
// ≈ 10 µs host hand-over, LOW chunks that yield to a gate within one chunk, and a decode step the host only enqueues.
//
// Protocol.  The slot-table kernel (A6) writes the command of MoE layer m into a DEVICE ring (same record layout as the
// host command) and then its `seq` word.  Every scout walks the layers in order:
//   wait for gate m (handing out LOW chunks meanwhile) → drop LOW jobs that target m → HIGH: for each needed
//   expert in launch order, every chunk whose flag does not show the slot's generation is CLAIMED (atomicCAS on
//   claims[slot][c]) by whichever CTA gets it and queued for its engine; the engine raises flags[slot][c] ← generation
//   once the chunk's bytes are in HBM → wait for the predicted part of the command → queue its LOW jobs.
// LOW chunks are claimed ONE at a time, by CTA 0 only, with a look at the next gate before each, so a HIGH chunk finds
// at most one LOW chunk in progress and one waiting; what LOW did not reach is fetched as HIGH if the gate needs
// the expert (Alg. 2 loops from ready_chunk).  Nothing here touches the logical slot table.
#include "kernels.h"

#ifdef PMK_FETCH_TRACE      // debug builds only: device printf of the worker's decisions
#include <cstdio>
#define FTRACE(...) do { if ((threadIdx.x & 31) == 0) printf(__VA_ARGS__); } while (0)
#else
#define FTRACE(...) do { } while (0)
#endif

namespace pmk {

constexpr int kFetchPiece = 32768;            // bytes per bulk copy
constexpr int kFetchStages = 6;               // shared-memory ring: 192 KB per CTA
constexpr int kMaxLowJobs = 64;

__device__ __forceinline__ uint32_t fs_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ unsigned ld_acquire_gpu(const unsigned* p) {
  unsigned v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_gpu(unsigned* p, unsigned v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

enum { FC_HIGH_BYTES = 0, FC_LOW_BYTES, FC_LOW_USEFUL, FC_HITS_LANDED, FC_OWED, FC_LANDED, FC_LANDED_OF, FC_FETCHED,
       FC_FETCHED_OF, FC_CHUNKS_HIGH, FC_CHUNKS_LOW, FC_CANCELLED, FC_BUSY_NS, FC_N };

struct LowJob { int layer, slot, expert, cursor; uint32_t gen; };
struct Chunk {                 // one claimed chunk: what to copy and which flag to raise when it is in HBM
  const uint8_t* src; uint8_t* dst; uint32_t* flag; uint32_t gen, bytes; int low;
};
enum { ACQ_OK = 0, ACQ_NONE = 1, ACQ_FINISHED = 2, ACQ_ERROR = 3 };
constexpr int kFetchAhead = kFetchStages - 1;   // loads in flight beside the stage being stored
constexpr int kFetchLag = 4;                    // a chunk's flag is raised once kFetchLag younger stores have been committed
constexpr int kHist = 16;

constexpr int kQueue = 8;
struct FetchQueue {             // scout warp → engine thread, in shared memory
  Chunk q[kQueue];
  volatile unsigned head, tail; // engine takes q[head % kQueue], scout fills q[tail % kQueue]
  volatile int end;             // 0 running, ACQ_FINISHED / ACQ_ERROR once the scout is done
};

// The SCOUT (warp 1 of a fetch CTA): finds out what has to be copied — polls the gates, scans flags and claims, keeps
// the LOW job list — and hands claimed chunks to the engine.  Its L2 round trips (≈ 1 µs each) run beside the copies.
struct Scout {
  const FetchArgs& a;
  LowJob* jobs; FetchQueue* fq;
  int* hi_order;                 // shared: the order in which this gate's needed records are looked at (on_gate)
  int lane;
  int m = 0, phase = 0;          // 0 wait for gate m, 1 HIGH of gate m, 2 wait for the predicted part of gate m, 3 done
  int n_needed = 0, hi_rec = 0, hi_pass = 0, hi_c0 = 0, hi_all = 1;
  unsigned hi_mask = 0; bool hi_scanned = false;
  int head = 0, tail = 0;        // LOW jobs = jobs[head .. tail), FIFO: nearest target layer first
  int low_limit;
  unsigned long long t_start, spins = 0;
  unsigned long long c_high_b = 0, c_low_b = 0, c_high_n = 0, c_low_n = 0;

  __device__ Scout(const FetchArgs& a_, LowJob* j, FetchQueue* q, int* ho) : a(a_), jobs(j), fq(q), hi_order(ho) {
    lane = threadIdx.x & 31; low_limit = a.low_cap > 0 ? min(a.low_cap, a.n_chunks) : a.n_chunks; t_start = globaltimer_ns();
  }
  __device__ void fill(Chunk* out, int layer, int slot, int expert, uint32_t gen, int cc, int low) {
    const size_t so = (size_t)layer * a.C + slot;
    const size_t off = (size_t)cc * a.chunk_bytes;
    out->src = (const uint8_t*)a.src[(size_t)layer * a.E + expert] + off;
    out->dst = a.slots + so * a.Be + off;
    out->flag = a.flags + so * a.n_chunks + cc; out->gen = gen; out->low = low;
    out->bytes = (uint32_t)min((unsigned long long)a.chunk_bytes, a.Be - off);
  }
  // CAS the claim word of chunk cc to (gen, low); warp-uniform result.
  // A copy of an OLDER generation may still be on its way into these bytes: a LOW chunk claimed just before its gate,
  // whose slot the gate has meanwhile given to another expert.  Two engines do not order their writes, so the new copy
  // may only be claimed once the old one has raised its flag (generations grow monotonically: a flag that shows a
  // generation >= the old claim's means nothing of it is in flight any more).
  __device__ int try_claim(uint32_t* fl, uint32_t* cl, int cc, uint32_t gen, int low) {
    int won = 0;
    if (lane == 0) {
      const uint32_t old = ld_acquire_gpu(cl + cc);
      // claims only move FORWARD in generation: a stale LOW job (its slot has been given away at a gate this scout has
      // not looked at yet) must never take a chunk back from the newer image
      if ((old >> 1) < (gen & 0x7fffffffu)) {
        if (old != 0) {
          FTRACE("[scout %d] chunk %d gen %u: old claim %u flag %u\n", blockIdx.x, cc, gen, old, ld_acquire_gpu(fl + cc));
          const unsigned long long t0 = globaltimer_ns();
          while ((ld_acquire_gpu(fl + cc) & 0x7fffffffu) < (old >> 1)) {
            if (globaltimer_ns() - t0 > kFlagTimeoutNs || *(volatile int*)a.err != 0) { atomicExch(a.err, 1); break; }
            __nanosleep(100);
          }
        }
        won = atomicCAS(cl + cc, old, (gen << 1) | (uint32_t)low) == old;
      }
    }
    return __shfl_sync(0xffffffffu, won, 0);
  }
  // chunks [c0, c0 + 32) of a slot: bit i set = chunk c0 + i neither landed nor claimed; *pend = some chunk not landed
  __device__ unsigned scan(const uint32_t* fl, const uint32_t* cl, uint32_t gen, int c0, int limit, int* pend) {
    const int c = c0 + lane;
    int miss = 0, p = 0;
    if (c < limit && ld_acquire_gpu(fl + c) != gen) { p = 1; miss = (ld_acquire_gpu(cl + c) >> 1) < (gen & 0x7fffffffu); }
    *pend = __any_sync(0xffffffffu, p);
    return __ballot_sync(0xffffffffu, miss);
  }
  __device__ int poll(const uint32_t* word, uint32_t seq) {
    unsigned v = 0;
    if (lane == 0) v = ld_acquire_gpu(word);
    return __shfl_sync(0xffffffffu, v, 0) == seq;
  }

  // a gate has been published: early preemption (Alg. 2 l.12) + the byte-accurate view of what had landed
  __device__ void on_gate() {
    const LayerCmd* cmd = a.cmd + m;
    n_needed = __ldcg(&cmd->n_needed);
    FTRACE("[scout %d] gate %d n %d jobs %d\n", blockIdx.x, m, n_needed, tail - head);
    if (a.preempt) {
      int w = head;
      for (int i = head; i < tail; ++i) {
        const LowJob j = jobs[i];
        __syncwarp();
        if (j.layer == m) {
          if (blockIdx.x == 0) {      // chunks that were never claimed = cancelled tasks
            int miss = 0;
            const uint32_t* cl = a.claims + ((size_t)m * a.C + j.slot) * a.n_chunks;
            for (int c = lane; c < a.n_chunks; c += 32) miss += (ld_acquire_gpu(cl + c) >> 1) != (j.gen & 0x7fffffffu);
            for (int o = 16; o > 0; o >>= 1) miss += __shfl_xor_sync(0xffffffffu, miss, o);
            if (lane == 0 && miss) atomicAdd(a.ctr + FC_CANCELLED, (unsigned long long)miss);
          }
          continue;
        }
        if (lane == 0) jobs[w] = j;
        ++w;
        __syncwarp();
      }
      tail = w;
    }
    if (blockIdx.x == 0) {
      for (int i = 0; i < n_needed; ++i) {
        const int32_t* r = (const int32_t*)cmd->need + 7 * i;
        const int cls = __ldcg(r + 1), slot = __ldcg(r + 2);
        const uint32_t gen = (uint32_t)__ldcg(r + 5);
        if (cls == 2) { if (lane == 0) atomicAdd(a.ctr + FC_OWED, (unsigned long long)a.Be); continue; }
        const size_t so = (size_t)m * a.C + slot;
        int landed = 0;
        unsigned long long lowb = 0, missb = 0;
        if (cls == 0 && ld_acquire_gpu(a.complete + so) == gen) landed = a.n_chunks;
        else {
          for (int c = lane; c < a.n_chunks; c += 32) {
            const unsigned long long len = min((unsigned long long)a.chunk_bytes, a.Be - (unsigned long long)c * a.chunk_bytes);
            if (ld_acquire_gpu(a.flags + so * a.n_chunks + c) == gen) {
              ++landed;
              if (ld_acquire_gpu(a.claims + so * a.n_chunks + c) == ((gen << 1) | 1u)) lowb += len;
            } else missb += len;
          }
          for (int o = 16; o > 0; o >>= 1) {
            landed += __shfl_xor_sync(0xffffffffu, landed, o);
            lowb += __shfl_xor_sync(0xffffffffu, lowb, o); missb += __shfl_xor_sync(0xffffffffu, missb, o);
          }
        }
        if (lane == 0) {
          if (landed == a.n_chunks) atomicAdd(a.ctr + FC_HITS_LANDED, 1ull);
          if (missb) atomicAdd(a.ctr + FC_OWED, missb);
          if (cls == 1) {
            atomicAdd(a.ctr + FC_LANDED, (unsigned long long)landed); atomicAdd(a.ctr + FC_LANDED_OF, (unsigned long long)a.n_chunks);
            atomicAdd(a.ctr + FC_FETCHED_OF, 1ull);
            if (landed == a.n_chunks) atomicAdd(a.ctr + FC_FETCHED, 1ull);
            if (lowb) atomicAdd(a.ctr + FC_LOW_USEFUL, lowb);
          }
        }
      }
    }
    // Records that NEED bytes first: class B (a partial prefetch) and class C (nothing there) in launch order, then class A.
    // A class-A image is normally complete, but proving it costs a scan of all its chunk flags the first time it is used
    // after its own fetch (`complete` is only set by a scan that finds every flag raised): with the records taken in launch
    // order A → B → C those scans stood between the gate and the first byte of the missing expert (measured: 9-20 us from
    // the gate word to the first claim; 0.5 us to seeing the word).
    if (n_needed <= 32) {        // decode: one parallel load of the classes, ranks by ballot
      const int cl_ = lane < n_needed ? __ldcg((const int32_t*)cmd->need + 7 * lane + 1) : 0;
      const unsigned need_m = __ballot_sync(0xffffffffu, lane < n_needed && cl_ != 0);
      const unsigned a_m = __ballot_sync(0xffffffffu, lane < n_needed && cl_ == 0);
      const unsigned lt_ = (1u << lane) - 1u;
      if (lane < n_needed) hi_order[cl_ != 0 ? __popc(need_m & lt_) : __popc(need_m) + __popc(a_m & lt_)] = lane;
    } else if (lane == 0) {
      int n = 0;
      for (int i = 0; i < n_needed; ++i) if (__ldcg((const int32_t*)cmd->need + 7 * i + 1) != 0) hi_order[n++] = i;
      for (int i = 0; i < n_needed; ++i) if (__ldcg((const int32_t*)cmd->need + 7 * i + 1) == 0) hi_order[n++] = i;
    }
    __syncwarp();
    hi_rec = 0; hi_pass = 0; hi_c0 = 0; hi_all = 1; hi_mask = 0; hi_scanned = false;
  }

  // the predicted part of gate m has been published: PushPredicted(m + stride) → LOW jobs in listed order (Alg. 2 l.1-10)
  __device__ void on_pred() {
    const LayerCmd* cmd = a.cmd + m;
    const int np = __ldcg(&cmd->n_pred), mt = __ldcg(&cmd->pred_target);
    if (mt >= a.Lm) return;
    for (int i = 0; i < np; ++i) {
      const int32_t* r = (const int32_t*)cmd->pred + 5 * i;
      const int e = __ldcg(r), action = __ldcg(r + 1), slot = __ldcg(r + 2);
      const uint32_t gen = (uint32_t)__ldcg(r + 4);
      if (action == 2 || slot < 0) continue;             // SKIP: no slot was assigned
      if (ld_acquire_gpu(a.complete + (size_t)mt * a.C + slot) == gen) continue;   // touch of a complete image: nothing to copy
      if (tail - head >= kMaxLowJobs) continue;           // cannot happen: <= top_k jobs per push, <= stride pushes pending
      if (tail == kMaxLowJobs) {                          // compact the FIFO to the front of the array
        for (int q = head; q < tail; ++q) { const LowJob t = jobs[q]; __syncwarp(); if (lane == 0) jobs[q - head] = t; __syncwarp(); }
        tail -= head; head = 0;
      }
      if (lane == 0) jobs[tail] = LowJob{mt, slot, e, 0, gen};
      ++tail;
      __syncwarp();
    }
  }

  // Next HIGH chunk of the current gate: the needed experts in launch order (Alg. 2 l.14-21); inside an image this CTA
  // first takes the chunks it owns (chunk index mod #CTAs — no two workers race for a claim), then whatever is left.
  __device__ int next_high(Chunk* out) {
    const LayerCmd* cmd = a.cmd + m;
    while (hi_rec < n_needed) {
      const int32_t* r = (const int32_t*)cmd->need + 7 * hi_order[hi_rec];
      const int e = __ldcg(r), cls_r = __ldcg(r + 1), slot = __ldcg(r + 2);
      const uint32_t gen = (uint32_t)__ldcg(r + 5);
      const size_t so = (size_t)m * a.C + slot;
      uint32_t* fl = a.flags + so * a.n_chunks;
      uint32_t* cl = a.claims + so * a.n_chunks;
      if (cls_r != 2 && !hi_scanned && hi_pass == 0 && hi_c0 == 0 && ld_acquire_gpu(a.complete + so) == gen) { ++hi_rec; continue; }
      while (hi_pass < 2) {
        while (hi_c0 < a.n_chunks) {
          if (!hi_scanned) {
            int pend = 1;
            // class C, own chunks: the slot's generation was made at this gate, so no flag can show it yet and nobody but
            // this CTA goes for these chunks in pass 0 — no need to read 32 flags and 32 claims before the first claim
            if (cls_r == 2 && hi_pass == 0 && gridDim.x > 1) {
              const int left = a.n_chunks - hi_c0;
              hi_mask = left >= 32 ? 0xffffffffu : ((1u << left) - 1u);
            } else hi_mask = scan(fl, cl, gen, hi_c0, a.n_chunks, &pend);
            if (pend) hi_all = 0;
            if (hi_pass == 0 && gridDim.x > 1) {          // own chunks first
              unsigned own = 0;
              for (int b = 0; b < 32; ++b) if ((unsigned)(hi_c0 + b) % gridDim.x == blockIdx.x) own |= 1u << b;
              hi_mask &= own;
            }
            hi_scanned = true;
          }
          while (hi_mask) {
            const int cc = hi_c0 + __ffs(hi_mask) - 1;
            hi_mask &= hi_mask - 1;
            if (try_claim(fl, cl, cc, gen, 0)) { fill(out, m, slot, e, gen, cc, 0); return 1; }
          }
          hi_c0 += 32; hi_scanned = false;
        }
        ++hi_pass; hi_c0 = 0; hi_scanned = false;
        if (gridDim.x == 1) ++hi_pass;
      }
      // nothing left to claim; scans that found every flag at `gen` prove the image complete: later gates skip it
      if (hi_all && lane == 0) st_release_gpu(a.complete + so, gen);
      ++hi_rec; hi_pass = 0; hi_c0 = 0; hi_all = 1; hi_scanned = false;
    }
    return 0;
  }

  // Next chunk to copy: HIGH before LOW; a LOW chunk is handed out only while the next gate has not been
  // published (one poll per chunk = the preemption point; the un-chunked ablation finishes a started image first).
  __device__ int acquire(Chunk* out) {
    while (true) {
      if (phase == 1) {
        if (next_high(out)) return ACQ_OK;
        phase = 2;
      }
      if (phase == 2 && poll((const uint32_t*)&a.cmd[m].seq_pred, a.step * 4096u + (uint32_t)m + 1u)) {
        on_pred();
        ++m;
        phase = m < a.Lm ? 0 : 3;
      }
      if (phase == 0) {
        const bool busy_low = a.unchunked && head < tail && jobs[head].cursor > 0 && jobs[head].cursor < low_limit;
        if (!busy_low && poll((const uint32_t*)&a.cmd[m].seq, a.step * 4096u + (uint32_t)m + 1u)) { on_gate(); phase = 1; continue; }
      }
      // LOW work (also while waiting for the predicted part, and — without early preemption — after the last gate).
      // Only the first low_ctas CTAs copy LOW chunks (default 1): one chunk in progress and one waiting per such CTA bound what
      // a gate can find in its way, whatever the number of workers; the other CTAs keep the list only to know what HIGH
      // must skip.  Several LOW CTAs share a job through the claim words (no chunk is taken twice).
      while (head < tail && (int)blockIdx.x < a.low_ctas) {
        const LowJob j = jobs[head];
        const size_t so = (size_t)j.layer * a.C + j.slot;
        int cur = j.cursor, got = 0;
        for (int c0 = cur; c0 < low_limit && !got; c0 += 32) {
          int pend;
          unsigned mask = scan(a.flags + so * a.n_chunks, a.claims + so * a.n_chunks, j.gen, c0, low_limit, &pend);
          while (mask && !got) {
            const int cc = c0 + __ffs(mask) - 1;
            mask &= mask - 1;
            if (try_claim(a.flags + so * a.n_chunks, a.claims + so * a.n_chunks, cc, j.gen, 1)) { fill(out, j.layer, j.slot, j.expert, j.gen, cc, 1); cur = cc + 1; got = 1; }
          }
          if (!got) cur = min(low_limit, c0 + 32);
        }
        if (lane == 0) jobs[head].cursor = cur;
        __syncwarp();
        if (got) return ACQ_OK;
        ++head;
      }
      if (phase == 3) return ACQ_FINISHED;
      int bad = 0;
      if (lane == 0 && (++spins & 63ull) == 0)
        bad = (*(volatile int*)a.err != 0) || (globaltimer_ns() - t_start > 2 * kFlagTimeoutNs);
      if (__shfl_sync(0xffffffffu, bad, 0)) { if (lane == 0) atomicExch(a.err, 1); return ACQ_ERROR; }
      return ACQ_NONE;
    }
  }

  __device__ void run() {
    unsigned pushed = 0;
    while (true) {
      Chunk c;
      const int r = acquire(&c);
      if (r == ACQ_NONE) { __nanosleep(100); continue; }
      if (r != ACQ_OK) { FTRACE("[scout %d] end %d\n", blockIdx.x, r); if (lane == 0) { __threadfence_block(); fq->end = r; } break; }
      // HIGH chunks may queue up in front of the engine; a LOW chunk only when nothing is waiting (it could not be taken back)
      const unsigned room = c.low ? 1u : (unsigned)kQueue - 1u;
      {   // every wait of the worker is bounded: a protocol error must surface as PROMOE_ETIMEOUT, never as a hang.
          // Lane 0 alone looks at the queue and the warp follows its verdict: with every lane polling for itself, lane 0
          // could leave the loop, push the chunk and let the engine take it — head then runs AHEAD of the `pushed` the
          // slower lanes still hold, `pushed - head` wraps, and they spin until the time-out (seen as 4 s fetch kernels
          // behind decode steps that had long finished)
        const unsigned long long t0 = globaltimer_ns();
        while (true) {
          int full = 0;
          if (lane == 0) {
            full = pushed - fq->head >= room;
            if (full && globaltimer_ns() - t0 > kFlagTimeoutNs) { atomicExch(a.err, 2); full = 0; }
          }
          if (!__shfl_sync(0xffffffffu, full, 0)) break;
          __nanosleep(40);
        }
      }
      FTRACE("[scout %d] push #%u low %d gen %u bytes %u flag %p\n", blockIdx.x, pushed, c.low, c.gen, c.bytes, (void*)c.flag);
      if (lane == 0) { fq->q[pushed % kQueue] = c; __threadfence_block(); fq->tail = pushed + 1; }
      ++pushed;
      if (c.low) { c_low_b += c.bytes; ++c_low_n; } else { c_high_b += c.bytes; ++c_high_n; }
      __syncwarp();
    }
    if (lane == 0) {
      if (c_high_b) atomicAdd(a.ctr + FC_HIGH_BYTES, c_high_b);
      if (c_low_b) atomicAdd(a.ctr + FC_LOW_BYTES, c_low_b);
      if (c_high_n) atomicAdd(a.ctr + FC_CHUNKS_HIGH, c_high_n);
      if (c_low_n) atomicAdd(a.ctr + FC_CHUNKS_LOW, c_low_n);
    }
  }
};

// The ENGINE (thread 0 of a fetch CTA): the copy pipeline.  Bulk loads (pinned host → shared-memory ring) run
// kFetchAhead pieces ahead of the bulk stores (ring → HBM slot), continuously across chunk boundaries; a chunk's flag is
// raised once its last store is known to be in HBM.
__device__ void fetch_engine(const FetchArgs& a, uint8_t* ring, uint64_t* bar, FetchQueue* fq) {
  unsigned long long n_loaded = 0, n_stored = 0, n_flagged = 0, busy_ns = 0, t_busy0 = 0;
  uint32_t* h_flag[kHist]; uint32_t h_gen[kHist];            // per committed store: flag to raise (nullptr: not the last piece)
  uint8_t* st_dst[kFetchStages]; uint32_t st_bytes[kFetchStages]; uint32_t* st_flag[kFetchStages]; uint32_t st_gen[kFetchStages];
  Chunk cur{}; uint32_t cur_off = 0; bool have = false, dead = false;
  unsigned taken = 0;
  const unsigned long long t_begin = globaltimer_ns();
  auto raise = [&](unsigned long long upto) {                // flags of the stores [n_flagged, upto): they are complete
    bool fenced = false;
    for (; n_flagged < upto; ++n_flagged) {
      uint32_t* f = h_flag[n_flagged % kHist];
      if (!f) continue;
      if (!fenced) { asm volatile("fence.proxy.async.global;" ::: "memory"); __threadfence(); fenced = true; }
      st_release_gpu(f, h_gen[n_flagged % kHist]);               // Alg. 1 l.10: ready_chunk
      FTRACE("[engine %d] flag %p <- %u\n", blockIdx.x, (void*)f, h_gen[n_flagged % kHist]);
    }
  };
  while (true) {
    // ---- keep the loads ahead
    while (n_loaded - n_stored < (unsigned long long)kFetchAhead) {
      if (!have) {
        if (fq->tail == taken) break;                         // nothing queued right now
        __threadfence_block();
        cur = fq->q[taken % kQueue];
        ++taken; fq->head = taken;
        have = true; cur_off = 0;
      }
      const int s = (int)(n_loaded % kFetchStages);
      const uint32_t n = min((uint32_t)kFetchPiece, cur.bytes - cur_off);
      const bool fin = cur_off + n == cur.bytes;
      if (n_loaded == n_stored) t_busy0 = globaltimer_ns();
      st_dst[s] = cur.dst + cur_off; st_bytes[s] = n; st_flag[s] = fin ? cur.flag : nullptr; st_gen[s] = cur.gen;
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(fs_u32(bar + s)), "r"(n) : "memory");
      asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                   ::"r"(fs_u32(ring + (size_t)s * kFetchPiece)), "l"(cur.src + cur_off), "r"(n), "r"(fs_u32(bar + s)) : "memory");
      cur_off += n;
      if (fin) have = false;
      ++n_loaded;
    }
    if (n_stored < n_loaded) {
      // ---- the oldest load: wait for it, store it, let the stage of the store before it be reused
      const int s = (int)(n_stored % kFetchStages);
      const uint32_t par = (uint32_t)((n_stored / kFetchStages) & 1);
      uint32_t ok;
      unsigned tries = 0;
      unsigned long long t0 = 0;
      do {
        asm volatile("{\n\t.reg .pred q;\n\tmbarrier.try_wait.parity.shared::cta.b64 q, [%1], %2;\n\tselp.u32 %0, 1, 0, q;\n\t}"
                     : "=r"(ok) : "r"(fs_u32(bar + s)), "r"(par) : "memory");
        if (!ok && (++tries & 1023u) == 0) {
          if (!t0) t0 = globaltimer_ns();
          else if (globaltimer_ns() - t0 > kFlagTimeoutNs) { atomicExch(a.err, 3); dead = true; break; }
        }
      } while (!ok);
      if (dead) break;
      asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                   ::"l"(st_dst[s]), "r"(fs_u32(ring + (size_t)s * kFetchPiece)), "r"(st_bytes[s]) : "memory");
      asm volatile("cp.async.bulk.commit_group;" ::: "memory");
      h_flag[n_stored % kHist] = st_flag[s]; h_gen[n_stored % kHist] = st_gen[s];
      asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");              // every store but this one has left its stage
      asm volatile("cp.async.bulk.wait_group %0;" ::"n"(kFetchLag) : "memory");   // stores older than kFetchLag are in HBM
      ++n_stored;
      if (n_stored > (unsigned long long)kFetchLag) raise(n_stored - kFetchLag);
    } else {
      // ---- pipeline empty: everything committed is in HBM once the group counter drains
      asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
      raise(n_stored);
      if (t_busy0) { busy_ns += globaltimer_ns() - t_busy0; t_busy0 = 0; }
      if (fq->tail == taken) {
        if (fq->end) { if (fq->tail == taken) break; }
        else if (globaltimer_ns() - t_begin > 3 * kFlagTimeoutNs) { atomicExch(a.err, 4); break; }
        else __nanosleep(60);
      }
    }
  }
  atomicMax(a.ctr + FC_BUSY_NS, busy_ns);
  FTRACE("[engine %d] exit stored %llu\n", blockIdx.x, n_stored);
}

__global__ void __launch_bounds__(64, 1) fetch_kernel(FetchArgs a) {
  extern __shared__ __align__(128) uint8_t fsm[];
  __shared__ __align__(8) uint64_t bar[kFetchStages];
  __shared__ LowJob jobs[kMaxLowJobs];
  __shared__ FetchQueue fq;
  __shared__ int hi_order[256];
  if (threadIdx.x == 0) {
    for (int s = 0; s < kFetchStages; ++s) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(fs_u32(bar + s)));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fq.head = 0; fq.tail = 0; fq.end = 0;
    if (blockIdx.x == 0) { __threadfence(); *(volatile uint32_t*)a.alive = a.step; }
  }
  __syncthreads();
  if (threadIdx.x >= 32) { Scout sc(a, jobs, &fq, hi_order); sc.run(); }
  else if (threadIdx.x == 0) fetch_engine(a, fsm, bar, &fq);
}

cudaError_t launch_fetch(const FetchArgs& a, int ctas, cudaStream_t st) {
  ++g_launches;
  static bool attr = false;
  const int smem = kFetchPiece * kFetchStages;
  if (!attr) {
    cudaError_t e = cudaFuncSetAttribute(fetch_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    attr = true;
  }
  fetch_kernel<<<ctas, 64, smem, st>>>(a);
  return cudaGetLastError();
}

// Load every kernel of this file NOW.  CUDA loads kernels lazily, on their first launch, and that load waits for every
// running kernel to finish: a first launch behind a kernel that spins on a flag (an expert kernel waiting for its bytes,
// the fetch worker waiting for a gate) would dead-lock until the spinner times out (profiles/r02_spin_probe.md).
void preload_fetch() {
  preload_fn((const void*)fetch_kernel);
}

}  // namespace pmk
