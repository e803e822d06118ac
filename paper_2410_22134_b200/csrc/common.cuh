// common.cuh — device helpers shared by the ProMoE sm_100a kernels (product code; shares nothing with oracle/).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace pmk {

constexpr int kWarp = 32;

// ---- programmatic dependent launch (PDL): the decode step is a chain of ~8 short kernels per layer; launching
// kernel n+1 while kernel n drains hides its launch / block-scheduling latency.  Every PDL-launched kernel calls
// pdl_enter() before its first global access: it lets ITS dependents be scheduled and then waits until the kernel
// in front of it has completed and flushed (so at most the prologue overlaps — no data hazard is possible).
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
// Where the trigger sits decides how long the dependent's CTAs sit resident (at griddepcontrol.wait) beside the running
// kernel.  At the top of the kernel the whole run-ahead queue of the decode step cascades onto the SMs (every kernel
// triggers its successor as soon as it is resident) and takes registers and thread slots from the one kernel that is
// actually running; after the main loop only the NEXT kernel overlaps, with the tail of this one.
#ifndef PMK_PDL_LATE
#define PMK_PDL_LATE 1
#endif
__device__ __forceinline__ void pdl_enter() { if (!PMK_PDL_LATE) pdl_trigger(); pdl_wait(); }
__device__ __forceinline__ void pdl_done() { if (PMK_PDL_LATE) pdl_trigger(); }
extern bool g_use_pdl;   // PROMOE_PDL=0 disables (A/B measurements)
template <typename... KArgs, typename... Args>
inline void launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = g_use_pdl ? 1 : 0;
  cfg.attrs = at; cfg.numAttrs = 1;
  cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

// force the (lazy) load of one kernel; see preload_* in every kernels_*.cu
inline void preload_fn(const void* f) { cudaFuncAttributes a; (void)cudaFuncGetAttributes(&a, f); }
void preload_dense(); void preload_attn(); void preload_route(); void preload_slot(); void preload_decode();
void preload_ffn(); void preload_tc(); void preload_fetch(); void preload_q4();
inline void preload_all() {
  preload_dense(); preload_attn(); preload_route(); preload_slot(); preload_decode(); preload_ffn(); preload_tc(); preload_fetch(); preload_q4();
}

// number of kernels launched by this library (host-side counter, bumped by every launch_* wrapper; promoe_stats)
extern unsigned long long g_launches;

// ---- 16-byte vectorised weight loads, widened exactly to fp32 (weights are bf16 or fp32; G1) -------------
template <typename WT> struct WVec;
template <> struct WVec<float> {
  static constexpr int N = 4;  // elements per 16-byte load
  __device__ __forceinline__ static void load(const float* p, float (&v)[4]) {
    float4 r = __ldcs(reinterpret_cast<const float4*>(p));
    v[0] = r.x; v[1] = r.y; v[2] = r.z; v[3] = r.w;
  }
};
template <> struct WVec<__nv_bfloat16> {
  static constexpr int N = 8;
  __device__ __forceinline__ static void load(const __nv_bfloat16* p, float (&v)[8]) {
    uint4 r = __ldcs(reinterpret_cast<const uint4*>(p));
    // bf16 -> fp32 is a 16-bit shift
    v[0] = __uint_as_float(r.x << 16); v[1] = __uint_as_float(r.x & 0xffff0000u);
    v[2] = __uint_as_float(r.y << 16); v[3] = __uint_as_float(r.y & 0xffff0000u);
    v[4] = __uint_as_float(r.z << 16); v[5] = __uint_as_float(r.z & 0xffff0000u);
    v[6] = __uint_as_float(r.w << 16); v[7] = __uint_as_float(r.w & 0xffff0000u);
  }
};
__device__ __forceinline__ float wload1(const float* p) { return *p; }
__device__ __forceinline__ float wload1(const __nv_bfloat16* p) { return __bfloat162float(*p); }

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ float silu(float a) { return a / (1.0f + expf(-a)); }

// ---- one weight row · x, fp32 accumulate: the HBM-streaming inner loop of every decode GEMV -------------------
// K must be a multiple of the 16-byte vector width; the summation order depends on (K, lane) only, so results
// are bit-identical wherever the row lives (slot, shared expert, any launch order).
template <typename WT, int UNR = 4>
__device__ __forceinline__ float row_dot(const WT* __restrict__ wrow, const float* __restrict__ x, int K, int lane) {
  constexpr int V = WVec<WT>::N;
  float acc[UNR];
#pragma unroll
  for (int u = 0; u < UNR; ++u) acc[u] = 0.f;
  int k = lane * V;
  const int step = 32 * V;
  for (; k + (UNR - 1) * step + V <= K; k += UNR * step) {
    float wv[UNR][V];
#pragma unroll
    for (int u = 0; u < UNR; ++u) WVec<WT>::load(wrow + k + u * step, wv[u]);
#pragma unroll
    for (int u = 0; u < UNR; ++u) {
      const float4* xp = reinterpret_cast<const float4*>(x + k + u * step);
#pragma unroll
      for (int q = 0; q < V / 4; ++q) {
        float4 xv = __ldg(xp + q);
        acc[u] = fmaf(wv[u][4 * q + 0], xv.x, acc[u]);
        acc[u] = fmaf(wv[u][4 * q + 1], xv.y, acc[u]);
        acc[u] = fmaf(wv[u][4 * q + 2], xv.z, acc[u]);
        acc[u] = fmaf(wv[u][4 * q + 3], xv.w, acc[u]);
      }
    }
  }
  for (; k + V <= K; k += step) {
    float wv[V];
    WVec<WT>::load(wrow + k, wv);
#pragma unroll
    for (int q = 0; q < V; ++q) acc[0] = fmaf(wv[q], __ldg(x + k + q), acc[0]);
  }
  float tot = 0.f;
  if (UNR == 4) tot = (acc[0] + acc[1]) + (acc[2] + acc[3]);
  else {
#pragma unroll
    for (int u = 0; u < UNR; ++u) tot += acc[u];
  }
  return warp_sum(tot);
}


// row_dot for SHORT rows (K <= NP passes of 32 lanes x 16 bytes; NP = 8: 2048 bf16 / 1024 fp32 elements): every load of the
// row is issued before the first FMA (row_dot keeps 4 in flight and then walks the tail one dependent load at a time:
// 3 latency rounds for K = 1408).  Same accumulators, same order → bit-identical to row_dot<WT, 4>.
template <typename WT> struct WRaw;
template <> struct WRaw<float> {
  typedef float4 T;
  __device__ __forceinline__ static T load(const float* p) { return __ldcs(reinterpret_cast<const float4*>(p)); }
  __device__ __forceinline__ static void cvt(const T& r, float (&v)[4]) { v[0] = r.x; v[1] = r.y; v[2] = r.z; v[3] = r.w; }
};
template <> struct WRaw<__nv_bfloat16> {
  typedef uint4 T;
  __device__ __forceinline__ static T load(const __nv_bfloat16* p) { return __ldcs(reinterpret_cast<const uint4*>(p)); }
  __device__ __forceinline__ static void cvt(const T& r, float (&v)[8]) {
    v[0] = __uint_as_float(r.x << 16); v[1] = __uint_as_float(r.x & 0xffff0000u);
    v[2] = __uint_as_float(r.y << 16); v[3] = __uint_as_float(r.y & 0xffff0000u);
    v[4] = __uint_as_float(r.z << 16); v[5] = __uint_as_float(r.z & 0xffff0000u);
    v[6] = __uint_as_float(r.w << 16); v[7] = __uint_as_float(r.w & 0xffff0000u);
  }
};
template <typename WT, int NP = 8>
__device__ __forceinline__ float row_dot_short(const WT* __restrict__ wrow, const float* __restrict__ x, int K, int lane) {
  constexpr int V = WVec<WT>::N;
  const int step = 32 * V, k0 = lane * V;
  typename WRaw<WT>::T raw[NP];
#pragma unroll
  for (int j = 0; j < NP; ++j)
    if (k0 + j * step + V <= K) raw[j] = WRaw<WT>::load(wrow + k0 + j * step);
  float acc[4] = {0.f, 0.f, 0.f, 0.f};
  bool main_ok = true;      // row_dot's main loop takes 4 passes at a time while the 4th exists, then the tail feeds acc[0]
#pragma unroll
  for (int j = 0; j < NP; ++j) {
    const int k = k0 + j * step;
    if ((j & 3) == 0) main_ok = main_ok && (k + 3 * step + V <= K);
    if (k + V <= K) {
      float wv[V];
      WRaw<WT>::cvt(raw[j], wv);
      float a = main_ok ? acc[j & 3] : acc[0];
#pragma unroll
      for (int q = 0; q < V / 4; ++q) {
        const float4 xv = __ldg(reinterpret_cast<const float4*>(x + k) + q);
        a = fmaf(wv[4 * q + 0], xv.x, a); a = fmaf(wv[4 * q + 1], xv.y, a);
        a = fmaf(wv[4 * q + 2], xv.z, a); a = fmaf(wv[4 * q + 3], xv.w, a);
      }
      if (main_ok) acc[j & 3] = a; else acc[0] = a;
    }
  }
  return warp_sum((acc[0] + acc[1]) + (acc[2] + acc[3]));
}


constexpr int kMaxK = 16;
// ---------------------------------------------------------------------------------------------------------
// Warp-shuffle top-k.  One warp per token; lane holds experts lane, lane+32, ... (NPL per lane, E <= 32*NPL).
// Selection order: descending value, ties → lower index (BASELINE.json north_star).
// Returns in lane j (j < k) nothing: winners are written by lane 0 through the callback arrays.
template <int NPL>
__device__ __forceinline__ void warp_topk(float (&v)[NPL], int E, int k, int lane, int* sel_out, float* val_out,
                                          float* next_val) {
  // sel_out / val_out: per-warp shared or global arrays of length k, written by lane 0.
  for (int it = 0; it <= k; ++it) {
    float best = -INFINITY; int bi = 0x7fffffff;
#pragma unroll
    for (int q = 0; q < NPL; ++q) {
      const int e = lane + 32 * q;
      if (e < E && (v[q] > best || (v[q] == best && e < bi))) { best = v[q]; bi = e; }
    }
    // lanes with nothing left keep bi = INT_MAX and best = -inf
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const float ob = __shfl_xor_sync(0xffffffffu, best, o);
      const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
      if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
    }
    if (it == k) { *next_val = (bi == 0x7fffffff) ? -INFINITY : best; break; }
    if (lane == 0) { sel_out[it] = bi; val_out[it] = best; }
    // retire the winner
#pragma unroll
    for (int q = 0; q < NPL; ++q)
      if (lane + 32 * q == bi) v[q] = -INFINITY;
    if (it + 1 == E) { *next_val = -INFINITY; break; }   // k == E: nothing left
  }
}


// ---- chunk-ready flags (Alg. 1 l.10 `ready_chunk`) --------------------------------------
// flag[c] holds the allocation generation whose chunk c has landed in this slot.  Written by the copy stream
// (DMA), read here with a system-scope acquire load.
__device__ __forceinline__ unsigned ld_acquire_sys(const unsigned* p) {
  unsigned v;
  asm volatile("ld.acquire.sys.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ unsigned long long globaltimer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
constexpr unsigned long long kFlagTimeoutNs = 4000000000ull;  // 4 s: then give up and raise the error word

// One thread waits until flags[c0..c1] == gen.  Returns false on timeout (error word set).
__device__ inline bool wait_chunks(const unsigned* flags, int c0, int c1, unsigned gen, int* err) {
  if (flags == nullptr) return true;
  unsigned long long t0 = 0;
  for (int c = c0; c <= c1; ++c) {
    while (ld_acquire_sys(flags + c) != gen) {
      if (t0 == 0) t0 = globaltimer_ns();
      if (globaltimer_ns() - t0 > kFlagTimeoutNs || *reinterpret_cast<volatile int*>(err) != 0) {
        atomicExch(err, 1);
        return false;
      }
      __nanosleep(256);
    }
  }
  return true;
}

// Gate word (fused decode): a kernel that needs only the FIRST half of the kernel in front of it waits for the word that
// kernel publishes (release) behind that half instead of griddepcontrol.wait, which would wait for all of it.
__device__ inline bool wait_gate_word(const unsigned* word, unsigned want, int* err) {
  unsigned long long t0 = 0;
  unsigned v;
  while (true) {
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(word) : "memory");
    if (v == want) return true;
    if (t0 == 0) t0 = globaltimer_ns();
    if (globaltimer_ns() - t0 > kFlagTimeoutNs || (err && *reinterpret_cast<volatile int*>(err) != 0)) { if (err) atomicExch(err, 1); return false; }
    __nanosleep(64);
  }
}

// One FFN problem = one SwiGLU MLP applied to a row range.  Routed experts: written
// by the slot-table kernel; shared/dense FFNs: written once at load time.
struct FfnProblem {
  const void* wg;          // [inter, H]
  const void* wu;          // [inter, H]
  const void* wd;          // [H, inter]
  const unsigned* flags;   // chunk flags of the slot, or nullptr (always resident)
  unsigned gen;            // generation the flags must show
  int inter;
  int row0, nrows;         // rows of the (permuted) activation matrix this problem covers
  int expert;              // routed expert id, or -1
  int pad;
};
static_assert(sizeof(FfnProblem) % 8 == 0, "FfnProblem is read in 8-byte pieces");
// a record written by a kernel that is still running (gate word): read past L1, 8 bytes at a time (records are 8-byte aligned)
__device__ __forceinline__ FfnProblem load_problem_cg(const FfnProblem* p) {
  FfnProblem pb;
  const unsigned long long* src = reinterpret_cast<const unsigned long long*>(p);
  unsigned long long* dst = reinterpret_cast<unsigned long long*>(&pb);
#pragma unroll
  for (int q = 0; q < (int)(sizeof(FfnProblem) / 8); ++q) dst[q] = __ldcg(src + q);
  return pb;
}

}  // namespace pmk
