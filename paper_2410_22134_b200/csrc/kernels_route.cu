// kernels_route.cu — router top-k + gate softmax (A4), predictor list (A5), token→expert permutation (A8),
// weighted combine (A10).  sm_100a.
#include "kernels.h"

namespace pmk {


// A4: z (+bias) → sel [T,k], gates = softmax over the selected logits (Σ = 1, reading G8), margin.
template <int NPL>
__global__ void __launch_bounds__(128) topk_gate_kernel(const float* __restrict__ z, const float* __restrict__ bias,
                                                        int T, int E, int k, float* __restrict__ z_out,
                                                        int32_t* __restrict__ sel, float* __restrict__ gates,
                                                        float* __restrict__ margin) {
  __shared__ int s_sel[4][kMaxK];
  __shared__ float s_val[4][kMaxK];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int t = blockIdx.x * 4 + w;
  if (t >= T) return;
  float v[NPL];
#pragma unroll
  for (int q = 0; q < NPL; ++q) {
    const int e = lane + 32 * q;
    v[q] = -INFINITY;
    if (e < E) {
      v[q] = z[(size_t)t * E + e] + (bias ? bias[e] : 0.f);
      if (z_out) z_out[(size_t)t * E + e] = v[q];
    }
  }
  float nxt;
  warp_topk<NPL>(v, E, k, lane, s_sel[w], s_val[w], &nxt);
  __syncwarp();
  const float zmax = s_val[w][0];
  float ex = (lane < k) ? expf(s_val[w][lane] - zmax) : 0.f;
  const float sum = warp_sum(ex);
  if (lane < k) {
    sel[(size_t)t * k + lane] = s_sel[w][lane];
    gates[(size_t)t * k + lane] = ex / sum;
  }
  if (lane == 0 && margin) margin[t] = (k < E) ? s_val[w][k - 1] - nxt : INFINITY;
}
void launch_topk_gate(const float* z, const float* bias, int T, int E, int k, float* z_out, int32_t* sel,
                      float* gates, float* margin, cudaStream_t st) {
  ++g_launches;
  const int blocks = (T + 3) / 4;
  if (E <= 32) topk_gate_kernel<1><<<blocks, 128, 0, st>>>(z, bias, T, E, k, z_out, sel, gates, margin);
  else if (E <= 64) topk_gate_kernel<2><<<blocks, 128, 0, st>>>(z, bias, T, E, k, z_out, sel, gates, margin);
  else if (E <= 128) topk_gate_kernel<4><<<blocks, 128, 0, st>>>(z, bias, T, E, k, z_out, sel, gates, margin);
  else topk_gate_kernel<8><<<blocks, 128, 0, st>>>(z, bias, T, E, k, z_out, sel, gates, margin);
}

// ---------------------------------------------------------------------------------------------------------
// A5 predictor list.  One CTA.  T == 1: the top-k list of p.  T > 1 (reading G7): per-token top-k →
// vote histogram (shared-memory integer atomics: order-independent, hence deterministic) → experts by votes
// descending, ties → lower id → the first min(#voted, cap).
// grid of CTAs (8 warps, one token per warp and turn); T > 1: every CTA adds its vote histogram into ws[0..E) (integer
// atomics: the sums do not depend on the order) and the LAST CTA to arrive (ws[256]) ranks the experts and leaves ws zeroed
// for the next call.  (One CTA for all tokens took 100 us at T = 512 — on the pre-gate critical path of every prefill layer.)
template <int NPL>
__global__ void __launch_bounds__(256) pred_list_kernel(const float* __restrict__ p, int T, int E, int k, int cap,
                                                        int32_t* __restrict__ pred, int32_t* __restrict__ ws) {
  __shared__ int votes[32 * NPL];
  __shared__ int s_sel[8][kMaxK];
  __shared__ float s_val[8][kMaxK];
  __shared__ int s_last;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int e = threadIdx.x; e < 32 * NPL; e += 256) votes[e] = 0;
  __syncthreads();
  for (int t = blockIdx.x * 8 + w; t < T; t += gridDim.x * 8) {
    float v[NPL];
#pragma unroll
    for (int q = 0; q < NPL; ++q) {
      const int e = lane + 32 * q;
      v[q] = (e < E) ? p[(size_t)t * E + e] : -INFINITY;
    }
    float nxt;
    warp_topk<NPL>(v, E, k, lane, s_sel[w], s_val[w], &nxt);
    __syncwarp();
    if (T == 1) {
      if (lane == 0) pred[0] = min(k, cap);
      if (lane < min(k, cap)) pred[1 + lane] = s_sel[w][lane];
    } else if (lane < k) {
      atomicAdd(&votes[s_sel[w][lane]], 1);
    }
    __syncwarp();
  }
  if (T == 1) return;
  __syncthreads();
  if (gridDim.x > 1) {
    for (int e = threadIdx.x; e < E; e += 256) if (votes[e]) atomicAdd(&ws[e], votes[e]);
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(&ws[256], 1) == (int)gridDim.x - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    for (int e = threadIdx.x; e < 32 * NPL; e += 256) votes[e] = e < E ? __ldcg(&ws[e]) : 0;
    __syncthreads();
    for (int e = threadIdx.x; e < E; e += 256) ws[e] = 0;      // leave the workspace zeroed for the next call
    if (threadIdx.x == 0) ws[256] = 0;
  }
  // rank of expert e among voted experts by (votes desc, id asc)
  int nvoted = 0;
  for (int e = 0; e < E; ++e) nvoted += votes[e] > 0;
  for (int e = threadIdx.x; e < E; e += 256) {
    const int ve = votes[e];
    if (ve == 0) continue;
    int rank = 0;
    for (int f = 0; f < E; ++f) rank += (votes[f] > ve) || (votes[f] == ve && f < e);
    if (rank < cap) pred[1 + rank] = e;
  }
  if (threadIdx.x == 0) pred[0] = min(nvoted, cap);
}
void launch_pred_list(const float* p, int T, int E, int k, int cap, int32_t* pred, cudaStream_t st, int32_t* ws) {
  ++g_launches;
  const int blocks = (ws && T > 8) ? min(64, (T + 7) / 8) : 1;      // ws: 257 zeroed int32 (votes + arrival counter)
  if (E <= 32) pred_list_kernel<1><<<blocks, 256, 0, st>>>(p, T, E, k, cap, pred, ws);
  else if (E <= 64) pred_list_kernel<2><<<blocks, 256, 0, st>>>(p, T, E, k, cap, pred, ws);
  else if (E <= 128) pred_list_kernel<4><<<blocks, 256, 0, st>>>(p, T, E, k, cap, pred, ws);
  else pred_list_kernel<8><<<blocks, 256, 0, st>>>(p, T, E, k, cap, pred, ws);
}

// ---------------------------------------------------------------------------------------------------------
// A8 permutation: stable counting sort of the flattened (t, j) pairs by expert — one CTA of 32 warps, no atomics.
// Warp w owns the contiguous pair range [w*per, (w+1)*per) and walks it 32 pairs at a time; inside a chunk
// `__match_any_sync` groups the lanes that hold the same expert, so a pair's rank among the chunk's pairs of its expert is
// a popcount and one leader lane per expert updates the warp's own counter row — "token-ascending inside a group" holds
// because ranges, chunks and lanes are all in pair order.
//   pass 1: per-warp histograms cnt[w][e];  scan: base[w][e] = Σ_{w' < w} cnt[w'][e], count[e], offset[e];
//   pass 2: pos = offset[e] + base[w][e] + rank in chunk, then base[w][e] += pairs of e in the chunk.
// Three block-wide barriers in all (the first version made 16 slab passes: 54 us at T·k = 2048, on the pre-gate critical path).
constexpr int PT = 1024, PW = PT / 32;
__global__ void __launch_bounds__(PT) permute_kernel(const int32_t* __restrict__ sel, int n, int E,
                                                     int32_t* __restrict__ count, int32_t* __restrict__ offset,
                                                     int32_t* __restrict__ perm, int32_t* __restrict__ inv) {
  __shared__ int cnt[PW][256];
  __shared__ int s_offset[257];
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int per = ((n + PW - 1) / PW + 31) & ~31;          // pairs per warp, a multiple of 32
  const int b = min(n, w * per), e_ = min(n, b + per);
  const unsigned lt = (1u << lane) - 1u;
  for (int e = lane; e < E; e += 32) cnt[w][e] = 0;
  __syncwarp();
  for (int i0 = b; i0 < e_; i0 += 32) {
    const int i = i0 + lane;
    const bool act = i < e_;
    const int ex = act ? sel[i] : -1 - lane;                  // inactive lanes: distinct keys that match nobody
    const unsigned m = __match_any_sync(0xffffffffu, ex);
    if (act && (m & lt) == 0) cnt[w][ex] += __popc(m);        // leader = lowest lane of the group
    __syncwarp();
  }
  __syncthreads();
  for (int e = tid; e < E; e += PT) {                         // exclusive scan over the warps, per expert
    int acc = 0;
    for (int q = 0; q < PW; ++q) { const int c = cnt[q][e]; cnt[q][e] = acc; acc += c; }
    count[e] = acc;
    s_offset[e + 1] = acc;                                    // totals, turned into offsets below
  }
  __syncthreads();
  if (w == 0) {                                               // exclusive scan over the experts (E <= 256: 8 per lane)
    int loc[8], tot = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) { const int e = lane * 8 + q; loc[q] = e < E ? s_offset[e + 1] : 0; tot += loc[q]; }
    int incl = tot;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int up = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += up; }
    int run = incl - tot;
    if (lane == 0) s_offset[0] = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) { const int e = lane * 8 + q; run += loc[q]; if (e < E) s_offset[e + 1] = run; }
  }
  __syncthreads();
  for (int e = tid; e <= E; e += PT) offset[e] = s_offset[e];
  for (int i0 = b; i0 < e_; i0 += 32) {
    const int i = i0 + lane;
    const bool act = i < e_;
    const int ex = act ? sel[i] : -1 - lane;
    const unsigned m = __match_any_sync(0xffffffffu, ex);
    int basev = 0;
    if (act) basev = cnt[w][ex];
    __syncwarp();
    if (act) {
      const int pos = s_offset[ex] + basev + __popc(m & lt);
      perm[pos] = i;
      inv[i] = pos;
      if ((m & lt) == 0) cnt[w][ex] = basev + __popc(m);
    }
    __syncwarp();
  }
}
void launch_permute(const int32_t* sel, int T, int k, int E, int32_t* count, int32_t* offset, int32_t* perm,
                    int32_t* inv, cudaStream_t st) {
  ++g_launches;
  permute_kernel<<<1, PT, 0, st>>>(sel, T * k, E, count, offset, perm, inv);
}

// ---------------------------------------------------------------------------------------------------------
// A10 combine: out[t,:] = hres[t,:] + Σ_j (ascending j) g[t,j]·yexp[row(t,j),:] (+ σ(sgate_logit[t])·shared[t,:]).
__global__ void __launch_bounds__(256) combine_kernel(const float* __restrict__ hres, const float* __restrict__ yexp,
                                                      const int32_t* __restrict__ row_of,
                                                      const float* __restrict__ gates, int k, int H,
                                                      const float* __restrict__ shared,
                                                      const float* __restrict__ sgate_logit, float* __restrict__ out) {
  const int t = blockIdx.x;
  float sg = 1.f;
  if (sgate_logit) sg = 1.f / (1.f + expf(-sgate_logit[t]));
  for (int c = threadIdx.x; c < H; c += 256) {
    float y = 0.f;
    for (int j = 0; j < k; ++j)
      y = fmaf(gates[(size_t)t * k + j], yexp[(size_t)row_of[(size_t)t * k + j] * H + c], y);
    if (shared) y += sg * shared[(size_t)t * H + c];
    out[(size_t)t * H + c] = hres[(size_t)t * H + c] + y;
  }
}
void launch_combine(const float* hres, const float* yexp, const int32_t* row_of, const float* gates, int T, int k,
                    int H, const float* shared, const float* sgate_logit, float* out, cudaStream_t st) {
  ++g_launches;
  combine_kernel<<<T, 256, 0, st>>>(hres, yexp, row_of, gates, k, H, shared, sgate_logit, out);
}

// Load every kernel of this file NOW.  CUDA loads kernels lazily, on their first launch, and that load waits for every
// running kernel to finish: a first launch behind a kernel that spins on a flag (an expert kernel waiting for its bytes,
// the fetch worker waiting for a gate) would dead-lock until the spinner times out (profiles/r02_spin_probe.md).
void preload_route() {
  preload_fn((const void*)topk_gate_kernel<1>);
  preload_fn((const void*)topk_gate_kernel<2>);
  preload_fn((const void*)topk_gate_kernel<4>);
  preload_fn((const void*)topk_gate_kernel<8>);
  preload_fn((const void*)pred_list_kernel<1>);
  preload_fn((const void*)pred_list_kernel<2>);
  preload_fn((const void*)pred_list_kernel<4>);
  preload_fn((const void*)pred_list_kernel<8>);
  preload_fn((const void*)permute_kernel);
  preload_fn((const void*)combine_kernel);
}

}  // namespace pmk
