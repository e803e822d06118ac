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
template <int NPL>
__global__ void __launch_bounds__(256) pred_list_kernel(const float* __restrict__ p, int T, int E, int k, int cap,
                                                        int32_t* __restrict__ pred) {
  __shared__ int votes[32 * NPL];
  __shared__ int s_sel[8][kMaxK];
  __shared__ float s_val[8][kMaxK];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int e = threadIdx.x; e < 32 * NPL; e += 256) votes[e] = 0;
  __syncthreads();
  for (int t = w; t < T; t += 8) {
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
void launch_pred_list(const float* p, int T, int E, int k, int cap, int32_t* pred, cudaStream_t st) {
  ++g_launches;
  if (E <= 32) pred_list_kernel<1><<<1, 256, 0, st>>>(p, T, E, k, cap, pred);
  else if (E <= 64) pred_list_kernel<2><<<1, 256, 0, st>>>(p, T, E, k, cap, pred);
  else if (E <= 128) pred_list_kernel<4><<<1, 256, 0, st>>>(p, T, E, k, cap, pred);
  else pred_list_kernel<8><<<1, 256, 0, st>>>(p, T, E, k, cap, pred);
}

// ---------------------------------------------------------------------------------------------------------
// A8 permutation, single CTA of 1024 threads, no atomics.  Thread i owns the contiguous pair range
// [i*per, (i+1)*per) of the flattened (t, j) list, so "token-ascending inside a group" is preserved:
//   pass 1: per-thread histogram in shared memory cnt[thread][e]  (E <= 256 → processed in expert slabs)
//   pass 2: for each expert, exclusive scan over threads (warp shuffles + one cross-warp step)
//   pass 3: scatter.
// To bound shared memory the experts are processed in slabs of 8; T*k <= 16384.
constexpr int PT = 1024, SLAB = 8;
__global__ void __launch_bounds__(PT) permute_kernel(const int32_t* __restrict__ sel, int n, int E,
                                                     int32_t* __restrict__ count, int32_t* __restrict__ offset,
                                                     int32_t* __restrict__ perm, int32_t* __restrict__ inv) {
  __shared__ int warp_tot[SLAB][32];
  __shared__ int s_count[256];
  __shared__ int s_offset[257];
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int per = (n + PT - 1) / PT;
  const int b = min(n, tid * per), e_ = min(n, b + per);
  // global histogram first (needed for offsets): per-thread partial counts, slab by slab
  for (int e0 = 0; e0 < E; e0 += SLAB) {
    int c[SLAB];
#pragma unroll
    for (int s = 0; s < SLAB; ++s) c[s] = 0;
    for (int i = b; i < e_; ++i) {
      const int d = sel[i] - e0;
#pragma unroll
      for (int s = 0; s < SLAB; ++s) c[s] += (d == s);
    }
#pragma unroll
    for (int s = 0; s < SLAB; ++s) {
      int tot = c[s];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
      if (lane == 0) warp_tot[s][w] = tot;
    }
    __syncthreads();
    if (tid < SLAB && e0 + tid < E) {
      int tot = 0;
      for (int i = 0; i < 32; ++i) tot += warp_tot[tid][i];
      s_count[e0 + tid] = tot;
    }
    __syncthreads();
  }
  if (tid == 0) {
    int acc = 0;
    for (int e = 0; e < E; ++e) { s_offset[e] = acc; acc += s_count[e]; }
    s_offset[E] = acc;
  }
  __syncthreads();
  for (int e = tid; e < E; e += PT) count[e] = s_count[e];
  for (int e = tid; e <= E; e += PT) offset[e] = s_offset[e];
  // scatter, slab by slab: exclusive prefix of this thread's count over lower threads
  for (int e0 = 0; e0 < E; e0 += SLAB) {
    int c[SLAB], pre[SLAB];
#pragma unroll
    for (int s = 0; s < SLAB; ++s) c[s] = 0;
    for (int i = b; i < e_; ++i) {
      const int d = sel[i] - e0;
#pragma unroll
      for (int s = 0; s < SLAB; ++s) c[s] += (d == s);
    }
#pragma unroll
    for (int s = 0; s < SLAB; ++s) {
      int incl = c[s];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int up = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += up;
      }
      pre[s] = incl - c[s];
      if (lane == 31) warp_tot[s][w] = incl;
    }
    __syncthreads();
#pragma unroll
    for (int s = 0; s < SLAB; ++s) {
      int base = 0;
      for (int i = 0; i < w; ++i) base += warp_tot[s][i];
      pre[s] += base;
    }
    for (int i = b; i < e_; ++i) {
      const int ex = sel[i], d = ex - e0;
      if (d >= 0 && d < SLAB) {
        int pos = 0;
#pragma unroll
        for (int s = 0; s < SLAB; ++s)
          if (d == s) { pos = s_offset[ex] + pre[s]; pre[s]++; }
        perm[pos] = i;
        inv[i] = pos;
      }
    }
    __syncthreads();
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
