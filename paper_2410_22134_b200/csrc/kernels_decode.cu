// kernels_decode.cu — fused kernels of the batch-1 decode step (T == 1).  The unfused step launched 19 kernels per
// layer, each 4-15 µs of mostly ramp-up (profiles/r01_launches_c2_small.md): 170 µs/layer of compute against 27 µs
// of HBM time, all of it exposed in front of the H2D copies.  Fused step, per MoE layer:
//   K1 norm_multi_gemv   RMSNorm(ln1) + QKV GEMV
//   K2 attn_decode_fused RoPE + KV append + split attention + last-block merge
//   K3 gemv_kernel       O-projection + residual                                   (kernels_dense.cu)
//   K4 norm_multi_gemv   RMSNorm(ln2) + router | predictor W1 (ReLU) | shared-gate GEMVs (dense layer: + FFN gate/up)
//   K5 slot_table_kernel top-k + gates + predictor W2 + predicted list + slot table (kernels_slot.cu, fused mode)
//   K5b ffn_gateup_gemv  shared expert gate/up — enqueued behind K5 to cover the host hand-over
//   K6 ffn_gateup_gemv   routed experts gate/up, flag-gated                        (kernels_ffn.cu)
//   K7 ffn_down_combine  routed + shared down GEMVs + weighted combine (fixed j order) + residual
#include "kernels.h"

namespace pmk {

// x·w row dot with x in SHARED memory (same lane/k order as row_dot → same summation order for a given K).
template <typename WT>
__device__ __forceinline__ float row_dot_s(const WT* __restrict__ wrow, const float* xs, int K, int lane) {
  constexpr int V = WVec<WT>::N;
  constexpr int UNR = 4;
  float acc[UNR] = {0.f, 0.f, 0.f, 0.f};
  int k = lane * V;
  const int step = 32 * V;
  for (; k + (UNR - 1) * step + V <= K; k += UNR * step) {
    float wv[UNR][V];
#pragma unroll
    for (int u = 0; u < UNR; ++u) WVec<WT>::load(wrow + k + u * step, wv[u]);
#pragma unroll
    for (int u = 0; u < UNR; ++u) {
      const float4* xp = reinterpret_cast<const float4*>(xs + k + u * step);
#pragma unroll
      for (int q = 0; q < V / 4; ++q) {
        const float4 xv = xp[q];
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
    for (int q = 0; q < V; ++q) acc[0] = fmaf(wv[q], xs[k + q], acc[0]);
  }
  return warp_sum((acc[0] + acc[1]) + (acc[2] + acc[3]));
}

// ---------------------------------------------------------------------------------------------------------------
// K1 / K4 / lm_head: u = RMSNorm(x; gain) staged once per CTA in shared memory, then one warp per weight row over a
// list of segments.  Persistent grid (≤ 148·6 CTAs = one resident wave; the QKV GEMV of c2/c3 is 768 CTAs, which at
// 48 registers / 5 CTAs per SM spilled into a 28-CTA second wave), rows dealt round-robin to warps.
template <typename WT>
__global__ void __launch_bounds__(256, 6) norm_multi_gemv_kernel(NormGemvArgs a) {
  extern __shared__ float xs[];            // [K]
  __shared__ float red[8];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  pdl_enter();
  float ss = 0.f;
  for (int i = threadIdx.x; i < a.K; i += 256) { const float v = a.x[i]; xs[i] = v; ss += v * v; }
  ss = warp_sum(ss);
  if (lane == 0) red[warp] = ss;
  __syncthreads();
  float tot = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) tot += red[i];
  const float r = rsqrtf(tot / (float)a.K + a.eps);
  for (int i = threadIdx.x; i < a.K; i += 256) {
    const float v = xs[i] * r * a.gain[i];
    xs[i] = v;
    if (a.u_out && blockIdx.x == 0) a.u_out[i] = v;
  }
  __syncthreads();
  const int total = a.n_rows_total;
  for (int row = blockIdx.x * 8 + warp; row < total; row += gridDim.x * 8) {
    int rr = row, s = 0;
    while (s < a.nseg && rr >= a.seg[s].n) { rr -= a.seg[s].n; ++s; }
    if (s < a.nseg) {
      float v = row_dot_s<WT>((const WT*)a.seg[s].w + (size_t)rr * a.K, xs, a.K, lane);
      if (lane == 0) {
        if (a.seg[s].flags & LIN_RELU) v = fmaxf(v, 0.f);
        a.seg[s].out[rr] = v;
      }
    } else {   // SwiGLU pair of the always-resident FFN: act[rr] = silu(Wg[rr]·u) · (Wu[rr]·u)
      const float g = row_dot_s<WT>((const WT*)a.wg + (size_t)rr * a.K, xs, a.K, lane);
      const float v = row_dot_s<WT>((const WT*)a.wu + (size_t)rr * a.K, xs, a.K, lane);
      if (lane == 0) a.act[rr] = silu(g) * v;
    }
  }
  pdl_done();
}
void launch_norm_multi_gemv(const NormGemvArgs& a_in, int wdtype, cudaStream_t st) {
  ++g_launches;
  NormGemvArgs a = a_in;
  a.n_rows_total = a.n_sw;
  for (int s = 0; s < a.nseg; ++s) a.n_rows_total += a.seg[s].n;
  int blocks = (a.n_rows_total + 7) / 8;
  if (blocks > 148 * 6) blocks = 148 * 6;   // 6 CTAs resident per SM (40 registers, __launch_bounds__(256, 6)): one wave
  if (blocks < 1) blocks = 1;
  const size_t smem = (size_t)a.K * sizeof(float);
  if (wdtype == 0) launch_pdl(norm_multi_gemv_kernel<float>, dim3(blocks), dim3(256), smem, st, a);
  else launch_pdl(norm_multi_gemv_kernel<__nv_bfloat16>, dim3(blocks), dim3(256), smem, st, a);
}

// ---------------------------------------------------------------------------------------------------------------
// K2: RoPE(q, k_new) + KV append + split attention over the cache + merge by the last CTA of each head.
// grid (nq, nsplit), 128 threads; 8 lanes share a key (d/8 contiguous floats each).  The new position `pos` is
// served from shared memory (rotated k, raw v) by every CTA whose split contains it; exactly one CTA per kv head
// also writes it into the cache.  counters[nq] must be zero on entry and is left zero.
constexpr int kMaxSplit = 64;
template <int D>
__global__ void __launch_bounds__(128) attn_decode_fused_kernel(const float* __restrict__ qkv,
                                                                const float* __restrict__ cos_t,
                                                                const float* __restrict__ sin_t,
                                                                float* __restrict__ kcache, float* __restrict__ vcache,
                                                                float* __restrict__ ws, float* __restrict__ out,
                                                                int* __restrict__ counters, int pos, int nq, int nkv,
                                                                int max_seq, int nsplit) {
  constexpr int PER = D / 8, HALF = D / 2;
  pdl_enter();
  const int h = blockIdx.x, sp = blockIdx.y;
  const int grp_sz = nq / nkv, g = h / grp_sz;
  const int sub = threadIdx.x & 7, grp = threadIdx.x >> 3;
  const int n_pos = pos + 1;
  __shared__ float sm_q[D], sm_k[D], sm_v[D];
  __shared__ float sm_m[16], sm_l[16], sm_o[16][D];
  __shared__ int s_last;
  const float scale = rsqrtf((float)D);
  if (threadIdx.x < HALF) {     // rotate-half RoPE of q (head h) and of the new k (kv head g)
    const int i = threadIdx.x;
    const float c = cos_t[(size_t)pos * HALF + i], s = sin_t[(size_t)pos * HALF + i];
    const float* qh = qkv + (size_t)h * D;
    const float* kh = qkv + (size_t)(nq + g) * D;
    const float* vh = qkv + (size_t)(nq + nkv + g) * D;
    const float q1 = qh[i], q2 = qh[i + HALF], k1 = kh[i], k2 = kh[i + HALF];
    sm_q[i] = (q1 * c - q2 * s) * scale; sm_q[i + HALF] = (q2 * c + q1 * s) * scale;
    sm_k[i] = k1 * c - k2 * s; sm_k[i + HALF] = k2 * c + k1 * s;
    sm_v[i] = vh[i]; sm_v[i + HALF] = vh[i + HALF];
  }
  __syncthreads();
  const int per_split = (n_pos + nsplit - 1) / nsplit;
  const int p0 = sp * per_split, p1 = min(n_pos, p0 + per_split);
  float* kb = kcache + (size_t)g * max_seq * D;
  float* vb = vcache + (size_t)g * max_seq * D;
  if ((h % grp_sz) == 0 && pos >= p0 && pos < p1) {     // the one writer of this kv head's new row
    for (int i = threadIdx.x; i < D; i += 128) { kb[(size_t)pos * D + i] = sm_k[i]; vb[(size_t)pos * D + i] = sm_v[i]; }
  }
  float q[PER];
#pragma unroll
  for (int i = 0; i < PER; ++i) q[i] = sm_q[sub * PER + i];
  float m = -INFINITY, l = 0.f, o[PER];
#pragma unroll
  for (int i = 0; i < PER; ++i) o[i] = 0.f;
  // NB passes of 16 keys per round: the loads of all NB passes are issued before the first is consumed (the loop is
  // latency-bound: 3-5 dependent passes at decode lengths); the arithmetic is per pass, in pass order, as before.
  constexpr int NB = 3;
  for (int pb0 = p0; pb0 < p1; pb0 += 16 * NB) {      // uniform trip counts: the 8-lane shuffles use the full mask
    float kv[NB][PER], vv[NB][PER];
#pragma unroll
    for (int j = 0; j < NB; ++j) {
      const int p = pb0 + 16 * j + grp;
      if (p < p1) {
        if (p == pos) {
#pragma unroll
          for (int i = 0; i < PER; ++i) { kv[j][i] = sm_k[sub * PER + i]; vv[j][i] = sm_v[sub * PER + i]; }
        } else {
          const float4* kr = reinterpret_cast<const float4*>(kb + (size_t)p * D + sub * PER);
          const float4* vr = reinterpret_cast<const float4*>(vb + (size_t)p * D + sub * PER);
#pragma unroll
          for (int i = 0; i < PER / 4; ++i) {
            const float4 a = __ldcs(kr + i), b = __ldcs(vr + i);
            kv[j][4 * i] = a.x; kv[j][4 * i + 1] = a.y; kv[j][4 * i + 2] = a.z; kv[j][4 * i + 3] = a.w;
            vv[j][4 * i] = b.x; vv[j][4 * i + 1] = b.y; vv[j][4 * i + 2] = b.z; vv[j][4 * i + 3] = b.w;
          }
        }
      }
    }
#pragma unroll
    for (int j = 0; j < NB; ++j) {
      if (pb0 + 16 * j >= p1) break;                  // uniform over the CTA
      const bool valid = pb0 + 16 * j + grp < p1;
      float s = 0.f;
      if (valid) {
#pragma unroll
        for (int i = 0; i < PER; ++i) s = fmaf(q[i], kv[j][i], s);
      }
      s += __shfl_xor_sync(0xffffffffu, s, 1);
      s += __shfl_xor_sync(0xffffffffu, s, 2);
      s += __shfl_xor_sync(0xffffffffu, s, 4);
      if (!valid) continue;
      const float mn = fmaxf(m, s);
      const float corr = expf(m - mn), pw = expf(s - mn);
      l = l * corr + pw;
#pragma unroll
      for (int i = 0; i < PER; ++i) o[i] = o[i] * corr + pw * vv[j][i];
      m = mn;
    }
  }
  pdl_done();
  // merge the 16 key groups of this CTA (fixed order)
  if (sub == 0) { sm_m[grp] = m; sm_l[grp] = l; }
#pragma unroll
  for (int i = 0; i < PER; ++i) sm_o[grp][sub * PER + i] = o[i];
  __syncthreads();
  float M = -INFINITY;
  for (int i = 0; i < 16; ++i) M = fmaxf(M, sm_m[i]);
  float* wout = ws + ((size_t)h * nsplit + sp) * (D + 2);
  for (int c = threadIdx.x; c < D; c += 128) {
    float acc = 0.f;
    for (int i = 0; i < 16; ++i) if (sm_m[i] != -INFINITY) acc += sm_o[i][c] * expf(sm_m[i] - M);
    wout[c] = acc;
  }
  if (threadIdx.x == 0) {
    float L = 0.f;
    for (int i = 0; i < 16; ++i) if (sm_m[i] != -INFINITY) L += sm_l[i] * expf(sm_m[i] - M);
    wout[D] = M; wout[D + 1] = L;
  }
  // last CTA of this head merges the splits (fixed split order → deterministic whoever arrives last)
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) {
    const int old = atomicAdd(counters + h, 1);
    s_last = (old == nsplit - 1);
    if (s_last) counters[h] = 0;
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  // (M, L) of every split staged in shared memory by one load round, partial rows read with all loads of a
  // 16-split group in flight (L2 loads: the partials were written by other SMs); same arithmetic order as a serial
  // loop over the splits.
  const float* base = ws + (size_t)h * nsplit * (D + 2);
  __shared__ float sm_M[kMaxSplit], sm_L[kMaxSplit];
  for (int s2 = threadIdx.x; s2 < nsplit; s2 += 128) {
    sm_M[s2] = __ldcg(base + (size_t)s2 * (D + 2) + D); sm_L[s2] = __ldcg(base + (size_t)s2 * (D + 2) + D + 1);
  }
  __syncthreads();
  float MM = -INFINITY;
  for (int s2 = 0; s2 < nsplit; ++s2) MM = fmaxf(MM, sm_M[s2]);
  float LL = 0.f;
  for (int s2 = 0; s2 < nsplit; ++s2) {
    const float ms = sm_M[s2];
    if (ms != -INFINITY) LL += sm_L[s2] * expf(ms - MM);
  }
  for (int c = threadIdx.x; c < D; c += 128) {
    float acc = 0.f;
    for (int s0 = 0; s0 < nsplit; s0 += 16) {
      float pv[16];
#pragma unroll
      for (int i = 0; i < 16; ++i) pv[i] = (s0 + i < nsplit) ? __ldcg(base + (size_t)(s0 + i) * (D + 2) + c) : 0.f;
#pragma unroll
      for (int i = 0; i < 16; ++i) {
        if (s0 + i >= nsplit) break;
        const float ms = sm_M[s0 + i];
        if (ms != -INFINITY) acc += pv[i] * expf(ms - MM);
      }
    }
    out[(size_t)h * D + c] = acc / LL;
  }
}
void launch_attn_decode_fused(const float* qkv, const float* cos_t, const float* sin_t, float* kcache, float* vcache,
                              float* ws, float* out, int* counters, int pos, int nq, int nkv, int d, int max_seq,
                              int nsplit, cudaStream_t st) {
  ++g_launches;
  if (nsplit > kMaxSplit) nsplit = kMaxSplit;       // engine uses 16
  dim3 grid(nq, nsplit);
  if (d == 128) launch_pdl(attn_decode_fused_kernel<128>, grid, dim3(128), 0, st, qkv, cos_t, sin_t, kcache, vcache, ws, out, counters, pos, nq, nkv, max_seq, nsplit);
  else launch_pdl(attn_decode_fused_kernel<64>, grid, dim3(128), 0, st, qkv, cos_t, sin_t, kcache, vcache, ws, out, counters, pos, nq, nkv, max_seq, nsplit);
}

// ---------------------------------------------------------------------------------------------------------------
// K7: x[h] += Σ_j (ascending j) g_j · (Wd_{e_j}[h,:]·act_j) + σ(sgate)·(Wsd[h,:]·sact)      (A9 down + A10)
// One CTA = 4 output rows; the (k + shared) dot products of a row are cut into pieces of ≤ 2048 elements dealt to
// the 8 warps, partial sums meet in shared memory and are combined in a FIXED order (deterministic, no atomics).
// Routed experts are read from their slots behind the chunk-ready flags of exactly the rows this CTA reads.
constexpr int DC_ROWS = 4, DC_PIECE = 2048, DC_MAX_ITEMS = 192;
template <typename WT>
__global__ void __launch_bounds__(256, 4) ffn_down_combine_kernel(const float* __restrict__ act, int act_stride,
                                                               const FfnProblem* __restrict__ probs,
                                                               const int32_t* __restrict__ row_of,
                                                               const float* __restrict__ gates, int k,
                                                               const FfnProblem* __restrict__ shared,
                                                               const float* __restrict__ sact,
                                                               const float* __restrict__ sgate_logit,
                                                               const float* __restrict__ shared_y, int H,
                                                               float* __restrict__ x, size_t chunk_bytes, int* err) {
  __shared__ const void* it_w[DC_MAX_ITEMS];     // weight matrix base of the item
  __shared__ const float* it_x[DC_MAX_ITEMS];    // activation vector of the item
  __shared__ int it_ld[DC_MAX_ITEMS], it_off[DC_MAX_ITEMS], it_len[DC_MAX_ITEMS], it_j[DC_MAX_ITEMS];
  __shared__ float part[DC_ROWS][DC_MAX_ITEMS];
  __shared__ int s_ni, s_ok;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int r0 = blockIdx.x * DC_ROWS;
  pdl_enter();
  // prologue in parallel: thread j loads problem j (j == k: the shared expert) and waits for the chunk flags of the
  // down rows this CTA reads; thread 0 then cuts the dot products into items
  __shared__ FfnProblem s_pb[kMaxK + 1];
  __shared__ const float* s_xv[kMaxK + 1];
  __shared__ int s_okj[kMaxK + 1];
  const int nj = k + (shared ? 1 : 0);
  if (threadIdx.x < nj) {
    const int j = threadIdx.x;
    const int row = (j < k) ? row_of[j] : 0;
    const FfnProblem pb = (j < k) ? probs[row] : *shared;
    int ok = 1;
    if (j < k && pb.flags) {      // bytes of rows [r0, r0 + DC_ROWS) of the down matrix inside the slot image
      const size_t row_b = (size_t)pb.inter * sizeof(WT), off = 2 * (size_t)pb.inter * H * sizeof(WT);
      const int c0 = (int)((off + (size_t)r0 * row_b) / chunk_bytes);
      const int c1 = (int)((off + (size_t)min(H, r0 + DC_ROWS) * row_b - 1) / chunk_bytes);
      ok = wait_chunks(pb.flags, c0, c1, pb.gen, err);
    }
    s_pb[j] = pb; s_xv[j] = (j < k) ? act + (size_t)row * act_stride : sact; s_okj[j] = ok;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    int ni = 0, ok = 1;
    for (int j = 0; j < nj; ++j) {
      ok = ok && s_okj[j];
      const int inter = s_pb[j].inter;
      for (int o = 0; o < inter && ni < DC_MAX_ITEMS; o += DC_PIECE) {
        it_w[ni] = s_pb[j].wd; it_x[ni] = s_xv[j]; it_ld[ni] = inter; it_off[ni] = o; it_len[ni] = min(DC_PIECE, inter - o);
        it_j[ni] = (j < k) ? j : k; ++ni;
      }
    }
    s_ni = ni; s_ok = ok;
  }
  __syncthreads();
  if (!s_ok) return;
  const int ni = s_ni;
  for (int w = warp; w < DC_ROWS * ni; w += 8) {
    const int rr = w / ni, it = w % ni, r = r0 + rr;
    if (r >= H) continue;
    // pieces are <= DC_PIECE = 2048 elements: bf16 rows always take the all-loads-in-flight form
    const WT* wr = (const WT*)it_w[it] + (size_t)r * it_ld[it] + it_off[it];
    const int len = it_len[it];
    const float v = len <= 8 * 32 * WVec<WT>::N ? row_dot_short<WT, 8>(wr, it_x[it] + it_off[it], len, lane)
                                                 : row_dot<WT>(wr, it_x[it] + it_off[it], len, lane);
    if (lane == 0) part[rr][it] = v;
  }
  pdl_done();
  __syncthreads();
  if (threadIdx.x < DC_ROWS && r0 + threadIdx.x < H) {
    const int rr = threadIdx.x;
    float y = 0.f;
    int it = 0;
    for (int j = 0; j < k; ++j) {
      float d = 0.f;
      for (; it < ni && it_j[it] == j; ++it) d += part[rr][it];
      y = fmaf(gates[j], d, y);
    }
    if (shared || shared_y) {     // shared expert: down rows computed here, or precomputed (shared_y) under the copies
      float d = 0.f;
      if (shared) { for (; it < ni; ++it) d += part[rr][it]; }
      else d = shared_y[r0 + rr];
      const float sg = sgate_logit ? 1.f / (1.f + expf(-sgate_logit[0])) : 1.f;
      y += sg * d;
    }
    x[r0 + rr] += y;
  }
}
void launch_ffn_down_combine(const float* act, int act_stride, const FfnProblem* probs, const int32_t* row_of,
                             const float* gates, int k, const FfnProblem* shared, const float* sact,
                             const float* sgate_logit, const float* shared_y, int H, float* x, int wdtype,
                             size_t chunk_bytes, int* err, cudaStream_t st) {
  ++g_launches;
  const int blocks = (H + DC_ROWS - 1) / DC_ROWS;
  if (wdtype == 0) launch_pdl(ffn_down_combine_kernel<float>, dim3(blocks), dim3(256), 0, st, act, act_stride, probs, row_of, gates, k, shared, sact, sgate_logit, shared_y, H, x, chunk_bytes, err);
  else launch_pdl(ffn_down_combine_kernel<__nv_bfloat16>, dim3(blocks), dim3(256), 0, st, act, act_stride, probs, row_of, gates, k, shared, sact, sgate_logit, shared_y, H, x, chunk_bytes, err);
}

// Load every kernel of this file NOW.  CUDA loads kernels lazily, on their first launch, and that load waits for every
// running kernel to finish: a first launch behind a kernel that spins on a flag (an expert kernel waiting for its bytes,
// the fetch worker waiting for a gate) would dead-lock until the spinner times out (profiles/r02_spin_probe.md).
void preload_decode() {
  preload_fn((const void*)norm_multi_gemv_kernel<float>);
  preload_fn((const void*)norm_multi_gemv_kernel<__nv_bfloat16>);
  preload_fn((const void*)attn_decode_fused_kernel<128>);
  preload_fn((const void*)attn_decode_fused_kernel<64>);
  preload_fn((const void*)ffn_down_combine_kernel<float>);
  preload_fn((const void*)ffn_down_combine_kernel<__nv_bfloat16>);
}

}  // namespace pmk
