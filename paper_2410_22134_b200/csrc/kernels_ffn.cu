// kernels_ffn.cu — A9: SwiGLU expert FFN.  Decode: HBM-streaming GEMV kernels over a problem list in launch
// order (ready experts first), each CTA gating on the chunk-ready flags of exactly the bytes it reads
// (Alg. 1 l.10 `ready_chunk`).  Prefill: grouped SIMT fp32 GEMMs (correctness path; tcgen05 path: gemm_tc.cu).
#include "kernels.h"

namespace pmk {

// chunk index range [c0, c1] covering bytes [b0, b1) of the slot image
__device__ __forceinline__ void chunk_range(size_t b0, size_t b1, size_t chunk_bytes, int* c0, int* c1) {
  *c0 = (int)(b0 / chunk_bytes);
  *c1 = (int)((b1 - 1) / chunk_bytes);
}

// ---------------------------------------------------------------------------------------------------------
// gate/up GEMV: grid.x = n_probs * tiles, tile = 8 rows (one per warp); problem-major so that the CTAs of the
// experts first in launch order are scheduled first.  act[p, i] = silu(Wg[i,:].u) * (Wu[i,:].u)
template <typename WT>
__global__ void __launch_bounds__(256) ffn_gateup_gemv_kernel(const float* __restrict__ u,
                                                              const FfnProblem* __restrict__ probs,
                                                              const int32_t* __restrict__ n_probs_dev, int tiles,
                                                              int H, float* __restrict__ act, int act_stride,
                                                              size_t chunk_bytes, int* err, int static_table,
                                                              const uint32_t* gate_seq, uint32_t gate_want) {
  const int p = blockIdx.x / tiles, tile = blockIdx.x % tiles;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int r0 = tile * 8;
  (void)static_table;   // early L2 prefetch of resident rows before the wait was measured slower (2.90 vs 2.81 ms/token)
  FfnProblem pb;
  if (gate_seq) {       // wait for the problem table only, not for the predictor half of the slot-table kernel
    __shared__ int gate_ok;
    if (threadIdx.x == 0) gate_ok = wait_gate_word(gate_seq, gate_want, err);
    __syncthreads();
    if (!gate_ok) return;
    pb = load_problem_cg(probs + p);
  } else {
    pdl_enter();
    pb = probs[p];
  }
  if (n_probs_dev && p >= *n_probs_dev) return;
  if (r0 >= pb.inter) return;
  const int r1 = min(pb.inter, r0 + 8);
  __shared__ int ok;
  if (threadIdx.x == 0) {
    ok = 1;
    if (pb.flags) {
      const size_t row_b = (size_t)H * sizeof(WT), up_off = (size_t)pb.inter * row_b;
      int c0, c1;
      chunk_range(r0 * row_b, r1 * row_b, chunk_bytes, &c0, &c1);
      ok = wait_chunks(pb.flags, c0, c1, pb.gen, err);
      chunk_range(up_off + r0 * row_b, up_off + r1 * row_b, chunk_bytes, &c0, &c1);
      ok = ok && wait_chunks(pb.flags, c0, c1, pb.gen, err);
    }
  }
  __syncthreads();
  if (!ok) return;
  const int r = r0 + warp;
  if (r >= pb.inter) return;
  // two passes (4 loads in flight per lane each): 48 registers keep 40 warps/SM resident, so the c2/c3 grid
  // (5632 / 8448 warps) is a single wave; a fused two-row variant (8 loads in flight per lane, 2 waves) measured slower: 16.1 vs 12.3 µs
#ifndef PROMOE_K6_UNR
#define PROMOE_K6_UNR 4
#endif
  const float g = row_dot<WT, PROMOE_K6_UNR>((const WT*)pb.wg + (size_t)r * H, u, H, lane);
  const float v = row_dot<WT, PROMOE_K6_UNR>((const WT*)pb.wu + (size_t)r * H, u, H, lane);
  pdl_done();
  if (lane == 0) act[(size_t)p * act_stride + r] = silu(g) * v;
}

// down GEMV: y[p, h] = Wd[h,:].act[p,:]
template <typename WT>
__global__ void __launch_bounds__(256) ffn_down_gemv_kernel(const float* __restrict__ act, int act_stride,
                                                            const FfnProblem* __restrict__ probs,
                                                            const int32_t* __restrict__ n_probs_dev, int tiles,
                                                            int H, float* __restrict__ y, size_t chunk_bytes,
                                                            int* err, int static_table) {
  const int p = blockIdx.x / tiles, tile = blockIdx.x % tiles;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int r0 = tile * 8;
  (void)static_table;
  pdl_enter();
  const FfnProblem pb = probs[p];
  if (n_probs_dev && p >= *n_probs_dev) return;
  if (r0 >= H) return;
  const int r1 = min(H, r0 + 8);
  __shared__ int ok;
  if (threadIdx.x == 0) {
    ok = 1;
    if (pb.flags) {
      const size_t row_b = (size_t)pb.inter * sizeof(WT), off = 2 * (size_t)pb.inter * H * sizeof(WT);
      int c0, c1;
      chunk_range(off + r0 * row_b, off + r1 * row_b, chunk_bytes, &c0, &c1);
      ok = wait_chunks(pb.flags, c0, c1, pb.gen, err);
    }
  }
  __syncthreads();
  if (!ok) return;
  const int r = r0 + warp;
  if (r >= H) return;
  const float v = row_dot<WT>((const WT*)pb.wd + (size_t)r * pb.inter, act + (size_t)p * act_stride, pb.inter, lane);
  pdl_done();
  if (lane == 0) y[(size_t)p * H + r] = v;
}

// ---------------------------------------------------------------------------------------------------------
// Prefill grouped SwiGLU FFN on CUDA cores (fp32 FMA over exactly-widened weights).  64x64x16 tiles.
// grid (ceil(N/64), ceil(max_rows/64), n_problems).
constexpr int FB = 64, FK = 16;
template <typename WT, bool SWIGLU>
__global__ void __launch_bounds__(256) ffn_gemm_simt_kernel(const float* __restrict__ a, int lda,
                                                            const int32_t* __restrict__ row_src, int src_div,
                                                            const FfnProblem* __restrict__ probs, int p0, int H,
                                                            float* __restrict__ out, int ldo, int rows_override) {
  FfnProblem pb = probs[p0 + blockIdx.z];
  if (rows_override > 0) pb.nrows = rows_override;
  const int m0 = blockIdx.y * FB;
  if (m0 >= pb.nrows) return;
  const int N = SWIGLU ? pb.inter : H;          // output features
  const int K = SWIGLU ? H : pb.inter;          // reduction length
  const int n0 = blockIdx.x * FB;
  if (n0 >= N) return;
  const WT* w1 = (const WT*)(SWIGLU ? pb.wg : pb.wd);
  const WT* w2 = (const WT*)pb.wu;
  __shared__ float as[FK][FB + 4];
  __shared__ float ws1[FK][FB + 4];
  __shared__ float ws2[SWIGLU ? FK : 1][FB + 4];
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  const int lr = threadIdx.x >> 2, lk = (threadIdx.x & 3) * 4;
  const int mrow = m0 + lr;
  const float* arow = nullptr;
  if (mrow < pb.nrows) {
    const int pr = pb.row0 + mrow;
    arow = a + (size_t)(row_src ? row_src[pr] / src_div : pr) * lda;
  }
  const int nrow = n0 + lr;
  float acc1[4][4] = {}, acc2[4][4] = {};
  for (int k0 = 0; k0 < K; k0 += FK) {
    float4 av = make_float4(0.f, 0.f, 0.f, 0.f);
    if (arow) av = *reinterpret_cast<const float4*>(arow + k0 + lk);
    as[lk][lr] = av.x; as[lk + 1][lr] = av.y; as[lk + 2][lr] = av.z; as[lk + 3][lr] = av.w;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      ws1[lk + q][lr] = (nrow < N) ? wload1(w1 + (size_t)nrow * K + k0 + lk + q) : 0.f;
      if (SWIGLU) ws2[lk + q][lr] = (nrow < N) ? wload1(w2 + (size_t)nrow * K + k0 + lk + q) : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < FK; ++kk) {
      float x[4], b1[4], b2[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) x[i] = as[kk][ty * 4 + i];
#pragma unroll
      for (int j = 0; j < 4; ++j) { b1[j] = ws1[kk][tx * 4 + j]; b2[j] = SWIGLU ? ws2[kk][tx * 4 + j] : 0.f; }
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          acc1[i][j] = fmaf(x[i], b1[j], acc1[i][j]);
          if (SWIGLU) acc2[i][j] = fmaf(x[i], b2[j], acc2[i][j]);
        }
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int mr = m0 + ty * 4 + i;
    if (mr >= pb.nrows) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int n = n0 + tx * 4 + j;
      if (n >= N) continue;
      out[(size_t)(pb.row0 + mr) * ldo + n] = SWIGLU ? silu(acc1[i][j]) * acc2[i][j] : acc1[i][j];
    }
  }
}

#define WDISPATCH(expr_f32, expr_bf16) do { if (wdtype == 0) { expr_f32; } else { expr_bf16; } } while (0)

void launch_ffn_gateup_gemv(const float* u, const FfnProblem* probs, int n_probs, int max_inter, int H, float* act,
                            int act_stride, int wdtype, size_t chunk_bytes, int* err, cudaStream_t st, int static_table,
                            const uint32_t* gate_seq, uint32_t gate_want) {
  ++g_launches;
  const int tiles = (max_inter + 7) / 8;
  const int32_t* nd = nullptr;
  WDISPATCH(launch_pdl(ffn_gateup_gemv_kernel<float>, dim3(n_probs * tiles), dim3(256), 0, st, u, probs, nd, tiles, H, act, act_stride, chunk_bytes, err, static_table, gate_seq, gate_want),
            launch_pdl(ffn_gateup_gemv_kernel<__nv_bfloat16>, dim3(n_probs * tiles), dim3(256), 0, st, u, probs, nd, tiles, H, act, act_stride, chunk_bytes, err, static_table, gate_seq, gate_want));
}
void launch_ffn_down_gemv(const float* act, int act_stride, const FfnProblem* probs, int n_probs, int max_inter,
                          int H, float* y, int wdtype, size_t chunk_bytes, int* err, cudaStream_t st, int static_table) {
  ++g_launches;
  (void)max_inter;
  const int tiles = (H + 7) / 8;
  const int32_t* nd = nullptr;
  WDISPATCH(launch_pdl(ffn_down_gemv_kernel<float>, dim3(n_probs * tiles), dim3(256), 0, st, act, act_stride, probs, nd, tiles, H, y, chunk_bytes, err, static_table),
            launch_pdl(ffn_down_gemv_kernel<__nv_bfloat16>, dim3(n_probs * tiles), dim3(256), 0, st, act, act_stride, probs, nd, tiles, H, y, chunk_bytes, err, static_table));
}
void launch_ffn_gateup_gemm_simt(const float* x, const int32_t* row_src, int src_div, const FfnProblem* probs,
                                 int p0, int np, int max_rows, int rows_override, int max_inter, int H, float* act,
                                 int act_stride, int wdtype, cudaStream_t st) {
  ++g_launches;
  dim3 grid((max_inter + FB - 1) / FB, (max_rows + FB - 1) / FB, np);
  WDISPATCH((ffn_gemm_simt_kernel<float, true><<<grid, 256, 0, st>>>(x, H, row_src, src_div, probs, p0, H, act,
                                                                     act_stride, rows_override)),
            (ffn_gemm_simt_kernel<__nv_bfloat16, true><<<grid, 256, 0, st>>>(x, H, row_src, src_div, probs, p0, H,
                                                                             act, act_stride, rows_override)));
}
void launch_ffn_down_gemm_simt(const float* act, int act_stride, const FfnProblem* probs, int p0, int np,
                               int max_rows, int rows_override, int max_inter, int H, float* y, int wdtype,
                               cudaStream_t st) {
  ++g_launches;
  (void)max_inter;
  dim3 grid((H + FB - 1) / FB, (max_rows + FB - 1) / FB, np);
  WDISPATCH((ffn_gemm_simt_kernel<float, false><<<grid, 256, 0, st>>>(act, act_stride, nullptr, 1, probs, p0, H, y,
                                                                      H, rows_override)),
            (ffn_gemm_simt_kernel<__nv_bfloat16, false><<<grid, 256, 0, st>>>(act, act_stride, nullptr, 1, probs, p0,
                                                                              H, y, H, rows_override)));
}

// Load every kernel of this file NOW.  CUDA loads kernels lazily, on their first launch, and that load waits for every
// running kernel to finish: a first launch behind a kernel that spins on a flag (an expert kernel waiting for its bytes,
// the fetch worker waiting for a gate) would dead-lock until the spinner times out (profiles/r02_spin_probe.md).
void preload_ffn() {
  preload_fn((const void*)ffn_gateup_gemv_kernel<float>);
  preload_fn((const void*)ffn_gateup_gemv_kernel<__nv_bfloat16>);
  preload_fn((const void*)ffn_down_gemv_kernel<float>);
  preload_fn((const void*)ffn_down_gemv_kernel<__nv_bfloat16>);
  preload_fn((const void*)(ffn_gemm_simt_kernel<float, true>));
  preload_fn((const void*)(ffn_gemm_simt_kernel<float, false>));
  preload_fn((const void*)(ffn_gemm_simt_kernel<__nv_bfloat16, true>));
  preload_fn((const void*)(ffn_gemm_simt_kernel<__nv_bfloat16, false>));
}

}  // namespace pmk

