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
                                                              size_t chunk_bytes, int* err, int static_table) {
  pdl_trigger();
  const int p = blockIdx.x / tiles, tile = blockIdx.x % tiles;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int r0 = tile * 8;
  (void)static_table;   // early L2 prefetch of resident rows before the wait was measured slower (2.90 vs 2.81 ms/token)
  pdl_wait();
  const FfnProblem pb = probs[p];
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
  if (lane == 0) act[(size_t)p * act_stride + r] = silu(g) * v;
}

// down GEMV: y[p, h] = Wd[h,:].act[p,:]
template <typename WT>
__global__ void __launch_bounds__(256) ffn_down_gemv_kernel(const float* __restrict__ act, int act_stride,
                                                            const FfnProblem* __restrict__ probs,
                                                            const int32_t* __restrict__ n_probs_dev, int tiles,
                                                            int H, float* __restrict__ y, size_t chunk_bytes,
                                                            int* err, int static_table) {
  pdl_trigger();
  const int p = blockIdx.x / tiles, tile = blockIdx.x % tiles;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int r0 = tile * 8;
  (void)static_table;
  pdl_wait();
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
                            int act_stride, int wdtype, size_t chunk_bytes, int* err, cudaStream_t st, int static_table) {
  ++g_launches;
  const int tiles = (max_inter + 7) / 8;
  const int32_t* nd = nullptr;
  WDISPATCH(launch_pdl(ffn_gateup_gemv_kernel<float>, dim3(n_probs * tiles), dim3(256), 0, st, u, probs, nd, tiles, H, act, act_stride, chunk_bytes, err, static_table),
            launch_pdl(ffn_gateup_gemv_kernel<__nv_bfloat16>, dim3(n_probs * tiles), dim3(256), 0, st, u, probs, nd, tiles, H, act, act_stride, chunk_bytes, err, static_table));
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

}  // namespace pmk

// ---------------------------------------------------------------------------------------------------------
// A9 decode gate/up GEMV, TMA-fed (bf16 weights, H <= 2048).  The register-fed kernel above tops out at ≈ 3.7 TB/s:
// its bytes in flight are bounded by registers × resident warps.  Here each persistent CTA (one per SM) streams
// blocks of 8 gate rows + the matching 8 up rows (2 × 8·H·2 bytes, both contiguous in the slot image) into a
// two-stage shared-memory ring with cp.async.bulk + mbarrier (64-128 KB in flight per SM), and its 8 warps reduce
// one row pair each from shared memory.  Items are dealt problem-major, so the experts first in launch order
// (cached → being prefetched → missing) are served first; the issuing thread waits for the chunk flags of
// exactly the bytes of the block it is about to fetch (Alg. 1 l.10).
// MEASURED (B200, promoe_kernel_time, back-to-back launches): c2 shape 14.4 µs vs 12.3 µs register-fed; c3 shape
// 19.4 vs 19.6 µs — no gain, so the step uses the register-fed kernel and this one stays reachable only through
// promoe_op_expert_ffn(path 4) (parity-tested) as the starting point for the next round's tuning.
namespace pmk {

constexpr int GT_ROWS = 8;
__device__ __forceinline__ uint32_t s_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void gt_mbar_init(uint64_t* b, uint32_t c) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(s_u32(b)), "r"(c));
}
__device__ __forceinline__ void gt_expect_tx(uint64_t* b, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(s_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void gt_wait(uint64_t* b, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(s_u32(b)), "r"(parity) : "memory");
  } while (!ok);
}
__device__ __forceinline__ void gt_bulk_load(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(s_u32(dst)), "l"(src), "r"(bytes), "r"(s_u32(bar)) : "memory");
}

__global__ void __launch_bounds__(256, 1) ffn_gateup_gemv_tma_kernel(const float* __restrict__ u,
                                                                     const FfnProblem* __restrict__ probs, int n_probs,
                                                                     int inter, int H, float* __restrict__ act,
                                                                     int act_stride, size_t chunk_bytes, int* err) {
  extern __shared__ __align__(128) uint8_t gt_smem[];
  const uint32_t blk_bytes = (uint32_t)GT_ROWS * H * 2;          // one block of 8 rows
  uint8_t* stage0 = gt_smem;                                      // [2 stages][gate block | up block]
  float* xs = (float*)(gt_smem + 4 * (size_t)blk_bytes);          // [H]
  uint64_t* full = (uint64_t*)(xs + H);                           // [2]
  __shared__ int s_fail;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nb = inter / GT_ROWS, total = n_probs * nb;
  if (threadIdx.x == 0) { gt_mbar_init(full, 1); gt_mbar_init(full + 1, 1); s_fail = 0; asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
  for (int i = threadIdx.x; i < H; i += 256) xs[i] = u[i];
  __syncthreads();
  // thread 0: fetch item `it` into stage s (after the flags of its bytes show the slot's generation)
  auto issue = [&](int it, int s) {
    const int p = it / nb, b = it % nb;
    const FfnProblem pb = probs[p];
    const size_t row_b = (size_t)H * 2, g_off = (size_t)b * GT_ROWS * row_b, u_off = (size_t)inter * row_b + g_off;
    if (pb.flags) {
      bool ok = wait_chunks(pb.flags, (int)(g_off / chunk_bytes), (int)((g_off + blk_bytes - 1) / chunk_bytes), pb.gen, err);
      ok = ok && wait_chunks(pb.flags, (int)(u_off / chunk_bytes), (int)((u_off + blk_bytes - 1) / chunk_bytes), pb.gen, err);
      if (!ok) s_fail = 1;
    }
    uint8_t* dst = stage0 + (size_t)s * 2 * blk_bytes;
    gt_expect_tx(full + s, 2 * blk_bytes);
    gt_bulk_load(dst, (const uint8_t*)pb.wg + g_off, blk_bytes, full + s);
    gt_bulk_load(dst + blk_bytes, (const uint8_t*)pb.wu + g_off, blk_bytes, full + s);
  };
  const int first = blockIdx.x, step = gridDim.x;
  if (threadIdx.x == 0) {
    if (first < total) issue(first, 0);
    if (first + step < total) issue(first + step, 1);
  }
  int n = 0;
  for (int it = first; it < total; it += step, ++n) {
    const int s = n & 1;
    gt_wait(full + s, (n >> 1) & 1);
    const uint8_t* blk = stage0 + (size_t)s * 2 * blk_bytes;
    const __nv_bfloat16* gr = (const __nv_bfloat16*)blk + (size_t)warp * H;
    const __nv_bfloat16* ur = (const __nv_bfloat16*)(blk + blk_bytes) + (size_t)warp * H;
    float ag0 = 0.f, ag1 = 0.f, au0 = 0.f, au1 = 0.f;      // two independent chains per row (fixed order)
    auto body = [&](int kk, float& ag, float& au) {
      const uint4 wg4 = *reinterpret_cast<const uint4*>(gr + kk);
      const uint4 wu4 = *reinterpret_cast<const uint4*>(ur + kk);
      const float4 x0 = *reinterpret_cast<const float4*>(xs + kk), x1 = *reinterpret_cast<const float4*>(xs + kk + 4);
      const uint32_t gw[4] = {wg4.x, wg4.y, wg4.z, wg4.w}, uw[4] = {wu4.x, wu4.y, wu4.z, wu4.w};
      const float xv[8] = {x0.x, x0.y, x0.z, x0.w, x1.x, x1.y, x1.z, x1.w};
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        ag = fmaf(__uint_as_float(gw[j] << 16), xv[2 * j], ag);
        ag = fmaf(__uint_as_float(gw[j] & 0xffff0000u), xv[2 * j + 1], ag);
        au = fmaf(__uint_as_float(uw[j] << 16), xv[2 * j], au);
        au = fmaf(__uint_as_float(uw[j] & 0xffff0000u), xv[2 * j + 1], au);
      }
    };
    for (int kk = lane * 8; kk < H; kk += 512) {
      body(kk, ag0, au0);
      if (kk + 256 < H) body(kk + 256, ag1, au1);
    }
    const float g = warp_sum(ag0 + ag1), v = warp_sum(au0 + au1);
    const int p = it / nb, b = it % nb;
    if (lane == 0 && !s_fail) act[(size_t)p * act_stride + b * GT_ROWS + warp] = silu(g) * v;
    __syncthreads();                               // every warp is done with stage s
    if (threadIdx.x == 0 && it + 2 * step < total) issue(it + 2 * step, s);
  }
}

bool launch_ffn_gateup_gemv_tma(const float* u, const FfnProblem* probs, int n_probs, int inter, int H, float* act,
                                int act_stride, size_t chunk_bytes, int* err, cudaStream_t st) {
  if (H > 2048 || H % 256 || inter % GT_ROWS) return false;      // stage = 2 × 8·H·2 bytes, two stages ≤ 128 KB
  ++g_launches;
  const size_t smem = 4 * (size_t)GT_ROWS * H * 2 + (size_t)H * 4 + 64;
  static bool attr = false;
  if (!attr) { cudaFuncSetAttribute(ffn_gateup_gemv_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024); attr = true; }
  const int total = n_probs * (inter / GT_ROWS);
  const int grid = total < 148 ? total : 148;
  ffn_gateup_gemv_tma_kernel<<<grid, 256, smem, st>>>(u, probs, n_probs, inter, H, act, act_stride, chunk_bytes, err);
  return true;
}

}  // namespace pmk
