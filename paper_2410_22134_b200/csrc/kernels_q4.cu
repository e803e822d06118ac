// kernels_q4.cu — A9 with INT4 group-quantised routed experts (§7.6: the expert
// parameters that cross PCIe and sit in the cache are 4-bit, the computation is unchanged).
//
// Format (G18; restated here, shared with nobody): per matrix W [N, K], K % 128 == 0, row-major:
//   codes  N·K/2 bytes — element (n, k) in byte (n·K + k)/2, even k in the low nibble;
//   scales N·K/128 bf16 — group k/128 of row n;          W[n, k] = (code − 8) · scale.
// Expert image = [gate codes | up codes | down codes | gate scales | up scales | down scales] (gate/up [I, H], down [H, I]):
// 0.515625 bytes per weight instead of 2, so a slot fill moves 3.88× fewer bytes over the link — the H2D term of the step
// roofline shrinks by that factor and the HBM / latency terms start to matter.
//
// Decode: HBM-streaming GEMVs that dequantise in registers (one 4-byte load = 8 weights per lane and block of 256; the
// scale multiplies the block's partial sum once).  Each CTA gates on the chunk-ready flags of exactly the code AND scale bytes it
// reads.  Prefill: the needed experts are dequantised (exactly) into an fp32 staging image and the fp32 SIMT grouped GEMM runs
// on that; see dequant_q4_kernel for why not bf16 + tcgen05.
#include <algorithm>

#include "kernels.h"

namespace pmk {

constexpr int kQ4Group = 128;

// Σ_k W[k]·x[k] over quantised rows of K elements (K % 128 == 0); summation order depends on (K, lane) only.
// Block b of 256 elements: lane handles the 8 elements [256·b + 8·lane, +8) — ONE 4-byte code load (a warp reads 128
// contiguous bytes) and two float4 loads of x whose addresses are 32 bytes apart across lanes, i.e. the same L1 pattern as
// the bf16 GEMVs.  (A first version gave each lane 32 consecutive elements per 16-byte load: the x loads of a warp then hit
// 32 different 128-byte lines per instruction and the kernel ran at 0.49 TB/s, L1-wavefront bound.)  16 lanes share a scale.
__device__ __forceinline__ float q4_dot8(uint32_t w, const float* __restrict__ x) {
  const float4 x0 = __ldg(reinterpret_cast<const float4*>(x));
  const float4 x1 = __ldg(reinterpret_cast<const float4*>(x + 4));
  const float xv[8] = {x0.x, x0.y, x0.z, x0.w, x1.x, x1.y, x1.z, x1.w};
  float acc = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    // nibble → float without an integer conversion: 2^23 + code as a bit pattern, minus (2^23 + 8)
    const float v = __uint_as_float(0x4B000000u | ((w >> (4 * i)) & 15u)) - 8388616.0f;
    acc = fmaf(v, xv[i], acc);
  }
  return acc;
}
// NR rows (1: a down row, 2: the gate and the up row of one output) against the same x; U blocks in flight per row.
template <int NR, int U>
__device__ __forceinline__ void rows_dot_q4(const uint8_t* const (&codes)[NR], const __nv_bfloat16* const (&scales)[NR],
                                            const float* __restrict__ x, int K, int lane, float (&out)[NR]) {
  float tot[NR];
#pragma unroll
  for (int r = 0; r < NR; ++r) tot[r] = 0.f;
  for (int k0 = 0; k0 < K; k0 += U * 256) {
    uint32_t c[NR][U]; float s[NR][U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int k = k0 + u * 256 + lane * 8;
      if (k < K) {
#pragma unroll
        for (int r = 0; r < NR; ++r) {
          c[r][u] = __ldcs(reinterpret_cast<const unsigned int*>(codes[r] + (k >> 1)));
          s[r][u] = __bfloat162float(scales[r][k / kQ4Group]);
        }
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int k = k0 + u * 256 + lane * 8;
      if (k < K) {
#pragma unroll
        for (int r = 0; r < NR; ++r) tot[r] = fmaf(s[r][u], q4_dot8(c[r][u], x + k), tot[r]);
      }
    }
  }
#pragma unroll
  for (int r = 0; r < NR; ++r) out[r] = warp_sum(tot[r]);
}
template <int U>
__device__ __forceinline__ float row_dot_q4(const uint8_t* codes, const __nv_bfloat16* scales, const float* __restrict__ x,
                                            int K, int lane) {
  const uint8_t* const c[1] = {codes};
  const __nv_bfloat16* const sc[1] = {scales};
  float o[1];
  rows_dot_q4<1, U>(c, sc, x, K, lane, o);
  return o[0];
}

struct Q4Image {       // byte offsets inside one expert image
  size_t nc, ns;       // code bytes / scale bytes per matrix
  __device__ Q4Image(int H, int inter) : nc((size_t)H * inter / 2), ns((size_t)H * inter / kQ4Group * 2) {}
};
__device__ __forceinline__ int q4_wait(const unsigned* flags, size_t b0, size_t b1, size_t chunk_bytes, unsigned gen, int* err) {
  return wait_chunks(flags, (int)(b0 / chunk_bytes), (int)((b1 - 1) / chunk_bytes), gen, err);
}

// gate/up GEMV: act[p, i] = silu(Wg[i,:]·u) · (Wu[i,:]·u); grid = n_probs · ceil(inter/8), one warp per row
__global__ void __launch_bounds__(256, 5) ffn_gateup_gemv_q4_kernel(const float* __restrict__ u, const FfnProblem* __restrict__ probs,
                                                                 int tiles, int H, float* __restrict__ act, int act_stride,
                                                                 size_t chunk_bytes, int* err, const uint32_t* gate_seq,
                                                                 uint32_t gate_want) {
  const int p = blockIdx.x / tiles, tile = blockIdx.x % tiles;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int r0 = tile * 8;
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
  if (r0 >= pb.inter) return;
  const int r1 = min(pb.inter, r0 + 8);
  const Q4Image im(H, pb.inter);
  const size_t crow = (size_t)H / 2, srow = (size_t)H / kQ4Group * 2;
  __shared__ int ok;
  if (threadIdx.x == 0) {
    ok = 1;
    if (pb.flags) {
      ok = q4_wait(pb.flags, r0 * crow, r1 * crow, chunk_bytes, pb.gen, err)
        && q4_wait(pb.flags, im.nc + r0 * crow, im.nc + r1 * crow, chunk_bytes, pb.gen, err)
        && q4_wait(pb.flags, 3 * im.nc + r0 * srow, 3 * im.nc + r1 * srow, chunk_bytes, pb.gen, err)
        && q4_wait(pb.flags, 3 * im.nc + im.ns + r0 * srow, 3 * im.nc + im.ns + r1 * srow, chunk_bytes, pb.gen, err);
    }
  }
  __syncthreads();
  if (!ok) return;
  const int r = r0 + warp;
  if (r >= pb.inter) return;
  const uint8_t* img = (const uint8_t*)pb.wg;
  const uint8_t* const cr[2] = {img + r * crow, img + im.nc + r * crow};
  const __nv_bfloat16* const sr[2] = {(const __nv_bfloat16*)(img + 3 * im.nc + r * srow), (const __nv_bfloat16*)(img + 3 * im.nc + im.ns + r * srow)};
  float gv[2];
  rows_dot_q4<2, 4>(cr, sr, u, H, lane, gv);        // gate and up row: 8 loads in flight per lane
  pdl_done();
  if (lane == 0) act[(size_t)p * act_stride + r] = silu(gv[0]) * gv[1];
}

// down GEMV: y[p, h] = Wd[h,:]·act[p,:]
__global__ void __launch_bounds__(256) ffn_down_gemv_q4_kernel(const float* __restrict__ act, int act_stride,
                                                               const FfnProblem* __restrict__ probs, int tiles, int H,
                                                               float* __restrict__ y, size_t chunk_bytes, int* err) {
  const int p = blockIdx.x / tiles, tile = blockIdx.x % tiles;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int r0 = tile * 8;
  pdl_enter();
  const FfnProblem pb = probs[p];
  if (r0 >= H) return;
  const int r1 = min(H, r0 + 8);
  const Q4Image im(H, pb.inter);
  const size_t crow = (size_t)pb.inter / 2, srow = (size_t)pb.inter / kQ4Group * 2;
  __shared__ int ok;
  if (threadIdx.x == 0) {
    ok = 1;
    if (pb.flags)
      ok = q4_wait(pb.flags, 2 * im.nc + r0 * crow, 2 * im.nc + r1 * crow, chunk_bytes, pb.gen, err)
        && q4_wait(pb.flags, 3 * im.nc + 2 * im.ns + r0 * srow, 3 * im.nc + 2 * im.ns + r1 * srow, chunk_bytes, pb.gen, err);
  }
  __syncthreads();
  if (!ok) return;
  const int r = r0 + warp;
  if (r >= H) return;
  const uint8_t* img = (const uint8_t*)pb.wg;
  const float v = row_dot_q4<8>(img + 2 * im.nc + r * crow, (const __nv_bfloat16*)(img + 3 * im.nc + 2 * im.ns + r * srow),
                                act + (size_t)p * act_stride, pb.inter, lane);
  pdl_done();
  if (lane == 0) y[(size_t)p * H + r] = v;
}

// K7 for INT4 experts: x[h] += Σ_j (ascending j) g_j · (Wd_{e_j}[h,:]·act_j) + σ(sgate)·shared_y[h]   (A9 down + A10)
// One CTA = 4 output rows × k experts; warp w takes (row, expert) pairs; fixed-order combine, no atomics.
__global__ void __launch_bounds__(256) ffn_down_combine_q4_kernel(const float* __restrict__ act, int act_stride,
                                                                  const FfnProblem* __restrict__ probs,
                                                                  const int32_t* __restrict__ row_of,
                                                                  const float* __restrict__ gates, int k,
                                                                  const float* __restrict__ sgate_logit,
                                                                  const float* __restrict__ shared_y, int H,
                                                                  float* __restrict__ x, size_t chunk_bytes, int* err) {
  constexpr int ROWS = 4;
  __shared__ FfnProblem s_pb[kMaxK];
  __shared__ const float* s_xv[kMaxK];
  __shared__ int s_okj[kMaxK];
  __shared__ float part[ROWS][kMaxK];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int r0 = blockIdx.x * ROWS, r1 = min(H, r0 + ROWS);
  pdl_enter();
  if (threadIdx.x < k) {
    const int j = threadIdx.x, row = row_of[j];
    const FfnProblem pb = probs[row];
    int ok = 1;
    if (pb.flags) {
      const Q4Image im(H, pb.inter);
      const size_t crow = (size_t)pb.inter / 2, srow = (size_t)pb.inter / kQ4Group * 2;
      ok = q4_wait(pb.flags, 2 * im.nc + r0 * crow, 2 * im.nc + r1 * crow, chunk_bytes, pb.gen, err)
        && q4_wait(pb.flags, 3 * im.nc + 2 * im.ns + r0 * srow, 3 * im.nc + 2 * im.ns + r1 * srow, chunk_bytes, pb.gen, err);
    }
    s_pb[j] = pb; s_xv[j] = act + (size_t)row * act_stride; s_okj[j] = ok;
  }
  __syncthreads();
  for (int j = 0; j < k; ++j) if (!s_okj[j]) return;
  for (int w = warp; w < ROWS * k; w += 8) {
    const int rr = w / k, j = w % k, r = r0 + rr;
    if (r >= H) continue;
    const FfnProblem& pb = s_pb[j];
    const Q4Image im(H, pb.inter);
    const size_t crow = (size_t)pb.inter / 2, srow = (size_t)pb.inter / kQ4Group * 2;
    const uint8_t* img = (const uint8_t*)pb.wg;
    const float v = row_dot_q4<8>(img + 2 * im.nc + r * crow, (const __nv_bfloat16*)(img + 3 * im.nc + 2 * im.ns + r * srow),
                                  s_xv[j], pb.inter, lane);
    if (lane == 0) part[rr][j] = v;
  }
  pdl_done();
  __syncthreads();
  if (threadIdx.x < ROWS && r0 + threadIdx.x < H) {
    const int rr = threadIdx.x;
    float y = 0.f;
    for (int j = 0; j < k; ++j) y = fmaf(gates[j], part[rr][j], y);
    if (shared_y) {
      const float sg = sgate_logit ? 1.f / (1.f + expf(-sgate_logit[0])) : 1.f;
      y += sg * shared_y[r0 + rr];
    }
    x[r0 + rr] += y;
  }
}

// Prefill: dequantise the INT4 images of problems [p0, p0 + np) into fp32 staging images [gate | up | down] and write the
// matching problem records (same row ranges, pointers into the staging region, no flags).  fp32 because (code − 8)·scale has
// up to 11 significant bits: a bf16 staging image would round it (2^-9 relative) and break the 1e-3 routing-margin rule of
// the parity contract; the fp32 SIMT grouped GEMM then runs on the staged images.  grid (blocks, np).
__global__ void __launch_bounds__(256) dequant_q4_kernel(const FfnProblem* __restrict__ probs, int p0, int H,
                                                         float* __restrict__ stage, size_t stage_stride_elems,
                                                         FfnProblem* __restrict__ out_probs) {
  const int pi = p0 + blockIdx.y;
  const FfnProblem pb = probs[pi];
  const int inter = pb.inter;
  const size_t hi = (size_t)H * inter;
  const Q4Image im(H, inter);
  const uint8_t* img = (const uint8_t*)pb.wg;
  float* dst = stage + (size_t)pi * stage_stride_elems;
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    FfnProblem o = pb;
    o.wg = dst; o.wu = dst + hi; o.wd = dst + 2 * hi; o.flags = nullptr; o.gen = 0;
    out_probs[pi] = o;
  }
  // 3·hi elements, 32 per 16-byte load; matrices 0/1 have K = H, matrix 2 has K = inter
  const size_t n32 = 3 * hi / 32;
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < n32; t += (size_t)gridDim.x * blockDim.x) {
    const size_t e0 = t * 32;
    const int mat = (int)(e0 / hi);
    const size_t within = e0 - (size_t)mat * hi;
    const int K = mat < 2 ? H : inter;
    const size_t row = within / K, col = within % K;
    const uint4 c = *reinterpret_cast<const uint4*>(img + e0 / 2);
    const float s = __bfloat162float(*reinterpret_cast<const __nv_bfloat16*>(img + 3 * im.nc + (size_t)mat * im.ns + (row * (K / kQ4Group) + col / kQ4Group) * 2));
    const uint32_t w[4] = {c.x, c.y, c.z, c.w};
    float4* d4 = reinterpret_cast<float4*>(dst + e0);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      float o[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) o[i] = ((float)((w[q] >> (4 * i)) & 15u) - 8.0f) * s;     // exact in fp32
      d4[2 * q] = make_float4(o[0], o[1], o[2], o[3]);
      d4[2 * q + 1] = make_float4(o[4], o[5], o[6], o[7]);
    }
  }
}

// Prefill on the tensor cores: the same dequantisation into a bf16 hi/lo PAIR of staging images — (code − 8)·scale has up to
// 11 significant bits, hi = bf16(w) keeps 8 and lo = w − hi (≤ 4 bits) is exact — so the tcgen05 GEMM runs one pass over
// each image with the same activation operand and accumulates (W_hi + W_lo)·x in fp32: exact weights, twice the MMAs.
__global__ void __launch_bounds__(256) dequant_q4_bf16_kernel(const FfnProblem* __restrict__ probs, int p0, int H,
                                                              __nv_bfloat16* __restrict__ stage, size_t lo_off,
                                                              size_t stage_stride_elems, FfnProblem* __restrict__ out_probs) {
  const int pi = p0 + blockIdx.y;
  const FfnProblem pb = probs[pi];
  const int inter = pb.inter;
  const size_t hi = (size_t)H * inter;
  const Q4Image im(H, inter);
  const uint8_t* img = (const uint8_t*)pb.wg;
  __nv_bfloat16* dst = stage + (size_t)pi * stage_stride_elems;
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    FfnProblem o = pb;
    o.wg = dst; o.wu = dst + hi; o.wd = dst + 2 * hi; o.flags = nullptr; o.gen = 0;
    out_probs[pi] = o;
  }
  const size_t n8 = 3 * hi / 8;        // 8 codes per 4-byte load: consecutive threads read consecutive words
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < n8; t += (size_t)gridDim.x * blockDim.x) {
    const size_t e0 = t * 8;
    const int mat = (int)(e0 / hi);
    const size_t within = e0 - (size_t)mat * hi;
    const int K = mat < 2 ? H : inter;
    const size_t row = within / K, col = within % K;
    const uint32_t w = *reinterpret_cast<const uint32_t*>(img + e0 / 2);
    const float s = __bfloat162float(*reinterpret_cast<const __nv_bfloat16*>(img + 3 * im.nc + (size_t)mat * im.ns + (row * (K / kQ4Group) + col / kQ4Group) * 2));
    __align__(16) __nv_bfloat16 oh[8], ol[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const float v = ((float)((w >> (4 * i)) & 15u) - 8.0f) * s;       // exact in fp32
      oh[i] = __float2bfloat16_rn(v);
      ol[i] = __float2bfloat16_rn(v - __bfloat162float(oh[i]));         // exact: at most 4 significant bits are left
    }
    *reinterpret_cast<uint4*>(dst + e0) = *reinterpret_cast<const uint4*>(oh);
    *reinterpret_cast<uint4*>(dst + lo_off + e0) = *reinterpret_cast<const uint4*>(ol);
  }
}
// gu [.., 2·I] fp32 = [gate | up] pre-activations of the rows of problems [p0, p0+np) → silu(g)·u as bf16 hi/lo planes
// [.., I] (the activation operand of the down GEMM).  grid (max_rows, np).
__global__ void __launch_bounds__(256) swiglu_split_kernel(const float* __restrict__ gu, const FfnProblem* __restrict__ probs,
                                                           int p0, int inter, __nv_bfloat16* __restrict__ o_hi, size_t o_lo_off) {
  const FfnProblem pb = probs[p0 + blockIdx.y];
  if ((int)blockIdx.x >= pb.nrows) return;
  const size_t r = (size_t)pb.row0 + blockIdx.x;
  const float* g = gu + r * 2 * inter;
  for (int i = threadIdx.x; i < inter; i += blockDim.x) {
    const float v = silu(g[i]) * g[inter + i];
    const __nv_bfloat16 hi = __float2bfloat16_rn(v);
    o_hi[r * inter + i] = hi;
    o_hi[r * inter + i + o_lo_off] = __float2bfloat16_rn(v - __bfloat162float(hi));
  }
}

void launch_ffn_gateup_gemv_q4(const float* u, const FfnProblem* probs, int n_probs, int max_inter, int H, float* act,
                               int act_stride, size_t chunk_bytes, int* err, cudaStream_t st, const uint32_t* gate_seq,
                               uint32_t gate_want) {
  ++g_launches;
  const int tiles = (max_inter + 7) / 8;
  launch_pdl(ffn_gateup_gemv_q4_kernel, dim3(n_probs * tiles), dim3(256), 0, st, u, probs, tiles, H, act, act_stride, chunk_bytes, err,
             gate_seq, gate_want);
}
void launch_ffn_down_gemv_q4(const float* act, int act_stride, const FfnProblem* probs, int n_probs, int H, float* y,
                             size_t chunk_bytes, int* err, cudaStream_t st) {
  ++g_launches;
  const int tiles = (H + 7) / 8;
  launch_pdl(ffn_down_gemv_q4_kernel, dim3(n_probs * tiles), dim3(256), 0, st, act, act_stride, probs, tiles, H, y, chunk_bytes, err);
}
void launch_ffn_down_combine_q4(const float* act, int act_stride, const FfnProblem* probs, const int32_t* row_of,
                                const float* gates, int k, const float* sgate_logit, const float* shared_y, int H, float* x,
                                size_t chunk_bytes, int* err, cudaStream_t st) {
  ++g_launches;
  launch_pdl(ffn_down_combine_q4_kernel, dim3((H + 3) / 4), dim3(256), 0, st, act, act_stride, probs, row_of, gates, k,
             sgate_logit, shared_y, H, x, chunk_bytes, err);
}
void launch_dequant_q4(const FfnProblem* probs, int p0, int np, int H, int max_inter, float* stage,
                       size_t stage_stride_elems, FfnProblem* out_probs, cudaStream_t st) {
  ++g_launches;
  if (np <= 0) return;
  const size_t n32 = (size_t)3 * H * max_inter / 32;
  const int bx = (int)std::min<size_t>((n32 + 255) / 256, 1024);
  dequant_q4_kernel<<<dim3(bx, np), 256, 0, st>>>(probs, p0, H, stage, stage_stride_elems, out_probs);
}

void launch_dequant_q4_bf16(const FfnProblem* probs, int p0, int np, int H, int max_inter, __nv_bfloat16* stage, size_t lo_off,
                            size_t stage_stride_elems, FfnProblem* out_probs, cudaStream_t st) {
  ++g_launches;
  if (np <= 0) return;
  const size_t n8 = (size_t)3 * H * max_inter / 8;
  const int bx = (int)std::min<size_t>((n8 + 255) / 256, 2048);
  dequant_q4_bf16_kernel<<<dim3(bx, np), 256, 0, st>>>(probs, p0, H, stage, lo_off, stage_stride_elems, out_probs);
}
void launch_swiglu_split(const float* gu, const FfnProblem* probs, int p0, int np, int max_rows, int inter, __nv_bfloat16* o_hi,
                         size_t o_lo_off, cudaStream_t st) {
  ++g_launches;
  if (np <= 0 || max_rows <= 0) return;
  swiglu_split_kernel<<<dim3(max_rows, np), 256, 0, st>>>(gu, probs, p0, inter, o_hi, o_lo_off);
}

void preload_q4() {
  preload_fn((const void*)dequant_q4_bf16_kernel);
  preload_fn((const void*)swiglu_split_kernel);
  preload_fn((const void*)ffn_gateup_gemv_q4_kernel);
  preload_fn((const void*)ffn_down_gemv_q4_kernel);
  preload_fn((const void*)ffn_down_combine_q4_kernel);
  preload_fn((const void*)dequant_q4_kernel);
}

}  // namespace pmk
