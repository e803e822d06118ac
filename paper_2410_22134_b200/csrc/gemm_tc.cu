// gemm_tc.cu — A9 (prefill) grouped SwiGLU expert GEMM and the T > 1 linears on the 5th-generation tensor cores:
// tcgen05.mma with accumulators in TMEM, operands staged in shared memory by TMA (cp.async.bulk.tensor) through an
// mbarrier pipeline.  sm_100a only.
//
// Shape of the problem: Y[rows, N] = X[rows, K] · W[N, K]^T with bf16 weights, fp32 activations and
// 12-200 rows per expert.  "Swap-AB": the WEIGHT tile is the UMMA A operand (M = 128 weight rows → 128 TMEM lanes),
// the token tile is the B operand (N = 64 tokens → 64 TMEM columns), so ragged small groups waste no MMA rows.
// Numerics (reading G1): activations must keep fp32 precision, so X is fed as a bf16 hi/lo pair (x ≈ hi + lo,
// |err| ≤ 2^-17|x|) against the EXACT bf16 weight tile: 2 MMAs per k-step into the same fp32 TMEM accumulator.
// SwiGLU mode: gate and up tiles share each X tile and accumulate into two TMEM regions; the epilogue computes
// silu(g)·u in fp32 and writes it straight as the bf16 hi/lo pair the down GEMM consumes.
//
// Warp roles (192 threads, 1 CTA/SM): warp 0 = TMA producer (one lane), warp 1 = TMEM allocator + MMA issuer (one
// lane), warps 2-5 = epilogue (tcgen05.ld 32 lanes × 32 columns each).  One output tile per CTA.
#include <cuda.h>

#include <cstdio>
#include <map>
#include <tuple>

#include "gemm_tc.h"

namespace pmk {

constexpr int TC_BM = 128;      // weight rows per tile (UMMA M)
constexpr int TC_BN = 64;       // tokens per tile (UMMA N)
constexpr int TC_BK = 64;       // k elements per stage (128 bytes of bf16 = one SWIZZLE_128B row)
constexpr int TC_UK = 16;       // UMMA K for 16-bit inputs
constexpr int TC_STAGES = 4;
constexpr int TC_A_BYTES = TC_BM * TC_BK * 2;   // 16 KB
constexpr int TC_B_BYTES = TC_BN * TC_BK * 2;   //  8 KB

// ---- PTX wrappers ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* b, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(smem_u32(b)), "r"(parity) : "memory");
  } while (!ok);
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void umma_bf16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(acc)
      : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, "
      "%24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
// K-major SWIZZLE_128B shared-memory matrix descriptor: rows of 128 bytes, 8-row groups 1024 bytes apart.
__device__ __forceinline__ uint64_t smem_desc_sw128(uint32_t saddr) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr & 0x3ffff) >> 4);        // start address, bits [0,14)
  d |= (uint64_t)1 << 16;                         // leading byte offset (unused for swizzled K-major), bits [16,30)
  d |= (uint64_t)(1024 >> 4) << 32;               // stride byte offset = 1024, bits [32,46)
  d |= (uint64_t)1 << 46;                         // descriptor version (sm_100)
  d |= (uint64_t)2 << 61;                         // layout type SWIZZLE_128B
  return d;
}
constexpr uint32_t kIdesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(TC_BN >> 3) << 17) | ((uint32_t)(TC_BM >> 4) << 24);

struct TcKernelArgs {
  int K, N, a1_row_off;
  const FfnProblem* probs;
  int p0, rows;
  const uint8_t* slot_base;
  unsigned long long a_batch_stride;
  __nv_bfloat16* o_hi;
  unsigned long long o_lo_off;
  int ldo;
  float* y;
  int ldy, flags;
};

// grid (ceil(N/128), ceil(max_rows/64), n_problems), 192 threads, dynamic smem = stages + barriers (1024-aligned).
template <bool SWIGLU>
__global__ void __launch_bounds__(192, 1) gemm_tc_kernel(const __grid_constant__ CUtensorMap mapA0,
                                                         const __grid_constant__ CUtensorMap mapA1,
                                                         const __grid_constant__ CUtensorMap mapB, TcKernelArgs a) {
  constexpr int STAGE_BYTES = (SWIGLU ? 2 : 1) * TC_A_BYTES + 2 * TC_B_BYTES;
  constexpr int TMEM_COLS = SWIGLU ? 2 * TC_BN : TC_BN;
  int row0 = 0, nrows = a.rows, batch = 0;
  if (a.probs) {
    const FfnProblem pb = a.probs[a.p0 + blockIdx.z];
    row0 = pb.row0; nrows = pb.nrows;
    if (a.slot_base) batch = (int)(((const uint8_t*)pb.wg - a.slot_base) / a.a_batch_stride);
  }
  const int rt0 = blockIdx.y * TC_BN;
  if (rt0 >= nrows) return;                       // uniform for the CTA: nothing allocated yet
  const int n0 = blockIdx.x * TC_BM;
  const int nkb = (a.K + TC_BK - 1) / TC_BK;

  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint64_t* full = (uint64_t*)(smem + TC_STAGES * STAGE_BYTES);
  uint64_t* empty = full + TC_STAGES;
  uint64_t* tmem_full = empty + TC_STAGES;
  uint32_t* tmem_slot = (uint32_t*)(tmem_full + 1);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int s = 0; s < TC_STAGES; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, 1); }
    mbar_init(tmem_full, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&mapA0) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&mapB) : "memory");
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(TMEM_COLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    if (lane == 0) {   // ===== TMA producer
      for (int kb = 0; kb < nkb; ++kb) {
        const int s = kb % TC_STAGES;
        mbar_wait(empty + s, ((kb / TC_STAGES) & 1) ^ 1);
        uint8_t* st = smem + s * STAGE_BYTES;
        mbar_expect_tx(full + s, STAGE_BYTES);
        const int kc = kb * TC_BK;
        tma_load_3d(st, &mapA0, full + s, kc, n0, batch);
        if (SWIGLU) tma_load_3d(st + TC_A_BYTES, &mapA1, full + s, kc, a.a1_row_off + n0, batch);
        uint8_t* sb = st + (SWIGLU ? 2 : 1) * TC_A_BYTES;
        tma_load_3d(sb, &mapB, full + s, kc, row0 + rt0, 0);
        tma_load_3d(sb + TC_B_BYTES, &mapB, full + s, kc, row0 + rt0, 1);
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {   // ===== MMA issuer
      for (int kb = 0; kb < nkb; ++kb) {
        const int s = kb % TC_STAGES;
        mbar_wait(full + s, (kb / TC_STAGES) & 1);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const uint32_t sa = smem_u32(smem + s * STAGE_BYTES);
        const uint32_t sb = sa + (SWIGLU ? 2 : 1) * TC_A_BYTES;
#pragma unroll
        for (int k4 = 0; k4 < TC_BK / TC_UK; ++k4) {
          const uint32_t ko = k4 * TC_UK * 2;          // byte advance inside the 128-byte swizzle row
          const uint64_t da0 = smem_desc_sw128(sa + ko);
          const uint64_t dbh = smem_desc_sw128(sb + ko);
          const uint64_t dbl = smem_desc_sw128(sb + TC_B_BYTES + ko);
          const uint32_t first = (kb | k4) ? 1u : 0u;
          umma_bf16(tmem_base, da0, dbh, kIdesc, first);
          umma_bf16(tmem_base, da0, dbl, kIdesc, 1u);
          if (SWIGLU) {
            const uint64_t da1 = smem_desc_sw128(sa + TC_A_BYTES + ko);
            umma_bf16(tmem_base + TC_BN, da1, dbh, kIdesc, first);
            umma_bf16(tmem_base + TC_BN, da1, dbl, kIdesc, 1u);
          }
        }
        umma_commit(empty + s);          // frees the stage when these MMAs have read it
      }
      umma_commit(tmem_full);            // accumulators complete
    }
  } else {             // ===== epilogue warps 2..5: TMEM lanes 32*(warp%4) .. +31
    mbar_wait(tmem_full, 0);
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const int q = warp & 3;
    const int n = n0 + q * 32 + lane;                 // weight row = output feature of this thread
    const uint32_t tlane = tmem_base + ((uint32_t)(q * 32) << 16);
#pragma unroll 1
    for (int c0 = 0; c0 < TC_BN; c0 += 32) {
      uint32_t g[32];
      tmem_ld32(tlane + c0, g);
      if (SWIGLU) {
        uint32_t u[32];
        tmem_ld32(tlane + TC_BN + c0, u);
#pragma unroll
        for (int c = 0; c < 32; ++c) {
          const int r = rt0 + c0 + c;
          if (r < nrows && n < a.N) {
            const float v = silu(__uint_as_float(g[c])) * __uint_as_float(u[c]);
            const __nv_bfloat16 hi = __float2bfloat16_rn(v);
            const __nv_bfloat16 lo = __float2bfloat16_rn(v - __bfloat162float(hi));
            const size_t o = (size_t)(row0 + r) * a.ldo + n;
            a.o_hi[o] = hi;
            a.o_hi[o + a.o_lo_off] = lo;
          }
        }
      } else {
#pragma unroll
        for (int c = 0; c < 32; ++c) {
          const int r = rt0 + c0 + c;
          if (r < nrows && n < a.N) {
            float v = __uint_as_float(g[c]);
            float* yp = a.y + (size_t)(row0 + r) * a.ldy + n;
            if (a.flags & 2) v = fmaxf(v, 0.f);
            if (a.flags & 1) v += *yp;
            *yp = v;
          }
        }
      }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  }
  __syncthreads();
  if (warp == 1) {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(TMEM_COLS) : "memory");
  }
}

// fp32 rows → bf16 hi/lo planes (x ≈ hi + lo); optional row gather through the permutation.
__global__ void __launch_bounds__(256) split_rows_kernel(const float* __restrict__ x, const int32_t* __restrict__ row_src,
                                                         int src_div, int K, __nv_bfloat16* __restrict__ hi,
                                                         size_t lo_off) {
  const int p = blockIdx.x;
  const float* xr = x + (size_t)(row_src ? row_src[p] / src_div : p) * K;
  __nv_bfloat16* h = hi + (size_t)p * K;
  for (int i = threadIdx.x * 4; i < K; i += 1024) {
    const float4 v = *reinterpret_cast<const float4*>(xr + i);
    const float f[4] = {v.x, v.y, v.z, v.w};
    __nv_bfloat16 hh[4], ll[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) { hh[j] = __float2bfloat16_rn(f[j]); ll[j] = __float2bfloat16_rn(f[j] - __bfloat162float(hh[j])); }
    *reinterpret_cast<uint2*>(h + i) = *reinterpret_cast<uint2*>(hh);
    *reinterpret_cast<uint2*>(h + lo_off + i) = *reinterpret_cast<uint2*>(ll);
  }
}
void launch_split_rows(const float* x, const int32_t* row_src, int src_div, int rows, int K, __nv_bfloat16* hi,
                       size_t lo_off, cudaStream_t st) {
  ++g_launches;
  if (rows > 0) split_rows_kernel<<<rows, 256, 0, st>>>(x, row_src, src_div, K, hi, lo_off);
}

// ---- host side ---------------------------------------------------------------------------------------------------
typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                              const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                              CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct TcContext {
  encode_fn encode = nullptr;
  // (base, K, rows, batches, batch stride, box rows) → map
  std::map<std::tuple<const void*, int, int, int, size_t, int>, CUtensorMap> cache;
  bool attr_set = false;
};

TcContext* tc_create(std::string* err) {
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qr;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess ||
      qr != cudaDriverEntryPointSuccess || !fn) {
    (void)cudaGetLastError();
    if (err) *err = "cuTensorMapEncodeTiled is not available from this driver";
    return nullptr;
  }
  TcContext* c = new TcContext();
  c->encode = (encode_fn)fn;
  return c;
}
void tc_destroy(TcContext* c) { delete c; }

// bf16 [batches][rows][K] row-major (K contiguous), box = 64 (k) × box_rows × 1, SWIZZLE_128B, OOB → zeros.
static const CUtensorMap* get_map(TcContext* c, const void* base, int K, int rows, int batches, size_t batch_stride,
                                  int box_rows, std::string* err) {
  auto key = std::make_tuple(base, K, rows, batches, batch_stride, box_rows);
  auto it = c->cache.find(key);
  if (it != c->cache.end()) return &it->second;
  if (((uintptr_t)base & 15) || (((size_t)K * 2) & 15) || (batch_stride & 15)) {
    if (err) *err = "tensor map: base / row pitch / batch stride must be 16-byte aligned";
    return nullptr;
  }
  CUtensorMap m;
  const cuuint64_t dims[3] = {(cuuint64_t)K, (cuuint64_t)rows, (cuuint64_t)batches};
  const cuuint64_t strides[2] = {(cuuint64_t)K * 2, (cuuint64_t)(batch_stride ? batch_stride : (size_t)rows * K * 2)};
  const cuuint32_t box[3] = {(cuuint32_t)TC_BK, (cuuint32_t)box_rows, 1};
  const cuuint32_t es[3] = {1, 1, 1};
  CUresult r = c->encode(&m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, es,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    if (err) *err = "cuTensorMapEncodeTiled failed (" + std::to_string((int)r) + ")";
    return nullptr;
  }
  if (c->cache.size() > 4096) c->cache.clear();
  return &(c->cache[key] = m);
}

bool tc_launch(TcContext* c, const TcGemm& g, cudaStream_t st, std::string* err) {
  ++g_launches;
  if (!c || !g.a0 || !g.b_hi || g.K < 8 || g.N < 1 || (g.K % 8)) { if (err) *err = "tc_launch: unsupported arguments"; return false; }
  const size_t stage = (g.swiglu ? 2 : 1) * (size_t)TC_A_BYTES + 2 * (size_t)TC_B_BYTES;
  const size_t smem = TC_STAGES * stage + 256 + 1024;
  if (!c->attr_set) {
    cudaFuncSetAttribute(gemm_tc_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(TC_STAGES * (2 * TC_A_BYTES + 2 * TC_B_BYTES) + 1280));
    cudaFuncSetAttribute(gemm_tc_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(TC_STAGES * (TC_A_BYTES + 2 * TC_B_BYTES) + 1280));
    c->attr_set = true;
  }
  const CUtensorMap* mA0 = get_map(c, g.a0, g.K, g.a_rows, g.a_batches, g.a_batch_stride, TC_BM, err);
  const CUtensorMap* mA1 = g.swiglu ? get_map(c, g.a1, g.K, g.a_rows, g.a_batches, g.a_batch_stride, TC_BM, err) : mA0;
  // hi and lo planes = "batches" 0 and 1 of the activation map
  const CUtensorMap* mB = get_map(c, g.b_hi, g.K, g.b_rows_cap, 2, g.b_lo_off * 2, TC_BN, err);
  if (!mA0 || !mA1 || !mB) return false;
  TcKernelArgs a{};
  a.K = g.K; a.N = g.N; a.a1_row_off = g.a1_row_off; a.probs = g.probs; a.p0 = g.p0; a.rows = g.rows;
  a.slot_base = g.slot_base; a.a_batch_stride = g.a_batch_stride;
  a.o_hi = g.o_hi; a.o_lo_off = g.o_lo_off; a.ldo = g.ldo; a.y = g.y; a.ldy = g.ldy; a.flags = g.flags;
  const int max_rows = g.probs ? g.max_rows : g.rows;
  if (max_rows <= 0) return true;
  dim3 grid((g.N + TC_BM - 1) / TC_BM, (max_rows + TC_BN - 1) / TC_BN, g.probs ? g.np : 1);
  if (g.swiglu) gemm_tc_kernel<true><<<grid, 192, smem, st>>>(*mA0, *mA1, *mB, a);
  else gemm_tc_kernel<false><<<grid, 192, smem, st>>>(*mA0, *mA1, *mB, a);
  return true;
}

// Load every kernel of this file NOW.  CUDA loads kernels lazily, on their first launch, and that load waits for every
// running kernel to finish: a first launch behind a kernel that spins on a flag (an expert kernel waiting for its bytes,
// the fetch worker waiting for a gate) would dead-lock until the spinner times out (profiles/r02_spin_probe.md).
void preload_tc() {
  preload_fn((const void*)gemm_tc_kernel<true>);
  preload_fn((const void*)gemm_tc_kernel<false>);
  preload_fn((const void*)split_rows_kernel);
}

}  // namespace pmk
