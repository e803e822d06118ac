// kernels_dense.cu — embedding, RMSNorm, linear (GEMV / SIMT GEMM) kernels.  sm_100a.
// Rows A0, A1 and the linear parts of A2/A3/A4/A5/A10 of DESIGN.md.
#include "kernels.h"

namespace pmk {

// ---------------------------------------------------------------------------------------------------------
// A0 embedding lookup
template <typename WT>
__global__ void embed_kernel(const int32_t* __restrict__ ids, const WT* __restrict__ emb, float* __restrict__ x,
                             int H, const uint32_t* alive, uint32_t alive_want, int* err) {
  if (alive) {      // fused decode: the step starts only once its fetch worker is resident (kernels.h)
    if (threadIdx.x == 0) {
      const unsigned long long t0 = globaltimer_ns();
      while (ld_acquire_sys(alive) != alive_want) {
        if (globaltimer_ns() - t0 > kFlagTimeoutNs) { atomicExch(err, 1); break; }
        __nanosleep(200);
      }
    }
    __syncthreads();
  }
  const int t = blockIdx.x;
  const WT* row = emb + (size_t)ids[t] * H;
  for (int i = threadIdx.x; i < H; i += blockDim.x) x[(size_t)t * H + i] = wload1(row + i);
}
void launch_embed(const int32_t* ids, const void* emb, float* x, int T, int H, int wdtype, cudaStream_t st,
                  const uint32_t* alive, uint32_t alive_want, int* err) {
  ++g_launches;
  if (wdtype == 0) embed_kernel<float><<<T, 256, 0, st>>>(ids, (const float*)emb, x, H, alive, alive_want, err);
  else embed_kernel<__nv_bfloat16><<<T, 256, 0, st>>>(ids, (const __nv_bfloat16*)emb, x, H, alive, alive_want, err);
}

// ---------------------------------------------------------------------------------------------------------
// A1 RMSNorm: one CTA of 256 threads per row; x row kept in registers between the two passes.
__global__ void __launch_bounds__(256) rmsnorm_kernel(const float* __restrict__ x, const float* __restrict__ w,
                                                      float* __restrict__ y, int H, float eps) {
  const int t = blockIdx.x;
  const float* xr = x + (size_t)t * H;
  float ss = 0.f;
  for (int i = threadIdx.x; i < H; i += 256) { float v = xr[i]; ss += v * v; }
  __shared__ float red[8];
  ss = warp_sum(ss);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = ss;
  __syncthreads();
  float tot = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) tot += red[i];
  const float r = rsqrtf(tot / (float)H + eps);
  for (int i = threadIdx.x; i < H; i += 256) y[(size_t)t * H + i] = xr[i] * r * w[i];
}
void launch_rmsnorm(const float* x, const float* w, float* y, int T, int H, float eps, cudaStream_t st) {
  ++g_launches;
  rmsnorm_kernel<<<T, 256, 0, st>>>(x, w, y, H, eps);
}

// ---------------------------------------------------------------------------------------------------------
// GEMV: y[n] (+)= sum_k x[k] W[n,k].  HBM-streaming: one warp per output row, each lane issues 16-byte
// weight loads (UNR independent loads in flight), x read through L1 (it is tiny and shared by all warps).
// Summation order is fixed by (K, lane) only, so results do not depend on where the weights live.
template <typename WT>
__global__ void __launch_bounds__(256) gemv_kernel(const float* __restrict__ x, const WT* __restrict__ w,
                                                   float* __restrict__ y, int N, int K, int flags) {
  const int lane = threadIdx.x & 31;
  const int warp = (blockIdx.x * 256 + threadIdx.x) >> 5;
  const int nwarps = (gridDim.x * 256) >> 5;
  pdl_enter();
  for (int n = warp; n < N; n += nwarps) {
    // rows of <= 8 passes (O-projection, K = 2048 bf16): every load in flight at once; same summation order
    float v = (K <= 8 * 32 * WVec<WT>::N) ? row_dot_short<WT, 8>(w + (size_t)n * K, x, K, lane) : row_dot<WT>(w + (size_t)n * K, x, K, lane);
    if (lane == 0) {
      if (flags & LIN_RELU) v = fmaxf(v, 0.f);
      if (flags & LIN_ACC) v += y[n];
      y[n] = v;
    }
  }
  pdl_done();
}
void launch_gemv(const float* x, const void* w, float* y, int N, int K, int wdtype, int flags, cudaStream_t st) {
  ++g_launches;
  int blocks = (N + 7) / 8;
  if (blocks > 148 * 8) blocks = 148 * 8;   // 8 CTAs x 8 warps resident per SM; grid-stride over rows
  if (wdtype == 0) launch_pdl(gemv_kernel<float>, dim3(blocks), dim3(256), 0, st, x, (const float*)w, y, N, K, flags);
  else launch_pdl(gemv_kernel<__nv_bfloat16>, dim3(blocks), dim3(256), 0, st, x, (const __nv_bfloat16*)w, y, N, K, flags);
}

// Small-N linear for T > 1 (e.g. the shared expert's scalar gate, N = 1): one warp per output element y[t, n].
template <typename WT>
__global__ void __launch_bounds__(256) linear_small_n_kernel(const float* __restrict__ x, const WT* __restrict__ w,
                                                             float* __restrict__ y, int T, int N, int K, int flags) {
  const int lane = threadIdx.x & 31;
  const int o = (blockIdx.x * 256 + threadIdx.x) >> 5;
  if (o >= T * N) return;
  const int t = o / N, n = o % N;
  float v = row_dot<WT>(w + (size_t)n * K, x + (size_t)t * K, K, lane);
  if (lane == 0) {
    if (flags & LIN_RELU) v = fmaxf(v, 0.f);
    if (flags & LIN_ACC) v += y[o];
    y[o] = v;
  }
}
void launch_linear_small_n(const float* x, const void* w, float* y, int T, int N, int K, int wdtype, int flags,
                           cudaStream_t st) {
  ++g_launches;
  const int blocks = (T * N + 7) / 8;
  if (wdtype == 0) linear_small_n_kernel<float><<<blocks, 256, 0, st>>>(x, (const float*)w, y, T, N, K, flags);
  else linear_small_n_kernel<__nv_bfloat16><<<blocks, 256, 0, st>>>(x, (const __nv_bfloat16*)w, y, T, N, K, flags);
}

// ---------------------------------------------------------------------------------------------------------
// SIMT fp32 GEMM  Y[T,N] (+)= X[T,K] . W[N,K]^T.  64x64x16 tiles, 256 threads, 4x4 micro-tile per thread.
// Correctness path for prefill (the tcgen05 kernel in gemm_tc.cu is the fast path for bf16 weights).
constexpr int GB = 64, GK = 16;
template <typename WT>
__global__ void __launch_bounds__(256) gemm_simt_kernel(const float* __restrict__ x, const WT* __restrict__ w,
                                                        float* __restrict__ y, int T, int N, int K, int flags) {
  __shared__ float xs[GK][GB + 4];
  __shared__ float ws[GK][GB + 4];
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  const int m0 = blockIdx.y * GB, n0 = blockIdx.x * GB;
  float acc[4][4] = {};
  const int lr = threadIdx.x >> 2;         // 0..63 row of the tile this thread loads
  const int lk = (threadIdx.x & 3) * 4;    // 0,4,8,12 k offset
  for (int k0 = 0; k0 < K; k0 += GK) {
    {
      const int m = m0 + lr;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int kk = k0 + lk + q;
        xs[lk + q][lr] = (m < T && kk < K) ? x[(size_t)m * K + kk] : 0.f;
      }
      const int n = n0 + lr;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int kk = k0 + lk + q;
        ws[lk + q][lr] = (n < N && kk < K) ? wload1(w + (size_t)n * K + kk) : 0.f;
      }
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < GK; ++kk) {
      float a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = xs[kk][ty * 4 + i];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = ws[kk][tx * 4 + j];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int m = m0 + ty * 4 + i;
    if (m >= T) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int n = n0 + tx * 4 + j;
      if (n >= N) continue;
      float v = acc[i][j];
      if (flags & LIN_RELU) v = fmaxf(v, 0.f);
      if (flags & LIN_ACC) v += y[(size_t)m * N + n];
      y[(size_t)m * N + n] = v;
    }
  }
}
void launch_gemm_simt(const float* x, const void* w, float* y, int T, int N, int K, int wdtype, int flags,
                      cudaStream_t st) {
  ++g_launches;
  dim3 grid((N + GB - 1) / GB, (T + GB - 1) / GB);
  if (wdtype == 0) gemm_simt_kernel<float><<<grid, 256, 0, st>>>(x, (const float*)w, y, T, N, K, flags);
  else gemm_simt_kernel<__nv_bfloat16><<<grid, 256, 0, st>>>(x, (const __nv_bfloat16*)w, y, T, N, K, flags);
}

__global__ void add_kernel(const float* __restrict__ a, const float* __restrict__ b, float* __restrict__ out,
                           size_t n) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = a[i] + b[i];
}
void launch_add(const float* a, const float* b, float* out, size_t n, cudaStream_t st) {
  ++g_launches;
  add_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(a, b, out, n);
}

// Load every kernel of this file NOW.  CUDA loads kernels lazily, on their first launch, and that load waits for every
// running kernel to finish: a first launch behind a kernel that spins on a flag (an expert kernel waiting for its bytes,
// the fetch worker waiting for a gate) would dead-lock until the spinner times out (profiles/r02_spin_probe.md).
void preload_dense() {
  preload_fn((const void*)embed_kernel<float>);
  preload_fn((const void*)embed_kernel<__nv_bfloat16>);
  preload_fn((const void*)rmsnorm_kernel);
  preload_fn((const void*)gemv_kernel<float>);
  preload_fn((const void*)gemv_kernel<__nv_bfloat16>);
  preload_fn((const void*)linear_small_n_kernel<float>);
  preload_fn((const void*)linear_small_n_kernel<__nv_bfloat16>);
  preload_fn((const void*)gemm_simt_kernel<float>);
  preload_fn((const void*)gemm_simt_kernel<__nv_bfloat16>);
  preload_fn((const void*)add_kernel);
}

}  // namespace pmk
