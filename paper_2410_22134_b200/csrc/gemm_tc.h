// gemm_tc.h — host interface of the tcgen05/TMEM/TMA GEMM (gemm_tc.cu).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

#include "common.cuh"

namespace pmk {

struct TcContext;   // tensor-map cache + driver entry point
TcContext* tc_create(std::string* err);
void tc_destroy(TcContext* c);

// One launch: Y[rows, N] = X[rows, K] · W[N, K]^T for one problem (probs == nullptr) or a problem list.
struct TcGemm {
  // weights (bf16, row-major [N, K]); swiglu: a0 = gate, a1 = up.  Slot images: a0 = a1 = slot region base,
  // a_rows = 2*I, a1_row_off = I, batches = number of slots, batch stride = Be.
  const void* a0 = nullptr;
  const void* a1 = nullptr;
  int a_rows = 0, a1_row_off = 0, a_batches = 1;
  size_t a_batch_stride = 0;
  // activations as a bf16 hi/lo pair: hi plane at b_hi [b_rows_cap, K], lo plane b_lo_off elements later
  const __nv_bfloat16* b_hi = nullptr;
  size_t b_lo_off = 0;
  int b_rows_cap = 0;
  int K = 0, N = 0;
  const FfnProblem* probs = nullptr;   // device; row ranges (and, with slot_base, the slot of each problem)
  int p0 = 0, np = 1, rows = 0, max_rows = 0;
  const uint8_t* slot_base = nullptr;  // batch index of a problem = (pb.wg - slot_base) / a_batch_stride
  // outputs
  bool swiglu = false;
  __nv_bfloat16* o_hi = nullptr;       // swiglu: silu(g)*u as hi/lo planes [.., ldo]
  size_t o_lo_off = 0;
  int ldo = 0;
  float* y = nullptr;                  // linear: fp32 [.., ldy]; flags LIN_ACC / LIN_RELU
  int ldy = 0, flags = 0;
};
// false + err when the shape is unsupported or the tensor map could not be encoded
bool tc_launch(TcContext* c, const TcGemm& g, cudaStream_t st, std::string* err);

// x fp32 [.., K] rows → bf16 hi/lo planes; row p reads x[row_src ? row_src[p] / src_div : p].
void launch_split_rows(const float* x, const int32_t* row_src, int src_div, int rows, int K, __nv_bfloat16* hi,
                       size_t lo_off, cudaStream_t st);

}  // namespace pmk
