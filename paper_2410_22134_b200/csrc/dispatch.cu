// dispatch.cu — choice between the tcgen05 tensor-core GEMMs (gemm_tc.cu) and the SIMT fp32 GEMMs for the
// T > 1 (prefill) linears and grouped expert FFNs.
#include "kernels.h"

namespace pmk {

void launch_linear_gemm(const float* x, const void* w, float* y, int T, int N, int K, int wdtype, int flags,
                        bool tensor, cudaStream_t st) {
  (void)tensor;
  launch_gemm_simt(x, w, y, T, N, K, wdtype, flags, st);
}
void launch_ffn_gateup_gemm(const float* x, const int32_t* row_src, int src_div, const FfnProblem* probs, int p0,
                            int np, int max_rows, int rows_override, int max_inter, int H, float* act,
                            int act_stride, int wdtype, bool tensor, cudaStream_t st) {
  (void)tensor;
  launch_ffn_gateup_gemm_simt(x, row_src, src_div, probs, p0, np, max_rows, rows_override, max_inter, H, act,
                              act_stride, wdtype, st);
}
void launch_ffn_down_gemm(const float* act, int act_stride, const FfnProblem* probs, int p0, int np, int max_rows,
                          int rows_override, int max_inter, int H, float* y, int wdtype, bool tensor,
                          cudaStream_t st) {
  (void)tensor;
  launch_ffn_down_gemm_simt(act, act_stride, probs, p0, np, max_rows, rows_override, max_inter, H, y, wdtype, st);
}

}  // namespace pmk
