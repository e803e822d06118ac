/* promoe_bench.h — measurement hooks of the B200-native ProMoE library used ONLY by bench.py (not product API).
 *
 * They exist because BASELINE.json's metric is a fraction of a roofline whose terms must be measured on the box:
 * the pinned host->device bandwidth (the H2D term, "chosen from measured PCIe H2D bandwidth") and the live duration
 * of the dominant decode kernel (tier framing (4): CUDA events on the launching stream, inside bench.py).
 * Same conventions as promoe.h: 0 or a negative PROMOE_E* code, plain pointers and sizes.
 */
#ifndef PROMOE_BENCH_H
#define PROMOE_BENCH_H
#include "promoe.h"
#ifdef __cplusplus
extern "C" {
#endif

/* Measured pinned host->device bandwidth (GB/s) for `bytes`-sized copies at queue depth `depth`, best of `reps`
 * (chunk size is chosen from this curve).  Allocates and frees its own buffers. */
PROMOE_API int promoe_bench_h2d(size_t bytes, int32_t depth, int32_t reps, double* gbs_out);

/* Live kernel timing for bench.py's roofline: runs `reps` launches of one hot kernel of the decode step on the
 * handle's compute stream, bracketed by CUDA events, over RESIDENT slots rotating through all layers (working set =
 * the whole slot region, far larger than L2).  which: 0 = A9 gate/up SwiGLU GEMV over top_k experts, 1 = A9 down +
 * combine over top_k experts.  Outputs the average launch duration (ms) and the algorithmic weight bytes one launch
 * streams.  The handle must have its experts loaded; its cache state is not touched. */
PROMOE_API int promoe_bench_kernel_time(promoe_t* h, int32_t which, int32_t reps, double* avg_ms_out, double* bytes_per_launch_out);

#ifdef __cplusplus
}
#endif
#endif /* PROMOE_BENCH_H */
