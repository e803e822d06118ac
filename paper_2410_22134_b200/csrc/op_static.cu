// op_static.cu — promoe_op_expert_ffn_static: the batch-1 SwiGLU expert FFN (A9 decode) for callers that
// may not allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// promoe_op_expert_ffn (api.cu) takes its scratch (the [I] activation vector between the gate/up and the down GEMV and
// the 64-byte problem record) from the caller.  This variant keeps that scratch in ONE file-scope device array of a
// fixed, modest size — kStaticMaxInter floats + one record = 64.25 KiB, held by every GPU that loads the library until
// the process exits — and calls no cudaMalloc, cudaFree or allocating library routine; the caller passes only inputs and
// the output.  The same GEMV kernels as the allocating path run (kernels_ffn.cu), so the result is bit-identical.
//
// The array's NAME is a host-side stand-in in host code, not a device address: its device address is taken once per
// device (with that device current) through cudaGetSymbolAddress and handed to the kernels.
// Every call on a device shares the array: two calls that overlap on the GPU (different streams, no ordering) race on
// it; calls on one stream are ordered.  Nothing in it has to start at zero — the gate/up GEMV overwrites all
// `inter` activations and the record is rewritten by every call — so the previous call's contents never matter.
#include "kernels.h"
#include "../../include/promoe.h"

using namespace pmk;

namespace {

constexpr int kStaticMaxInter = 16384;      // floats of activation scratch: covers c4's I = 14336 (BASELINE.json configs[3])
constexpr int kStaticRecordOff = kStaticMaxInter * (int)sizeof(float);
constexpr int kStaticBytes = kStaticRecordOff + 256;
constexpr int kMaxDevices = 64;

}  // namespace

static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];

// The problem record travels as a kernel argument (no host→device copy from the caller's stack: capture-safe).
__global__ void static_record_kernel(FfnProblem* dst, FfnProblem pb) { *dst = pb; }

// device address of g_static_scratch on the CURRENT device, resolved once per device
static unsigned char* static_scratch_ptr(int* rc) {
  static unsigned char* ptr[kMaxDevices] = {};
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) { *rc = PROMOE_ECUDA; return nullptr; }
  if (!ptr[dev]) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_static_scratch) != cudaSuccess || !p) { (void)cudaGetLastError(); *rc = PROMOE_ECUDA; return nullptr; }
    ptr[dev] = (unsigned char*)p;
  }
  *rc = PROMOE_OK;
  return ptr[dev];
}

extern "C" int promoe_op_expert_ffn_static(const float* x, const void* wg, const void* wu, const void* wd, float* y,
                                           int32_t H, int32_t I, int32_t wdtype, void* stream) {
  if (!x || !wg || !wu || !wd || !y || H < 16 || I < 16 || H % 16 || I % 16 || (wdtype != 0 && wdtype != 1)) return PROMOE_EINVAL;
  if (I > kStaticMaxInter) return PROMOE_EINVAL;     // beyond the static scratch: use promoe_op_expert_ffn with caller scratch
  int rc = PROMOE_OK;
  unsigned char* base = static_scratch_ptr(&rc);
  if (!base) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  float* act = (float*)base;
  FfnProblem* rec = (FfnProblem*)(base + kStaticRecordOff);
  FfnProblem pb{};
  pb.wg = wg; pb.wu = wu; pb.wd = wd; pb.flags = nullptr; pb.gen = 0; pb.inter = I; pb.row0 = 0; pb.nrows = 1; pb.expert = -1;
  ++g_launches;
  static_record_kernel<<<1, 1, 0, st>>>(rec, pb);
  launch_ffn_gateup_gemv(x, rec, 1, I, H, act, I, wdtype, (size_t)1 << 20, nullptr, st);
  launch_ffn_down_gemv(act, I, rec, 1, I, H, y, wdtype, (size_t)1 << 20, nullptr, st);
  return cudaGetLastError() == cudaSuccess ? PROMOE_OK : PROMOE_ECUDA;
}

extern "C" int promoe_op_expert_ffn_static_max_inter(void) { return kStaticMaxInter; }
