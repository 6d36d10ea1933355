// apex4_static_ws.cu -- apex4_w4a4_gemm_static_ws: the W4A4 GEMM for callers that cannot allocate device memory
// (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// The only scratch memory of the GEMM path is the stream-K workspace of the CTA-pair kernel (a6: FP32 partial tiles
// + arrival counters, used when the K loop of an output tile is shared between CTAs).  apex4_w4a4_gemm takes it from the
// caller; this entry point takes it from a file-scope __device__ array of APEX4_STATIC_WORKSPACE_BYTES, which every
// GPU that loads the library holds until the process exits.  Nothing here calls cudaMalloc, cudaFree or an allocating
// library routine; the kernels, the dispatch and the arithmetic are those of apex4_w4a4_gemm (bit-identical outputs).
//
// The array's NAME is a host-side stand-in in host code, not a device address: its address is resolved once per device
// with cudaGetSymbolAddress (that device current, return code checked) and that pointer is what the kernel gets.
// All calls share the array and it keeps the last call's contents: the bytes a call needs are cleared on its stream
// before the launch (the kernel also leaves them zero-filled, but a launch that failed half-way would not), and two calls
// that overlap on the GPU (different streams, no dependency) race on it -- serialise them or use apex4_w4a4_gemm.
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "../../include/apex4.h"

namespace {

static __device__ __align__(256) unsigned char g_static_workspace[APEX4_STATIC_WORKSPACE_BYTES];

constexpr int kMaxDevices = 64;
void* g_ws_ptr[kMaxDevices] = {};      // device address of the array, per device ordinal
std::mutex g_ws_mutex;

// Device address of g_static_workspace on the CURRENT device (resolved on first use, then cached).
int static_workspace(void** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return APEX4_ERR_CUDA;
  if (dev < 0 || dev >= kMaxDevices) return APEX4_ERR_INVALID_ARG;
  std::lock_guard<std::mutex> lock(g_ws_mutex);
  if (g_ws_ptr[dev] == nullptr) {
    void* ptr = nullptr;
    if (cudaGetSymbolAddress(&ptr, g_static_workspace) != cudaSuccess || ptr == nullptr) return APEX4_ERR_CUDA;
    g_ws_ptr[dev] = ptr;
  }
  *out = g_ws_ptr[dev];
  return APEX4_OK;
}

}  // namespace

extern "C" int apex4_w4a4_gemm_static_ws(const void* qA_packed, const void* sA_f16, const void* qW_packed, const void* sW_f16,
                                         void* Y, int out_dtype, int M, int N, int K, int group_size, int gran, int layer,
                                         void* stream) {
  // shape / group-size errors come from the GEMM call below (it validates before it looks at the workspace);
  // an unsupported problem reports 0 bytes here
  const size_t need = apex4_workspace_bytes(M, N, K, group_size, gran, layer);
  if (need > static_cast<size_t>(APEX4_STATIC_WORKSPACE_BYTES)) return APEX4_ERR_WORKSPACE;   // beyond the static maximum
  void* ws = nullptr;
  if (need > 0) {
    const int rc = static_workspace(&ws);
    if (rc != APEX4_OK) return rc;
    if (cudaMemsetAsync(ws, 0, need, static_cast<cudaStream_t>(stream)) != cudaSuccess) return APEX4_ERR_CUDA;
  }
  return apex4_w4a4_gemm(qA_packed, sA_f16, qW_packed, sW_f16, Y, out_dtype, M, N, K, group_size, gran, layer, ws, need, stream);
}
