// apex4_fused_quant.cu -- the activation quantizer of Eq. 7 fused into the op that produces
// its input (the paper only says activations are "quantized online"):
//   apex4_rmsnorm_quantize   x -> RMSNorm(x) * gamma -> INT4 codes + FP16 group scales   (QKV / gate-up inputs)
//   apex4_silu_mul_quantize  SiLU(gate) * up         -> INT4 codes + FP16 group scales   (down_proj input)
// so that the FP16 activation never makes the 2 M K-byte round trip through HBM between its producer and the
// stand-alone quantizer.  The results are DEFINED as quantize(rmsnorm(.)) / quantize(silu_mul(.)) of the
// oracle -- readings R17 / R18 of DESIGN.md -- and are bit-identical to it:
//   R17  ss = sum x^2 exact (FP32 squares of FP16 values are exact; their sum is exact in FP64 in any order),
//        ms = float(ss / K), inv = 1.0f / sqrtf(ms + eps) (IEEE add, sqrt, divide), y = fp16((x * inv) * gamma)
//   R18  y = fp16(silu(gate) * up), the real-valued product rounded once (silu_mul_one in apex4_quant_core.cuh).
// RMSNorm needs a row statistic first: one block per token row, a thread holds U 32-element chunks in registers from
// the load to the packed store.  SiLU * up is elementwise: it is the stand-alone quantizer's kernels with another
// producer of the chunk (apex4_quant.cu).
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "apex4_gemm.cuh"
#include "apex4_layout.cuh"
#include "apex4_ptx.cuh"
#include "apex4_quant_core.cuh"

namespace apex4 {

namespace fused {

constexpr int kThreads = 256;
constexpr int kMaxGroups = 1024;          // K <= 32768, g >= 32

struct RowSmem {
  uint32_t gmax[kMaxGroups];              // FP16 bit pattern of max |y| per group (atomicMax: non-negative halves order as integers)
  double red[kThreads / 32];
  float bcast;
};

// the common tail: y (FP16 words in w[u][16]) -> group absmax -> scales -> codes -> PT4 / ST16, optional FP16 copy
template <int U>
__device__ __forceinline__ void quantize_row_tail(uint32_t (&w)[U][16], RowSmem& sm, int r, int K, int g, uint8_t* __restrict__ q,
                                                  __half* __restrict__ S, __half* __restrict__ y_out) {
  const int cpr = K / 32, cpg = g / 32, G = K / g;
  const int nthr = blockDim.x;
  for (int i = threadIdx.x; i < G; i += nthr) sm.gmax[i] = 0u;
  __syncthreads();
#pragma unroll
  for (int u = 0; u < U; ++u) {
    const int c = threadIdx.x + u * nthr;
    if (c < cpr) {
      atomicMax(&sm.gmax[c / cpg], chunk_absmax_bits(w[u]));
      if (y_out != nullptr) {
        uint4* dst = reinterpret_cast<uint4*>(y_out + static_cast<size_t>(r) * K + c * 32);
#pragma unroll
        for (int i = 0; i < 4; ++i) dst[i] = make_uint4(w[u][4 * i], w[u][4 * i + 1], w[u][4 * i + 2], w[u][4 * i + 3]);
      }
    }
  }
  __syncthreads();
#pragma unroll
  for (int u = 0; u < U; ++u) {
    const int c = threadIdx.x + u * nthr;
    if (c < cpr) {
      const int gamma = c / cpg;
      __half Sh;
      const float s = scale_from_absmax_bits(sm.gmax[gamma], &Sh);
      uint4 packed = quant_chunk(w[u], s);
      if (r & 1) packed = nibble_swap(packed);
      *reinterpret_cast<uint4*>(q + chunk_dst_offset(r, c, K)) = packed;
      if (c % cpg == 0) S[st16_index(r, gamma, G)] = Sh;
    }
  }
}

// rows R .. roundup(R, 128) - 1: zero codes and zero scales (the GEMM kernels bulk-copy whole 128-row blobs)
__device__ __forceinline__ void zero_padding_row(int r, int K, int g, uint8_t* __restrict__ q, __half* __restrict__ S) {
  const int cpr = K / 32, G = K / g;
  for (int c = threadIdx.x; c < cpr; c += blockDim.x) *reinterpret_cast<uint4*>(q + chunk_dst_offset(r, c, K)) = make_uint4(0u, 0u, 0u, 0u);
  for (int i = threadIdx.x; i < G; i += blockDim.x) S[st16_index(r, i, G)] = __float2half_rn(0.f);
}

template <int U>
__global__ void __launch_bounds__(kThreads) rmsnorm_quantize_kernel(const __half* __restrict__ X, const __half* __restrict__ gamma, float eps,
                                                                    int R, int K, int g, uint8_t* __restrict__ q, __half* __restrict__ S,
                                                                    __half* __restrict__ y_out) {
  __shared__ RowSmem sm;
  griddep_wait();
  griddep_launch();
  const int r = blockIdx.x;
  if (r >= R) { zero_padding_row(r, K, g, q, S); return; }
  const int cpr = K / 32, nthr = blockDim.x;
  uint32_t w[U][16];
  double ss = 0.0;
#pragma unroll
  for (int u = 0; u < U; ++u) {
    const int c = threadIdx.x + u * nthr;
    if (c < cpr) {
      const uint4* src = reinterpret_cast<const uint4*>(X + static_cast<size_t>(r) * K + c * 32);
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const uint4 v = __ldg(src + i);
        w[u][4 * i] = v.x; w[u][4 * i + 1] = v.y; w[u][4 * i + 2] = v.z; w[u][4 * i + 3] = v.w;
      }
      // x^2 is exact in binary32 (11-bit significands); groups of four squares are summed in binary32 only where
      // that is exact too -- it is not in general, so every square goes to the FP64 sum on its own
#pragma unroll
      for (int i = 0; i < 16; ++i) {
        const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&w[u][i]));
        ss += static_cast<double>(__fmul_rn(f.x, f.x));
        ss += static_cast<double>(__fmul_rn(f.y, f.y));
      }
    } else {
#pragma unroll
      for (int i = 0; i < 16; ++i) w[u][i] = 0u;
    }
  }
  // exact sum: any order
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, d);
  if ((threadIdx.x & 31) == 0) sm.red[threadIdx.x >> 5] = ss;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int i = 0; i < nthr / 32; ++i) t += sm.red[i];
    const float ms = __double2float_rn(__ddiv_rn(t, static_cast<double>(K)));
    sm.bcast = __fdiv_rn(1.0f, __fsqrt_rn(__fadd_rn(ms, eps)));
  }
  __syncthreads();
  const float inv = sm.bcast;
#pragma unroll
  for (int u = 0; u < U; ++u) {
    const int c = threadIdx.x + u * nthr;
    if (c < cpr) {
      const uint4* gsrc = reinterpret_cast<const uint4*>(gamma + c * 32);
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const uint4 gv = __ldg(gsrc + i);
        const uint32_t gw[4] = {gv.x, gv.y, gv.z, gv.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&w[u][4 * i + j]));
          const float2 gm = __half22float2(*reinterpret_cast<const __half2*>(&gw[j]));
          const __half2 y = __floats2half2_rn(__fmul_rn(__fmul_rn(f.x, inv), gm.x), __fmul_rn(__fmul_rn(f.y, inv), gm.y));
          w[u][4 * i + j] = *reinterpret_cast<const uint32_t*>(&y);
        }
      }
    }
  }
  quantize_row_tail<U>(w, sm, r, K, g, q, S, y_out);
}

}  // namespace fused

static int row_threads(int K, int* U) {
  const int cpr = K / 32;
  const int thr = cpr >= fused::kThreads ? fused::kThreads : (cpr + 31) / 32 * 32;
  const int u = (cpr + thr - 1) / thr;
  *U = u <= 1 ? 1 : u <= 2 ? 2 : 4;
  return thr;
}

cudaError_t launch_rmsnorm_quantize(const void* x, const void* gamma, float eps, int R, int K, int g, void* q, void* s, void* y_out,
                                    cudaStream_t st) {
  int U;
  const int thr = row_threads(K, &U);
  if (K / 32 > 4 * thr || K / g > fused::kMaxGroups) return cudaErrorInvalidValue;
  const dim3 grid(round_up(R, kTileRows)), block(thr);
  const __half* X = static_cast<const __half*>(x);
  const __half* Gm = static_cast<const __half*>(gamma);
  uint8_t* Q = static_cast<uint8_t*>(q);
  __half* S = static_cast<__half*>(s);
  __half* Y = static_cast<__half*>(y_out);
  cudaError_t e;
  if (U == 1) e = launch_pdl(fused::rmsnorm_quantize_kernel<1>, grid, block, 0, st, X, Gm, eps, R, K, g, Q, S, Y);
  else if (U == 2) e = launch_pdl(fused::rmsnorm_quantize_kernel<2>, grid, block, 0, st, X, Gm, eps, R, K, g, Q, S, Y);
  else e = launch_pdl(fused::rmsnorm_quantize_kernel<4>, grid, block, 0, st, X, Gm, eps, R, K, g, Q, S, Y);
  return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace apex4
