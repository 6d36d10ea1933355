// apex4_quant.cu -- a0/a1 of the hot path: the symmetric INT4 group quantizer of Eq. 7
// (PAPER.md:146-150), used online for activations and offline for weights, writing the PT4 / PW4 / ST16
// device layouts of apex4_layout.cuh; plus the code packer / unpacker and scale re-layout twins.
//
// Arithmetic (readings R1-R5 of DESIGN.md): a = max|x| exact in FP16; S = fp16_rn(float(a) / 7.0f)
// with an IEEE binary32 division; q = clamp(rne(x / float(S)), -8, 7) with an IEEE binary32 division
// (rne of the binary32 quotient equals rne of the true quotient for FP16 x and S, lemma L1);
// S == 0 -> q = 0.  Never build this file with -use_fast_math.
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "apex4_gemm.cuh"
#include "apex4_layout.cuh"
#include "apex4_ptx.cuh"
#include "apex4_quant_core.cuh"

namespace apex4 {

// One thread = one 32-element chunk; a group is GL = g/32 consecutive lanes of a warp (GL in 1..32).
// Rows R .. roundup(R, 128) - 1 (the padding of the last 128-row blob, which the GEMM kernels bulk-copy and
// consume) are written as zero codes and zero scales.
template <int GL, class Producer>
__global__ void __launch_bounds__(256) quantize_small_g_kernel(const Producer prod, int R, int Rp,
                                                               int K, uint8_t* __restrict__ q,
                                                               __half* __restrict__ S, int weights) {
  // programmatic dependent launch: X may come from the previous kernel on the stream (wait for it); the next
  // kernel (the GEMM) may start streaming its weights while this one runs
  griddep_wait();
  if (!weights) griddep_launch();   // never ahead of a weight pack: the decode GEMM reads weights before its own wait
  // 32-bit chunk index (the launcher checks Rp * K / 32 < 2^32)
  const uint32_t cpr = static_cast<uint32_t>(K) / 32u;
  const uint32_t total = static_cast<uint32_t>(Rp) * cpr;
  uint32_t gid = blockIdx.x * 256u + threadIdx.x;
  const bool active = gid < total;
  if (!active) gid = total - 1;   // keep the warp converged for the shuffles; results discarded
  const int r = static_cast<int>(gid / cpr);
  const int c = static_cast<int>(gid - static_cast<uint32_t>(r) * cpr);
  uint32_t w[16];
  if (r < R && active) {
    prod.load(r, c, w);
  } else {
#pragma unroll
    for (int i = 0; i < 16; ++i) w[i] = 0u;
  }
  uint32_t m = chunk_absmax_bits(w);
#pragma unroll
  for (int d = 1; d < GL; d <<= 1) m = absmax_bits_max(m, __shfl_xor_sync(0xffffffffu, m, d));
  __half Sh;
  const float s = scale_from_absmax_bits(m, &Sh);
  uint4 packed = quant_chunk(w, s);
  if (!weights && (r & 1)) packed = nibble_swap(packed);
  if (active) {
    *reinterpret_cast<uint4*>(q + chunk_dst_offset(r, c, K)) = packed;
    if ((c % GL) == 0) S[st16_index(r, c / GL, cpr / GL)] = Sh;
  }
}

// One block = one (row, group) with g/32 <= 4 * blockDim chunks; data stays in registers between
// the absmax pass and the quantize pass.
constexpr int kLargeThreads = 256;
constexpr int kLargeUnroll = 4;
template <int U, class Producer>   // U chunks per thread (1, 2 or kLargeUnroll): fewer live registers, more blocks per SM
__global__ void __launch_bounds__(kLargeThreads) quantize_large_g_kernel(
    const Producer prod, int R, int K, int g, uint8_t* __restrict__ q,
    __half* __restrict__ S, int weights) {
  griddep_wait();
  if (!weights) griddep_launch();
  const int G = K / g;
  const int r = blockIdx.x / G;          // r in [0, Rp)
  const int gamma = blockIdx.x % G;
  const int cpg = g / 32;
  const int c0 = gamma * cpg;
  __shared__ uint32_t red[kLargeThreads / 32];
  const int nthr = blockDim.x;          // min(256, chunks per group rounded up to a warp): no idle warps
  uint32_t w[U][16];
  uint32_t m = 0;
#pragma unroll
  for (int u = 0; u < U; ++u) {
    const int cl = threadIdx.x + u * nthr;
    if (cl < cpg && r < R) {
      prod.load(r, c0 + cl, w[u]);
      m = absmax_bits_max(m, chunk_absmax_bits(w[u]));
    } else {
#pragma unroll
      for (int i = 0; i < 16; ++i) w[u][i] = 0u;
    }
  }
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) m = absmax_bits_max(m, __shfl_xor_sync(0xffffffffu, m, d));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
  __syncthreads();
  m = red[0];
  for (int i = 1; i < nthr / 32; ++i) m = absmax_bits_max(m, red[i]);
  __half Sh;
  const float s = scale_from_absmax_bits(m, &Sh);
  if (threadIdx.x == 0) S[st16_index(r, gamma, G)] = Sh;
#pragma unroll
  for (int u = 0; u < U; ++u) {
    const int cl = threadIdx.x + u * nthr;
    if (cl < cpg) {
      uint4 packed = quant_chunk(w[u], s);
      if (!weights && (r & 1)) packed = nibble_swap(packed);
      *reinterpret_cast<uint4*>(q + chunk_dst_offset(r, c0 + cl, K)) = packed;
    }
  }
}

// codes int8 [R,K] -> PT4 (weights = 0) / PW4 (weights = 1)
__global__ void __launch_bounds__(256) pack_codes_kernel(const int8_t* __restrict__ codes, int R,
                                                         int K, uint8_t* __restrict__ q, int weights) {
  const int cpr = K / 32;
  const long long gid = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (gid >= static_cast<long long>(R) * cpr) return;
  const int r = static_cast<int>(gid / cpr), c = static_cast<int>(gid % cpr);
  const uint4* src = reinterpret_cast<const uint4*>(codes + static_cast<size_t>(r) * K + c * 32);
  uint4 in[2] = {__ldg(src), __ldg(src + 1)};
  const int8_t* cd = reinterpret_cast<const int8_t*>(in);
  const int swap = weights ? 0 : (r & 1);
  uint32_t out[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    uint32_t word = 0;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      const int y = 4 * i + b;
      const int lo = swap ? cd[16 + y] : cd[y];
      const int hi = swap ? cd[y] : cd[16 + y];
      word |= static_cast<uint32_t>((lo & 0xF) | ((hi & 0xF) << 4)) << (8 * b);
    }
    out[i] = word;
  }
  *reinterpret_cast<uint4*>(q + chunk_dst_offset(r, c, K)) = make_uint4(out[0], out[1], out[2], out[3]);
}

// PT4 / PW4 -> codes int8 [R,K]
__global__ void __launch_bounds__(256) unpack_codes_kernel(const uint8_t* __restrict__ q, int R,
                                                           int K, int8_t* __restrict__ codes, int weights) {
  const int cpr = K / 32;
  const long long gid = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (gid >= static_cast<long long>(R) * cpr) return;
  const int r = static_cast<int>(gid / cpr), c = static_cast<int>(gid % cpr);
  const uint4 p = __ldg(reinterpret_cast<const uint4*>(q + chunk_dst_offset(r, c, K)));
  const uint8_t* pb = reinterpret_cast<const uint8_t*>(&p);
  const int swap = weights ? 0 : (r & 1);
  int8_t out[32];
#pragma unroll
  for (int y = 0; y < 16; ++y) {
    int lo = pb[y] & 0xF, hi = pb[y] >> 4;
    lo = lo >= 8 ? lo - 16 : lo;
    hi = hi >= 8 ? hi - 16 : hi;
    out[y] = static_cast<int8_t>(swap ? hi : lo);
    out[16 + y] = static_cast<int8_t>(swap ? lo : hi);
  }
  uint4* dst = reinterpret_cast<uint4*>(codes + static_cast<size_t>(r) * K + c * 32);
  dst[0] = *reinterpret_cast<uint4*>(&out[0]);
  dst[1] = *reinterpret_cast<uint4*>(&out[16]);
}

__global__ void scales_from_natural_kernel(const __half* __restrict__ nat, int R, int G,
                                           __half* __restrict__ tiled) {
  const long long gid = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  const long long total = static_cast<long long>(round_up(R, kTileRows)) * G;
  if (gid >= total) return;
  // gid indexes the tiled buffer: ((rt*G + gamma)*128 + rr)
  const int rr = static_cast<int>(gid % kTileRows);
  const long long t = gid / kTileRows;
  const int gamma = static_cast<int>(t % G);
  const int r = static_cast<int>(t / G) * kTileRows + rr;
  tiled[gid] = (r < R) ? nat[static_cast<size_t>(r) * G + gamma] : __float2half_rn(0.f);
}
__global__ void scales_to_natural_kernel(const __half* __restrict__ tiled, int R, int G,
                                         __half* __restrict__ nat) {
  const long long gid = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (gid >= static_cast<long long>(R) * G) return;
  const int r = static_cast<int>(gid / G), gamma = static_cast<int>(gid % G);
  nat[gid] = tiled[st16_index(r, gamma, G)];
}

// ---------------------------------------------------------------------------------- launchers
template <class Producer>
static cudaError_t launch_quantize_with(const Producer& prod, int R, int K, int g, void* q, void* s, int weights, cudaStream_t st) {
  uint8_t* Q = static_cast<uint8_t*>(q);
  __half* S = static_cast<__half*>(s);
  const int gl = g / 32;
  const int Rp = round_up(R, kTileRows);                 // padding rows are written as zeros
  const long long total = static_cast<long long>(Rp) * (K / 32);
  const unsigned blocks = static_cast<unsigned>((total + 255) / 256);
  const bool pow2 = (gl & (gl - 1)) == 0;
  cudaError_t e = cudaSuccess;
  if (pow2 && gl <= 32) {
    if (total + 256 > 0xFFFFFFFFll) return cudaErrorInvalidValue;   // 32-bit chunk index in the kernel
    switch (gl) {
      case 1: e = launch_pdl(quantize_small_g_kernel<1, Producer>, dim3(blocks), dim3(256), 0, st, prod, R, Rp, K, Q, S, weights); break;
      case 2: e = launch_pdl(quantize_small_g_kernel<2, Producer>, dim3(blocks), dim3(256), 0, st, prod, R, Rp, K, Q, S, weights); break;
      case 4: e = launch_pdl(quantize_small_g_kernel<4, Producer>, dim3(blocks), dim3(256), 0, st, prod, R, Rp, K, Q, S, weights); break;
      case 8: e = launch_pdl(quantize_small_g_kernel<8, Producer>, dim3(blocks), dim3(256), 0, st, prod, R, Rp, K, Q, S, weights); break;
      case 16: e = launch_pdl(quantize_small_g_kernel<16, Producer>, dim3(blocks), dim3(256), 0, st, prod, R, Rp, K, Q, S, weights); break;
      default: e = launch_pdl(quantize_small_g_kernel<32, Producer>, dim3(blocks), dim3(256), 0, st, prod, R, Rp, K, Q, S, weights); break;
    }
  } else {
    if (gl > kLargeThreads * kLargeUnroll) return cudaErrorInvalidValue;
    const long long nb = static_cast<long long>(Rp) * (K / g);
    const int threads = gl >= kLargeThreads ? kLargeThreads : (gl + 31) / 32 * 32;
    const unsigned nbu = static_cast<unsigned>(nb);
    if (gl <= kLargeThreads) e = launch_pdl(quantize_large_g_kernel<1, Producer>, dim3(nbu), dim3(threads), 0, st, prod, R, K, g, Q, S, weights);
    else if (gl <= 2 * kLargeThreads) e = launch_pdl(quantize_large_g_kernel<2, Producer>, dim3(nbu), dim3(threads), 0, st, prod, R, K, g, Q, S, weights);
    else e = launch_pdl(quantize_large_g_kernel<kLargeUnroll, Producer>, dim3(nbu), dim3(threads), 0, st, prod, R, K, g, Q, S, weights);
  }
  return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_quantize(const void* x, int R, int K, int g, void* q, void* s, int weights, cudaStream_t st) {
  return launch_quantize_with(PlainLoad{static_cast<const __half*>(x), K}, R, K, g, q, s, weights, st);
}

// SiLU(gate) * up fused into the quantizer: the same kernels with another producer of the chunk
cudaError_t launch_silu_mul_quantize(const void* gate, const void* up, int ld, int R, int K, int g, void* q, void* s, void* y_out,
                                     cudaStream_t st) {
  return launch_quantize_with(SiluMulLoad{static_cast<const __half*>(gate), static_cast<const __half*>(up), static_cast<__half*>(y_out), ld, K},
                              R, K, g, q, s, 0, st);
}

bool quantize_supports_group(int g) {
  const int gl = g / 32;
  return ((gl & (gl - 1)) == 0 && gl <= 32) || gl <= kLargeThreads * kLargeUnroll;
}
cudaError_t launch_pack_codes(const int8_t* codes, int R, int K, void* q, int weights, cudaStream_t st) {
  const long long total = static_cast<long long>(R) * (K / 32);
  pack_codes_kernel<<<static_cast<unsigned>((total + 255) / 256), 256, 0, st>>>(
      codes, R, K, static_cast<uint8_t*>(q), weights);
  return cudaGetLastError();
}
cudaError_t launch_unpack_codes(const void* q, int R, int K, int8_t* codes, int weights, cudaStream_t st) {
  const long long total = static_cast<long long>(R) * (K / 32);
  unpack_codes_kernel<<<static_cast<unsigned>((total + 255) / 256), 256, 0, st>>>(
      static_cast<const uint8_t*>(q), R, K, codes, weights);
  return cudaGetLastError();
}
cudaError_t launch_scales_from_natural(const void* nat, int R, int G, void* tiled, cudaStream_t st) {
  const long long total = static_cast<long long>(round_up(R, kTileRows)) * G;
  scales_from_natural_kernel<<<static_cast<unsigned>((total + 255) / 256), 256, 0, st>>>(
      static_cast<const __half*>(nat), R, G, static_cast<__half*>(tiled));
  return cudaGetLastError();
}
cudaError_t launch_scales_to_natural(const void* tiled, int R, int G, void* nat, cudaStream_t st) {
  const long long total = static_cast<long long>(R) * G;
  scales_to_natural_kernel<<<static_cast<unsigned>((total + 255) / 256), 256, 0, st>>>(
      static_cast<const __half*>(tiled), R, G, static_cast<__half*>(nat));
  return cudaGetLastError();
}

}  // namespace apex4
