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

namespace apex4 {

__device__ __forceinline__ uint32_t hmax2_abs(uint32_t acc, uint32_t v) {
  __half2 a = *reinterpret_cast<__half2*>(&acc);
  __half2 b = __habs2(*reinterpret_cast<__half2*>(&v));
  __half2 m = __hmax2(a, b);
  return *reinterpret_cast<uint32_t*>(&m);
}

__device__ __forceinline__ int quant_one(float x, float s) {
  // s > 0 here.  IEEE division, round-half-to-even, clamp (Eq. 7).
  int q = __float2int_rn(__fdiv_rn(x, s));
  return max(-8, min(7, q));
}

// 32 FP16 values (4 x uint4) -> 16 packed bytes (one PT4 / PW4 chunk).  swap: the second
// 16-element half lands in the low nibbles (PT4 odd rows; never for PW4, apex4_layout.cuh).
__device__ __forceinline__ uint4 quant_pack_chunk(const uint4 (&v)[4], float s, int swap) {
  int code[32];
  const uint32_t* w = reinterpret_cast<const uint32_t*>(v);
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    __half2 h = *reinterpret_cast<const __half2*>(&w[i]);
    float2 f = __half22float2(h);
    code[2 * i] = (s == 0.f) ? 0 : quant_one(f.x, s);
    code[2 * i + 1] = (s == 0.f) ? 0 : quant_one(f.y, s);
  }
  uint32_t out[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    uint32_t word = 0;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      const int y = 4 * i + b;
      const int lo = swap ? code[16 + y] : code[y];
      const int hi = swap ? code[y] : code[16 + y];
      word |= static_cast<uint32_t>((lo & 0xF) | ((hi & 0xF) << 4)) << (8 * b);
    }
    out[i] = word;
  }
  return make_uint4(out[0], out[1], out[2], out[3]);
}

// The same 16 bytes without a division per element.  rne(x / s) is decided from two products that
// bracket the true quotient, x * inv * (1 -/+ 2^-20) with inv = rn(1 / s): each FFMA adds 1.5 * 2^23, so
// the FP32 rounding of the sum IS round-half-to-even to an integer, and its low mantissa nibble is the
// two's-complement code.  Rounding is monotonic, so when both ends give the same integer the true
// quotient (and by lemma L1 the binary32 quotient of quant_one) rounds to it too.  When they differ for
// any element of the chunk (the quotient is within ~1e-5 of a half-integer: ~5e-4 of all chunks), or S
// is an FP16 subnormal (only then can |x / S| exceed 7.5 and the clamp of Eq. 7 act), the chunk is
// redone by quant_pack_chunk with IEEE divisions.  Codes are bit-identical to quant_pack_chunk's.
__device__ __forceinline__ uint4 quant_pack_chunk_fast(const uint4 (&v)[4], float s, int swap) {
  if (s == 0.f) return make_uint4(0u, 0u, 0u, 0u);
  if (s < 6.103515625e-05f) return quant_pack_chunk(v, s, swap);   // S below 2^-14
  const float inv = __frcp_rn(s);
  const float inv_lo = inv * 0.99999904632568359375f;   // 1 - 2^-20
  const float inv_hi = inv * 1.00000095367431640625f;   // 1 + 2^-20
  const float magic = 12582912.0f;                      // 1.5 * 2^23: ulp 1, integer in the mantissa
  const uint32_t* w = reinterpret_cast<const uint32_t*>(v);
  uint32_t chk = 0;
  uint32_t byte[16];                                    // byte y = element y (low nibble), 16 + y (high)
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const float2 fa = __half22float2(*reinterpret_cast<const __half2*>(&w[swap ? 8 + i : i]));
    const float2 fb = __half22float2(*reinterpret_cast<const __half2*>(&w[swap ? i : 8 + i]));
    const uint32_t a0 = __float_as_uint(__fmaf_rn(fa.x, inv_lo, magic)), a0h = __float_as_uint(__fmaf_rn(fa.x, inv_hi, magic));
    const uint32_t a1 = __float_as_uint(__fmaf_rn(fa.y, inv_lo, magic)), a1h = __float_as_uint(__fmaf_rn(fa.y, inv_hi, magic));
    const uint32_t b0 = __float_as_uint(__fmaf_rn(fb.x, inv_lo, magic)), b0h = __float_as_uint(__fmaf_rn(fb.x, inv_hi, magic));
    const uint32_t b1 = __float_as_uint(__fmaf_rn(fb.y, inv_lo, magic)), b1h = __float_as_uint(__fmaf_rn(fb.y, inv_hi, magic));
    chk |= (a0 ^ a0h) | (a1 ^ a1h);
    chk |= (b0 ^ b0h) | (b1 ^ b1h);
    byte[2 * i] = (a0 & 0xFu) | (b0 << 4);              // bits 8.. are junk, dropped by the byte gather
    byte[2 * i + 1] = (a1 & 0xFu) | (b1 << 4);
  }
  if (chk != 0) return quant_pack_chunk(v, s, swap);
  uint32_t out[4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
    out[i] = __byte_perm(__byte_perm(byte[4 * i], byte[4 * i + 1], 0x0040),
                         __byte_perm(byte[4 * i + 2], byte[4 * i + 3], 0x0040), 0x5410);
  return make_uint4(out[0], out[1], out[2], out[3]);
}

__device__ __forceinline__ float scale_from_absmax_bits(uint32_t amax_bits, __half* S_out) {
  __half a = __ushort_as_half(static_cast<unsigned short>(amax_bits));
  float s32 = __fdiv_rn(__half2float(a), 7.0f);
  __half S = __float2half_rn(s32);
  *S_out = S;
  return __half2float(S);
}

__device__ __forceinline__ size_t chunk_dst_offset(int r, int c, int K) {
  const int rt = r / kTileRows, rr = r % kTileRows;
  const int kb = c >> 2, s = c & 3;
  const int j = s ^ ((rr >> 1) & 3);
  return pt4_blob_offset(rt, kb, K) + static_cast<size_t>(rr) * kRowBytes + j * 16;
}

// One thread = one 32-element chunk; a group is GL = g/32 consecutive lanes of a warp (GL in 1..32).
template <int GL>
__global__ void __launch_bounds__(256) quantize_small_g_kernel(const __half* __restrict__ X, int R,
                                                               int K, uint8_t* __restrict__ q,
                                                               __half* __restrict__ S, int weights) {
  // 32-bit chunk index (the launcher checks R * K / 32 < 2^32): a 64-bit division here was ~150 of the
  // ~500 instructions of a thread
  // programmatic dependent launch: X may come from the previous kernel on the stream (wait for it); the next
  // kernel (the GEMM) may start streaming its weights while this one runs
  griddep_wait();
  if (!weights) griddep_launch();   // never ahead of a weight pack: the decode GEMM reads weights before its own wait
  const uint32_t cpr = static_cast<uint32_t>(K) / 32u;
  const uint32_t total = static_cast<uint32_t>(R) * cpr;
  uint32_t gid = blockIdx.x * 256u + threadIdx.x;
  const bool active = gid < total;
  if (!active) gid = total - 1;   // keep the warp converged for the shuffles; results discarded
  const int r = static_cast<int>(gid / cpr);
  const int c = static_cast<int>(gid - static_cast<uint32_t>(r) * cpr);
  const uint4* src = reinterpret_cast<const uint4*>(X + static_cast<size_t>(r) * K + c * 32);
  uint4 v[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) v[i] = __ldg(src + i);
  uint32_t m = 0;
  const uint32_t* w = reinterpret_cast<const uint32_t*>(v);
#pragma unroll
  for (int i = 0; i < 16; ++i) m = hmax2_abs(m, w[i]);
  {  // fold the two halves, then across the group's lanes
    __half2 mm = *reinterpret_cast<__half2*>(&m);
    __half h = __hmax(__low2half(mm), __high2half(mm));
    m = __half_as_ushort(h);
  }
#pragma unroll
  for (int d = 1; d < GL; d <<= 1) {
    uint32_t o = __shfl_xor_sync(0xffffffffu, m, d);
    __half a = __ushort_as_half(static_cast<unsigned short>(m));
    __half b = __ushort_as_half(static_cast<unsigned short>(o));
    m = __half_as_ushort(__hmax(a, b));
  }
  __half Sh;
  const float s = scale_from_absmax_bits(m, &Sh);
  const uint4 packed = quant_pack_chunk_fast(v, s, weights ? 0 : (r & 1));
  if (active) {
    *reinterpret_cast<uint4*>(q + chunk_dst_offset(r, c, K)) = packed;
    if ((c % GL) == 0) S[st16_index(r, c / GL, cpr / GL)] = Sh;
  }
}

// One block = one (row, group) with g/32 <= 4 * blockDim chunks; data stays in registers between
// the absmax pass and the quantize pass.
constexpr int kLargeThreads = 256;
constexpr int kLargeUnroll = 4;
template <int U>   // chunks per thread (1, 2 or kLargeUnroll): fewer live registers, more blocks per SM
__global__ void __launch_bounds__(kLargeThreads) quantize_large_g_kernel(
    const __half* __restrict__ X, int R, int K, int g, uint8_t* __restrict__ q,
    __half* __restrict__ S, int weights) {
  griddep_wait();
  if (!weights) griddep_launch();
  const int G = K / g;
  const int r = blockIdx.x / G;
  const int gamma = blockIdx.x % G;
  const int cpg = g / 32;
  const int c0 = gamma * cpg;
  __shared__ uint32_t red[kLargeThreads / 32];
  const int nthr = blockDim.x;          // min(256, chunks per group rounded up to a warp): no idle warps
  uint4 v[U][4];
  uint32_t m = 0;
#pragma unroll
  for (int u = 0; u < U; ++u) {
    const int cl = threadIdx.x + u * nthr;
    if (cl < cpg) {
      const uint4* src =
          reinterpret_cast<const uint4*>(X + static_cast<size_t>(r) * K + (c0 + cl) * 32);
#pragma unroll
      for (int i = 0; i < 4; ++i) v[u][i] = __ldg(src + i);
      const uint32_t* w = reinterpret_cast<const uint32_t*>(v[u]);
#pragma unroll
      for (int i = 0; i < 16; ++i) m = hmax2_abs(m, w[i]);
    }
  }
  {
    __half2 mm = *reinterpret_cast<__half2*>(&m);
    m = __half_as_ushort(__hmax(__low2half(mm), __high2half(mm)));
  }
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    uint32_t o = __shfl_xor_sync(0xffffffffu, m, d);
    m = __half_as_ushort(__hmax(__ushort_as_half(static_cast<unsigned short>(m)),
                                __ushort_as_half(static_cast<unsigned short>(o))));
  }
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
  __syncthreads();
  m = red[0];
  for (int i = 1; i < nthr / 32; ++i)
    m = __half_as_ushort(__hmax(__ushort_as_half(static_cast<unsigned short>(m)),
                                __ushort_as_half(static_cast<unsigned short>(red[i]))));
  __half Sh;
  const float s = scale_from_absmax_bits(m, &Sh);
  if (threadIdx.x == 0) S[st16_index(r, gamma, G)] = Sh;
#pragma unroll
  for (int u = 0; u < U; ++u) {
    const int cl = threadIdx.x + u * nthr;
    if (cl < cpg) {
      const uint4 packed = quant_pack_chunk_fast(v[u], s, weights ? 0 : (r & 1));
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
cudaError_t launch_quantize(const void* x, int R, int K, int g, void* q, void* s, int weights,
                            cudaStream_t st) {
  const __half* X = static_cast<const __half*>(x);
  uint8_t* Q = static_cast<uint8_t*>(q);
  __half* S = static_cast<__half*>(s);
  const int gl = g / 32;
  const long long total = static_cast<long long>(R) * (K / 32);
  const unsigned blocks = static_cast<unsigned>((total + 255) / 256);
  const bool pow2 = (gl & (gl - 1)) == 0;
  cudaError_t e = cudaSuccess;
  if (pow2 && gl <= 32) {
    if (total + 256 > 0xFFFFFFFFll) return cudaErrorInvalidValue;   // 32-bit chunk index in the kernel
    switch (gl) {
      case 1: e = launch_pdl(quantize_small_g_kernel<1>, dim3(blocks), dim3(256), 0, st, X, R, K, Q, S, weights); break;
      case 2: e = launch_pdl(quantize_small_g_kernel<2>, dim3(blocks), dim3(256), 0, st, X, R, K, Q, S, weights); break;
      case 4: e = launch_pdl(quantize_small_g_kernel<4>, dim3(blocks), dim3(256), 0, st, X, R, K, Q, S, weights); break;
      case 8: e = launch_pdl(quantize_small_g_kernel<8>, dim3(blocks), dim3(256), 0, st, X, R, K, Q, S, weights); break;
      case 16: e = launch_pdl(quantize_small_g_kernel<16>, dim3(blocks), dim3(256), 0, st, X, R, K, Q, S, weights); break;
      default: e = launch_pdl(quantize_small_g_kernel<32>, dim3(blocks), dim3(256), 0, st, X, R, K, Q, S, weights); break;
    }
  } else {
    if (gl > kLargeThreads * kLargeUnroll) return cudaErrorInvalidValue;
    const long long nb = static_cast<long long>(R) * (K / g);
    const int threads = gl >= kLargeThreads ? kLargeThreads : (gl + 31) / 32 * 32;
    const unsigned nbu = static_cast<unsigned>(nb);
    if (gl <= kLargeThreads) e = launch_pdl(quantize_large_g_kernel<1>, dim3(nbu), dim3(threads), 0, st, X, R, K, g, Q, S, weights);
    else if (gl <= 2 * kLargeThreads) e = launch_pdl(quantize_large_g_kernel<2>, dim3(nbu), dim3(threads), 0, st, X, R, K, g, Q, S, weights);
    else e = launch_pdl(quantize_large_g_kernel<kLargeUnroll>, dim3(nbu), dim3(threads), 0, st, X, R, K, g, Q, S, weights);
  }
  return e != cudaSuccess ? e : cudaGetLastError();
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
