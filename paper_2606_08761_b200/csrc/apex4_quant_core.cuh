// apex4_quant_core.cuh -- the arithmetic of Eq. 7 on one 32-element chunk held in
// registers, shared by the stand-alone quantizer (apex4_quant.cu) and the producer-fused quantizers
// (apex4_fused_quant.cu).  Readings R1-R5 of DESIGN.md: a = max|x| exact in FP16; S = fp16_rn(float(a) / 7.0f)
// with an IEEE binary32 division; q = clamp(rne(x / float(S)), -8, 7); S == 0 -> q = 0.
// Never build with -use_fast_math.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "apex4_layout.cuh"

namespace apex4 {

// max |x| over 16 packed half2 words -> FP16 bit pattern of the maximum (a non-negative half)
__device__ __forceinline__ uint32_t chunk_absmax_bits(const uint32_t (&w)[16]) {
  __half2 m = __habs2(*reinterpret_cast<const __half2*>(&w[0]));
#pragma unroll
  for (int i = 1; i < 16; ++i) m = __hmax2(m, __habs2(*reinterpret_cast<const __half2*>(&w[i])));
  return __half_as_ushort(__hmax(__low2half(m), __high2half(m)));
}
__device__ __forceinline__ uint32_t absmax_bits_max(uint32_t a, uint32_t b) {
  // non-negative FP16 bit patterns order like unsigned integers
  return a > b ? a : b;
}

// S = fp16_rn(float(absmax) / 7.0f); returns float(S)
__device__ __forceinline__ float scale_from_absmax_bits(uint32_t amax_bits, __half* S_out) {
  const __half a = __ushort_as_half(static_cast<unsigned short>(amax_bits));
  const __half S = __float2half_rn(__fdiv_rn(__half2float(a), 7.0f));
  *S_out = S;
  return __half2float(S);
}

__device__ __forceinline__ int quant_one(float x, float s) {
  // s > 0 here.  IEEE division, round-half-to-even, clamp (Eq. 7).
  const int q = __float2int_rn(__fdiv_rn(x, s));
  return max(-8, min(7, q));
}

__device__ __forceinline__ uint32_t quant_byte(float lo, float hi, float s) {
  return static_cast<uint32_t>(quant_one(lo, s) & 0xF) | (static_cast<uint32_t>(quant_one(hi, s) & 0xF) << 4);
}

// Reference path: one IEEE division per element.  Output word j of the 16-byte chunk = bytes 4j .. 4j + 3; byte y
// holds element y in the low nibble and element 16 + y in the high nibble (apex4_layout.cuh; the PT4 odd-row
// exchange is applied by the caller through nibble_swap).  Word j comes from input words 2j, 2j + 1 (elements
// 4j .. 4j + 3) and 8 + 2j, 9 + 2j (elements 16 + 4j .. 16 + 4j + 3).
__device__ __forceinline__ uint32_t quant_word_exact(uint32_t wa0, uint32_t wa1, uint32_t wb0, uint32_t wb1, float s) {
  if (s == 0.f) return 0u;
  const float2 a0 = __half22float2(*reinterpret_cast<const __half2*>(&wa0)), a1 = __half22float2(*reinterpret_cast<const __half2*>(&wa1));
  const float2 b0 = __half22float2(*reinterpret_cast<const __half2*>(&wb0)), b1 = __half22float2(*reinterpret_cast<const __half2*>(&wb1));
  return quant_byte(a0.x, b0.x, s) | (quant_byte(a0.y, b0.y, s) << 8) | (quant_byte(a1.x, b1.x, s) << 16) | (quant_byte(a1.y, b1.y, s) << 24);
}
__device__ __forceinline__ uint4 quant_chunk_exact(const uint32_t (&w)[16], float s) {
  return make_uint4(quant_word_exact(w[0], w[1], w[8], w[9], s), quant_word_exact(w[2], w[3], w[10], w[11], s),
                    quant_word_exact(w[4], w[5], w[12], w[13], s), quant_word_exact(w[6], w[7], w[14], w[15], s));
}

// The same 16 bytes without a division per element.  rne(x / s) is decided from two products that bracket
// the true quotient, x * inv * (1 -/+ 2^-20) with inv = rn(1 / s): each FFMA adds 1.5 * 2^23, so the FP32
// rounding of the sum IS round-half-to-even to an integer, and its low mantissa nibble is the two's-complement
// code.  Rounding is monotonic, so when both ends give the same integer the true quotient (and by lemma L1 of
// SURVEY 8(c) the binary32 quotient of quant_one) rounds to it too.  When they differ for an element (the
// quotient is within ~1e-5 of a half-integer or -- far more often with FP16 operands -- EXACTLY a half-integer:
// ~3e-4 of all elements), the 8-element output word it belongs to is redone with IEEE divisions; the whole chunk
// is when S is an FP16 subnormal (only then can |x / S| exceed 7.5 and the clamp of Eq. 7 act).  The fallback
// is per word, not per chunk: one flagged lane makes its whole warp walk the branch (a quarter of all warps
// did, at ~480 instructions per chunk).
__device__ __forceinline__ uint4 quant_chunk(const uint32_t (&w)[16], float s) {
  if (s < 6.103515625e-05f) return quant_chunk_exact(w, s);   // S = 0 or below 2^-14
  const float inv = __frcp_rn(s);
  const float inv_lo = inv * 0.99999904632568359375f;   // 1 - 2^-20
  const float inv_hi = inv * 1.00000095367431640625f;   // 1 + 2^-20
  const float magic = 12582912.0f;                      // 1.5 * 2^23: ulp 1, integer in the mantissa
  uint32_t out[4];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    uint32_t lo[4], hi[4];
    uint32_t chk = 0;
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const float2 fa = __half22float2(*reinterpret_cast<const __half2*>(&w[2 * j + h]));
      const float2 fb = __half22float2(*reinterpret_cast<const __half2*>(&w[8 + 2 * j + h]));
      const uint32_t a0 = __float_as_uint(__fmaf_rn(fa.x, inv_lo, magic)), a0h = __float_as_uint(__fmaf_rn(fa.x, inv_hi, magic));
      const uint32_t a1 = __float_as_uint(__fmaf_rn(fa.y, inv_lo, magic)), a1h = __float_as_uint(__fmaf_rn(fa.y, inv_hi, magic));
      const uint32_t b0 = __float_as_uint(__fmaf_rn(fb.x, inv_lo, magic)), b0h = __float_as_uint(__fmaf_rn(fb.x, inv_hi, magic));
      const uint32_t b1 = __float_as_uint(__fmaf_rn(fb.y, inv_lo, magic)), b1h = __float_as_uint(__fmaf_rn(fb.y, inv_hi, magic));
      chk |= (a0 ^ a0h) | (a1 ^ a1h);
      chk |= (b0 ^ b0h) | (b1 ^ b1h);
      lo[2 * h] = a0; lo[2 * h + 1] = a1; hi[2 * h] = b0; hi[2 * h + 1] = b1;
    }
    // low bytes of lo[0..3] -> one word, of hi[0..3] -> one word; then nibble-interleave
    const uint32_t L = __byte_perm(__byte_perm(lo[0], lo[1], 0x0040), __byte_perm(lo[2], lo[3], 0x0040), 0x5410);
    const uint32_t H = __byte_perm(__byte_perm(hi[0], hi[1], 0x0040), __byte_perm(hi[2], hi[3], 0x0040), 0x5410);
    out[j] = (L & 0x0F0F0F0Fu) | ((H << 4) & 0xF0F0F0F0u);
    if (chk != 0) out[j] = quant_word_exact(w[2 * j], w[2 * j + 1], w[8 + 2 * j], w[9 + 2 * j], s);
  }
  return make_uint4(out[0], out[1], out[2], out[3]);
}

// ------------------------------------------------------------------ producers of a chunk (what the quantizer kernels read)
// plain: the FP16 activation / weight matrix itself
struct PlainLoad {
  const __half* X;
  int K;
  __device__ __forceinline__ void load(int r, int c, uint32_t (&w)[16]) const {
    const uint4* src = reinterpret_cast<const uint4*>(X + static_cast<size_t>(r) * K + c * 32);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const uint4 v = __ldg(src + i);
      w[4 * i] = v.x; w[4 * i + 1] = v.y; w[4 * i + 2] = v.z; w[4 * i + 3] = v.w;
    }
  }
};

// y = fp16(silu(g) * u), silu(g) = g / (1 + exp(-g)): the real-valued product rounded ONCE (R18).
// Fast path in binary32 with relative error below 1.25 * 2^-21 = 10 * 2^-24:
//   exp(-g) = ex2(th) * (1 + tl ln 2), th + tl = -g log2(e) to ~2^-45 (th = fl(-g L1), tl its FMA residual plus -g L2):
//             ex2.approx <= 2^-22 relative (PTX ISA), the correction factor adds 2^-24;
//   1 + e: 2^-24;  rcp.approx: 2^-23 (PTX ISA);  g * r and * u: 2^-24 each.
// The result is accepted when both ends of a +-2^-20 interval round to the same FP16 value (rounding is monotonic);
// otherwise (~0.3 % of the elements: an FP16 rounding boundary inside the interval), and for |g| > 83 where ex2 leaves
// its normal range, it is recomputed in binary64.
__device__ __forceinline__ __half silu_mul_one(float g, float u) {
  const float L1 = 1.44269502162933349609375f;          // fl(log2 e)
  const float L2 = 1.9259629911783013e-08f;             // log2 e - L1
  const float th = __fmul_rn(-g, L1);
  const float tl = __fmaf_rn(-g, L2, __fmaf_rn(-g, L1, -th));
  float e;
  asm("ex2.approx.f32 %0, %1;" : "=f"(e) : "f"(th));
  e = __fmul_rn(e, __fmaf_rn(tl, 0.693147182464599609375f, 1.0f));
  const float d = __fadd_rn(1.0f, e);
  float r;
  asm("rcp.approx.f32 %0, %1;" : "=f"(r) : "f"(d));
  const float y = __fmul_rn(__fmul_rn(g, r), u);
  const __half lo = __float2half_rn(y * 0.99999904632568359375f);   // 1 - 2^-20
  const __half hi = __float2half_rn(y * 1.00000095367431640625f);   // 1 + 2^-20
  // th in the normal range of ex2 and 1 + e finite: otherwise (g < -87: e overflows; g > 87: e is flushed) take the slow path
  if (__half_as_ushort(lo) == __half_as_ushort(hi) && fabsf(th) < 120.0f) return lo;
  const double gd = static_cast<double>(g);
  const double s = gd / (1.0 + exp(-gd));               // exp(-gd) = inf for gd < -709: s = -0, as in the oracle
  return __double2half(s * static_cast<double>(u));
}

struct SiluMulLoad {
  const __half* gate;
  const __half* up;
  __half* y_out;                                        // optional FP16 copy [M,K]
  int ld, K;
  __device__ __forceinline__ void load(int r, int c, uint32_t (&w)[16]) const {
    const uint4* gsrc = reinterpret_cast<const uint4*>(gate + static_cast<size_t>(r) * ld + c * 32);
    const uint4* usrc = reinterpret_cast<const uint4*>(up + static_cast<size_t>(r) * ld + c * 32);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const uint4 gv = __ldg(gsrc + i), uv = __ldg(usrc + i);
      const uint32_t gw[4] = {gv.x, gv.y, gv.z, gv.w}, uw[4] = {uv.x, uv.y, uv.z, uv.w};
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const float2 gf = __half22float2(*reinterpret_cast<const __half2*>(&gw[j]));
        const float2 uf = __half22float2(*reinterpret_cast<const __half2*>(&uw[j]));
        const __half2 y = __halves2half2(silu_mul_one(gf.x, uf.x), silu_mul_one(gf.y, uf.y));
        w[4 * i + j] = *reinterpret_cast<const uint32_t*>(&y);
      }
    }
    if (y_out != nullptr) {
      uint4* dst = reinterpret_cast<uint4*>(y_out + static_cast<size_t>(r) * K + c * 32);
#pragma unroll
      for (int i = 0; i < 4; ++i) dst[i] = make_uint4(w[4 * i], w[4 * i + 1], w[4 * i + 2], w[4 * i + 3]);
    }
  }
};

// PT4 odd rows keep the second 16-element half in the LOW nibbles (apex4_layout.cuh): exchange the nibbles of every byte
__device__ __forceinline__ uint4 nibble_swap(uint4 v) {
  auto sw = [](uint32_t x) { return ((x >> 4) & 0x0F0F0F0Fu) | ((x << 4) & 0xF0F0F0F0u); };
  return make_uint4(sw(v.x), sw(v.y), sw(v.z), sw(v.w));
}

// destination of chunk c (32 elements) of row r inside the PT4 / PW4 buffer
__device__ __forceinline__ size_t chunk_dst_offset(int r, int c, int K) {
  const int rt = r / kTileRows, rr = r % kTileRows;
  const int kb = c >> 2, s = c & 3;
  const int j = s ^ ((rr >> 1) & 3);
  return pt4_blob_offset(rt, kb, K) + static_cast<size_t>(rr) * kRowBytes + j * 16;
}

}  // namespace apex4
