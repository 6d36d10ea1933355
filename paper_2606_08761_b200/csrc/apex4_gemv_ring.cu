// apex4_gemv_ring.cu -- decode-regime kernel for 32 < M <= 64 (three or four m16 token tiles), g = 128.
// Same arithmetic and lane -> k assignment as apex4_gemv.cu (read its header first); what differs is the
// staging.  With 48-64 tokens the token rows of a k-block are 3-4 KB, so per-warp shared-memory stages
// would spend most of their bytes on tokens; here the token fragments of ONE k-block stay in registers
// while the warp walks down all its row blocks, and the weights stream through a per-warp REGISTER ring
// (D - 1 coalesced 512-byte loads in flight per warp).  Partial sums of the 16 warps meet in shared
// memory once per batch of row blocks.
#include <type_traits>

#include "apex4_gemm.cuh"
#include "apex4_layout.cuh"
#include "apex4_ptx.cuh"

namespace apex4 {

namespace gemvr {

constexpr int kWarps = 16;
constexpr int kThreads = 32 * kWarps;
constexpr uint32_t kMask = 0xF0F0F0F0u;
constexpr int kSlotBudget = 192 * 1024;                 // shared memory for the partial sums of a batch

__device__ __forceinline__ uint4 ldg_stream(const uint8_t* p) {   // weights: read once, keep out of L1
  uint4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
               : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}
__device__ __forceinline__ uint4 ldg_cached(const uint8_t* p) {   // tokens: re-read by every CTA
  uint4 v;
  asm volatile("ld.global.nc.v4.u32 {%0, %1, %2, %3}, [%4];"
               : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}
__device__ __forceinline__ uint32_t ldg_u32(const void* p) {
  uint32_t v;
  asm volatile("ld.global.nc.u32 %0, [%1];" : "=r"(v) : "l"(p));
  return v;
}
// D[16x8] = A[16x32] * B[32x8] + C, signed 8-bit operands, INT32 accumulate
__device__ __forceinline__ void mma_s8(int (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k32.row.col.s32.s8.s8.s32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, "
      "{%0, %1, %2, %3};"
      : "+r"(d[0]), "+r"(d[1]), "+r"(d[2]), "+r"(d[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t word(const uint4& v, int i) {
  return i == 0 ? v.x : i == 1 ? v.y : i == 2 ? v.z : v.w;
}

}  // namespace gemvr

using namespace gemvr;

// MT: m16 token tiles (M <= 16 MT); C: k-blocks whose token fragments a warp keeps in registers.
// p.tiles_n = 8-row row blocks, p.upt = row blocks per batch (shared-memory slots), p.kbu = k-blocks
// per group.
template <int MT, int C, bool DUMP>
__global__ void __launch_bounds__(kThreads, 1) w4a4_gemv_ring_kernel(const GemmParams p) {
  constexpr int D = MT == 1 ? 8 : 6;                    // register ring depth (D - 1 loads in flight)
  extern __shared__ float4 slots[];                     // [row block of the batch][warp][MT][lane]
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int q = lane >> 2, t = lane & 3;
  const int KB = p.K / kBlockK;
  const int kbw0 = KB * w / kWarps, kbw1 = KB * (w + 1) / kWarps;    // this warp's k-blocks
  const int rb0 = static_cast<int>(static_cast<long long>(p.tiles_n) * blockIdx.x / gridDim.x);
  const int rb1 = static_cast<int>(static_cast<long long>(p.tiles_n) * (blockIdx.x + 1) / gridDim.x);
  const int rbB = p.upt;
  const size_t row_pitch = static_cast<size_t>(KB) * kBlobBytes;
  const bool swap = (q & 1) != 0;                       // odd token rows: lo / hi nibbles exchanged (PT4)
  // byte offset of this lane's 16-byte chunk (K slice t of row q) inside an 8-row group of a blob
  const uint32_t lane_off = q * kRowBytes + ((t ^ ((q >> 1) & 3)) << 4);

  for (int b0 = rb0; b0 < rb1; b0 += rbB) {
    const int nb = min(rbB, rb1 - b0);
    for (int i = 0; i < nb; ++i)
#pragma unroll
      for (int mi = 0; mi < MT; ++mi) slots[((i * kWarps + w) * MT + mi) * 32 + lane] = make_float4(0.f, 0.f, 0.f, 0.f);

    float yfr[MT][4];
    // One pass = CC k-blocks (kc .. kc + CC - 1) against every row block of the batch.  CC is a
    // compile-time constant so that every register index below is static (a run-time choice of the
    // token fragment compiled to predicated copies of every MMA: 140 instructions per 512-byte unit).
    auto pass = [&](int kc, auto cc_c) {
      constexpr int CC = decltype(cc_c)::value;
      // ---- token fragments and token scales (registers, reused by every row block)
      uint32_t af[CC][MT][4][4];
      float sa[CC][MT][2];
      int gam[CC];
#pragma unroll
      for (int c = 0; c < CC; ++c) {
        const int kb = kc + c;
        gam[c] = kb / p.kbu;
        const uint8_t* ap = p.qA + static_cast<size_t>(kb) * kBlobBytes + lane_off;
#pragma unroll
        for (int mi = 0; mi < MT; ++mi) {
          const uint4 x0 = ldg_cached(ap + (16 * mi) * kRowBytes);
          const uint4 x1 = ldg_cached(ap + (16 * mi + 8) * kRowBytes);
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const uint32_t l0 = rotl4(word(x0, i)) & kMask, h0 = word(x0, i) & kMask;
            const uint32_t l1 = rotl4(word(x1, i)) & kMask, h1 = word(x1, i) & kMask;
            af[c][mi][i][0] = swap ? h0 : l0; af[c][mi][i][2] = swap ? l0 : h0;   // token q: k lo / hi half
            af[c][mi][i][1] = swap ? h1 : l1; af[c][mi][i][3] = swap ? l1 : h1;   // token q + 8
          }
          sa[c][mi][0] = __half2float(p.sA[static_cast<size_t>(gam[c]) * kTileRows + 16 * mi + q]);
          sa[c][mi][1] = __half2float(p.sA[static_cast<size_t>(gam[c]) * kTileRows + 16 * mi + q + 8]);
        }
      }
      // ---- stream the weights of (row block i, k-block c), c fastest, through the register ring:
      // ring slot d always holds k-block d % CC (D is a multiple of CC)
      static_assert(D % CC == 0, "ring depth");
      uint4 wq[D];
      uint32_t sq[D];
      const uint8_t* wbase = p.qW + static_cast<size_t>(kc) * kBlobBytes + lane_off;
      auto issue = [&](int buf, int i, int c) {         // c is static at every call site
        const int row0 = (b0 + i) * 8;
        wq[buf] = ldg_stream(wbase + static_cast<size_t>(row0 >> 7) * row_pitch + static_cast<size_t>(c) * kBlobBytes +
                             (row0 & 127) * kRowBytes);
        const int n0 = row0 + 2 * t;                    // columns 2t, 2t+1 of the accumulator fragment
        sq[buf] = ldg_u32(p.sW + (static_cast<size_t>(n0 >> 7) * p.G + gam[c]) * kTileRows + (n0 & 127));
      };
      constexpr int RB = D / CC;                        // row blocks per ring revolution
#pragma unroll
      for (int d = 0; d < D - 1; ++d)
        if (d / CC < nb) issue(d, d / CC, d % CC);
      for (int ib = 0; ib < nb; ib += RB) {
#pragma unroll
        for (int d = 0; d < D; ++d) {
          const int i = ib + d / CC;                    // row block of the batch
          const int c = d % CC;
          if (i >= nb) break;
          {                                             // prefetch the unit D - 1 ahead
            const int dn = d + D - 1;
            const int in = ib + dn / CC;
            if (in < nb) issue(dn % D, in, dn % CC);
          }
          int acc[MT][4];
#pragma unroll
          for (int mi = 0; mi < MT; ++mi)
#pragma unroll
            for (int e = 0; e < 4; ++e) acc[mi][e] = 0;
#pragma unroll
          for (int k4 = 0; k4 < 4; ++k4) {
            const uint32_t x = word(wq[d], k4);
            const uint32_t b0w = rotl4(x) & kMask, b1w = x & kMask;
#pragma unroll
            for (int mi = 0; mi < MT; ++mi) mma_s8(acc[mi], af[c][mi][k4], b0w, b1w);
          }
          // this k-block's sums: INT32 -> FP32, x sW / 256, x sA (a5)
          const __half2 sw2 = *reinterpret_cast<const __half2*>(&sq[d]);
          const float sw0 = __low2float(sw2) * 0.00390625f, sw1 = __high2float(sw2) * 0.00390625f;
#pragma unroll
          for (int mi = 0; mi < MT; ++mi) {
            const float s0 = sa[c][mi][0], s1 = sa[c][mi][1];
            if (c == 0) {
              yfr[mi][0] = __int2float_rn(acc[mi][0]) * sw0 * s0;
              yfr[mi][1] = __int2float_rn(acc[mi][1]) * sw1 * s0;
              yfr[mi][2] = __int2float_rn(acc[mi][2]) * sw0 * s1;
              yfr[mi][3] = __int2float_rn(acc[mi][3]) * sw1 * s1;
            } else {
              yfr[mi][0] = fmaf(__int2float_rn(acc[mi][0]) * sw0, s0, yfr[mi][0]);
              yfr[mi][1] = fmaf(__int2float_rn(acc[mi][1]) * sw1, s0, yfr[mi][1]);
              yfr[mi][2] = fmaf(__int2float_rn(acc[mi][2]) * sw0, s1, yfr[mi][2]);
              yfr[mi][3] = fmaf(__int2float_rn(acc[mi][3]) * sw1, s1, yfr[mi][3]);
            }
            if constexpr (DUMP) {
#pragma unroll
              for (int e = 0; e < 4; ++e) {
                const int m = 16 * mi + q + 8 * (e >> 1), n = (b0 + i) * 8 + 2 * t + (e & 1);
                if (m >= p.pm0 && m < p.pm1 && n >= p.pn0 && n < p.pn1)   // P_out is zero-filled by the caller
                  atomicAdd(p.P_out + (static_cast<size_t>(m - p.pm0) * (p.pn1 - p.pn0) + (n - p.pn0)) * p.G + gam[c],
                            acc[mi][e] >> 8);
              }
            }
          }
          if (c == CC - 1) {                            // row block done for this pass: add to the warp's slot
#pragma unroll
            for (int mi = 0; mi < MT; ++mi) {
              float4* sl = &slots[((i * kWarps + w) * MT + mi) * 32 + lane];
              float4 v = *sl;
              v.x += yfr[mi][0]; v.y += yfr[mi][1]; v.z += yfr[mi][2]; v.w += yfr[mi][3];
              *sl = v;
            }
          }
        }
      }
    };
    int kc = kbw0;
    for (; kc + C <= kbw1; kc += C) pass(kc, std::integral_constant<int, C>{});
    for (; kc < kbw1; ++kc) pass(kc, std::integral_constant<int, 1>{});

    // ---- a6 / a7: sum the 16 warps' partials of every row block of the batch, cast, store
    __syncthreads();
    if (p.Y != nullptr) {
      for (int i = w; i < nb; i += kWarps) {
#pragma unroll
        for (int mi = 0; mi < MT; ++mi) {
          float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
          for (int ww = 0; ww < kWarps; ++ww) {
            const float4 x = slots[((i * kWarps + ww) * MT + mi) * 32 + lane];
            v.x += x.x; v.y += x.y; v.z += x.z; v.w += x.w;
          }
          const int n = (b0 + i) * 8 + 2 * t;
          const int m = 16 * mi + q;
          if (n < p.N) {
            if (p.out_f32) {
              float* y = static_cast<float*>(p.Y);
              if (m < p.M) *reinterpret_cast<float2*>(y + static_cast<size_t>(m) * p.N + n) = make_float2(v.x, v.y);
              if (m + 8 < p.M) *reinterpret_cast<float2*>(y + static_cast<size_t>(m + 8) * p.N + n) = make_float2(v.z, v.w);
            } else {
              __half* y = static_cast<__half*>(p.Y);
              if (m < p.M) *reinterpret_cast<__half2*>(y + static_cast<size_t>(m) * p.N + n) = __floats2half2_rn(v.x, v.y);
              if (m + 8 < p.M) *reinterpret_cast<__half2*>(y + static_cast<size_t>(m + 8) * p.N + n) = __floats2half2_rn(v.z, v.w);
            }
          }
        }
      }
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------ launcher
template <int MT, int C>
static cudaError_t launch_gemv_ring_mc(const GemmParams& p, bool dump, int grid, cudaStream_t st) {
  const int smem = p.upt * kWarps * MT * 512;
  cudaError_t e;
  if (dump) {
    auto kern = w4a4_gemv_ring_kernel<MT, C, true>;
    if ((e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSlotBudget)) != cudaSuccess) return e;
    kern<<<grid, kThreads, smem, st>>>(p);
  } else {
    auto kern = w4a4_gemv_ring_kernel<MT, C, false>;
    if ((e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSlotBudget)) != cudaSuccess) return e;
    kern<<<grid, kThreads, smem, st>>>(p);
  }
  return cudaGetLastError();
}

// mt: m16 token tiles (1..4).  p.upt (row blocks per batch) must be <= gemv_max_batch(mt).
cudaError_t launch_gemv_ring(const GemmParams& p, int mt, bool dump, int grid, cudaStream_t st) {
  switch (mt) {
    case 3: return launch_gemv_ring_mc<3, 1>(p, dump, grid, st);
    case 4: return launch_gemv_ring_mc<4, 1>(p, dump, grid, st);
    default: return cudaErrorInvalidValue;
  }
}

int gemv_ring_max_batch(int mt) { return kSlotBudget / (kWarps * mt * 512); }

}  // namespace apex4
