// apex4_gemm.cu -- a2..a7 of the hot path: the W4A4 group-dequant GEMM of Eq. 8
// for sm_100a.  One CTA computes one 128 x NC output tile over a k-block range:
//
//   warp 0      producer : 1-D bulk async copies (TMA engine) of PT4 blobs + ST16 scales -> smem ring
//   warp 1      MMA      : one thread issues tcgen05.mma kind::i8 (K = 32 per instruction) into the
//                          TMEM accumulator of the current K-group; tcgen05.commit hands stages back
//   warps 4-7   wideners : packed INT4 -> INT8 (x16, sign kept) straight into the 128B-swizzled UMMA
//                          operand layout; also FP16 -> FP32 scale conversion into a small ring
//   warps 8+    epilogue : tcgen05.ld the finished group's INT32 tile, I2F, x sC (uniform), FMA with
//                          sR (per row) into FP32 registers -- while the next group's MMAs run into
//                          the other TMEM buffer (the overlap the paper says Ampere cannot do,
//                          PAPER.md:84); finally cast + store (or split-K reduce).
//
// Integer exactness: operands are 16*q, so the accumulator holds 256 * P_g with |256 P_g| <= 2^21
// for g <= 128 and < 2^31 for any K <= 32768; the 2^-8 is folded into the row scale (exact).
#include "apex4_gemm.cuh"
#include "apex4_layout.cuh"
#include "apex4_ptx.cuh"

namespace apex4 {

template <int NC>
struct GemmCfg {
  static constexpr int kColHalves = NC > 128 ? 2 : 1;          // epilogue warpgroups
  static constexpr int kCPT = NC / kColHalves;                 // accumulator columns per epilogue thread
  static constexpr int kThreads = 256 + 128 * kColHalves;
  static constexpr int kPkStages = 4;
  static constexpr int kI8Stages = NC > 128 ? 2 : 3;
  static constexpr int kScfSlots = 8;
  static constexpr int kCTiles = (NC + 127) / 128;             // 128-row blobs per C tile
  static constexpr int kCPackedBytes = NC * kRowBytes;         // packed bytes of a C tile per k-block
  static constexpr int kPkRBytes = kBlobBytes;
  static constexpr int kPkScaleRBytes = 4 * 256;               // up to 4 groups per k-block
  static constexpr int kPkScaleCBytes = 4 * 256 * kCTiles;
  static constexpr int kPkStageBytes = kPkRBytes + kCPackedBytes + kPkScaleRBytes + kPkScaleCBytes;
  static constexpr int kI8RBytes = kTileRows * kBlockK;        // 16384
  static constexpr int kI8CBytes = NC * kBlockK;
  static constexpr int kI8StageBytes = kI8RBytes + kI8CBytes;
  static constexpr int kScfSlotBytes = (kTileRows + NC) * 4;
  static constexpr int kTmemColsPerBuf = NC;
  static constexpr uint32_t kTmemCols = (2 * NC <= 32) ? 32 : (2 * NC <= 64) ? 64 : (2 * NC <= 128) ? 128
                                        : (2 * NC <= 256) ? 256 : 512;
  // register re-balancing between warpgroups (setmaxnreg): only the CPT = 128 epilogues need it
  static constexpr bool kRebalance = kCPT == 128;
  static constexpr int kRegsCtl = NC > 128 ? 40 : 56;      // warps 0-3 (producer, MMA)
  static constexpr int kRegsWiden = NC > 128 ? 88 : 96;    // warps 4-7
  static constexpr int kRegsEpi = NC > 128 ? 192 : 240;    // warps 8+
  static constexpr int kNumBars = 2 * kPkStages + 2 * kI8Stages + 2 * kScfSlots + 4;
  static constexpr int kSmemBytes = 1024 /*align slack*/ + kI8Stages * kI8StageBytes +
                                    kPkStages * kPkStageBytes + kScfSlots * kScfSlotBytes +
                                    kNumBars * 8 + 64;
};

__device__ __forceinline__ float i2f(uint32_t v) { return __int2float_rn(static_cast<int>(v)); }

template <int NC, bool DUMP>
__global__ void __launch_bounds__(GemmCfg<NC>::kThreads, 1) w4a4_gemm_kernel(const GemmParams p) {
  using Cfg = GemmCfg<NC>;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));

  // ---- carve-up (offsets from the 1024-aligned base)
  constexpr uint32_t offI8 = 0;
  constexpr uint32_t offPk = offI8 + Cfg::kI8Stages * Cfg::kI8StageBytes;
  constexpr uint32_t offScf = offPk + Cfg::kPkStages * Cfg::kPkStageBytes;
  constexpr uint32_t offBar = offScf + Cfg::kScfSlots * Cfg::kScfSlotBytes;
  constexpr uint32_t offTmemPtr = offBar + Cfg::kNumBars * 8;
  auto bar = [&](int i) { return smem_base + offBar + 8u * i; };
  constexpr int bPkFull = 0, bPkEmpty = bPkFull + Cfg::kPkStages, bI8Full = bPkEmpty + Cfg::kPkStages,
                bI8Empty = bI8Full + Cfg::kI8Stages, bScfFull = bI8Empty + Cfg::kI8Stages,
                bScfEmpty = bScfFull + Cfg::kScfSlots, bAccFull = bScfEmpty + Cfg::kScfSlots,
                bAccEmpty = bAccFull + 2;

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const int ct = blockIdx.x, rt = blockIdx.y, split = blockIdx.z;
  const int KB = p.K / kBlockK;
  const int kb0 = split * p.kb_per_split;
  const int kb1 = min(KB, kb0 + p.kb_per_split);
  const int nkb = kb1 - kb0;
  const int g = p.g;
  const int gpk = g < kBlockK ? kBlockK / g : 1;        // groups per k-block (1, 2, 4)
  const int kbpg = g > kBlockK ? g / kBlockK : 1;       // k-blocks per group
  const int ngroups = g < kBlockK ? nkb * gpk : nkb / kbpg;
  // valid packed rows of the C tile (the last tile of an operand with an odd number of 128-row
  // blobs has only one blob)
  const int Cp = round_up(p.C, kTileRows);
  const int c_row0 = ct * NC;
  const int c_rows = min(NC, Cp - c_row0);

  if (threadIdx.x == 0) {
    for (int i = 0; i < Cfg::kPkStages; ++i) { mbar_init(bar(bPkFull + i), 1); mbar_init(bar(bPkEmpty + i), 128); }
    for (int i = 0; i < Cfg::kI8Stages; ++i) { mbar_init(bar(bI8Full + i), 128); mbar_init(bar(bI8Empty + i), 1); }
    for (int i = 0; i < Cfg::kScfSlots; ++i) { mbar_init(bar(bScfFull + i), 128); mbar_init(bar(bScfEmpty + i), 128 * Cfg::kColHalves); }
    for (int i = 0; i < 2; ++i) { mbar_init(bar(bAccFull + i), 1); mbar_init(bar(bAccEmpty + i), 128 * Cfg::kColHalves); }
    fence_mbar_init();
  }
  if (warp == 1) tmem_alloc<Cfg::kTmemCols>(smem_base + offTmemPtr);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(smem_gen + offTmemPtr);

  // =========================================================================== producer
  if (warp < 4) {
    if constexpr (Cfg::kRebalance) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(Cfg::kRegsCtl));
    if (warp == 0 && lane == 0) {
      const int c_tiles_valid = (c_rows + kTileRows - 1) / kTileRows;
      const uint32_t sc_bytes = gpk * 256;
      for (int it = 0; it < nkb; ++it) {
        const int kb = kb0 + it;
        const int s = it % Cfg::kPkStages;
        const uint32_t ph = (it / Cfg::kPkStages) & 1;
        mbar_wait(bar(bPkEmpty + s), ph ^ 1);
        const uint32_t st = smem_base + offPk + s * Cfg::kPkStageBytes;
        const bool has_scales = (kbpg == 1) || (it % kbpg == 0);
        const int gfirst = g < kBlockK ? kb * gpk : kb / kbpg;
        uint32_t bytes = kBlobBytes + c_rows * kRowBytes;
        if (has_scales) bytes += sc_bytes * (1 + c_tiles_valid);
        mbar_arrive_expect_tx(bar(bPkFull + s), bytes);
        bulk_g2s(st, p.qR + pt4_blob_offset(rt, kb, p.K), kBlobBytes, bar(bPkFull + s));
        for (int b = 0; b < c_tiles_valid; ++b) {
          const int rows_b = min(kTileRows, c_rows - b * kTileRows);
          const int crow = c_row0 + b * kTileRows;
          bulk_g2s(st + Cfg::kPkRBytes + b * kBlobBytes,
                   p.qC + pt4_blob_offset(crow / kTileRows, kb, p.K) + (crow % kTileRows) * kRowBytes,
                   rows_b * kRowBytes, bar(bPkFull + s));
        }
        if (has_scales) {
          bulk_g2s(st + Cfg::kPkRBytes + Cfg::kCPackedBytes,
                   p.sR + (static_cast<size_t>(rt) * p.G + gfirst) * kTileRows, sc_bytes,
                   bar(bPkFull + s));
          for (int b = 0; b < c_tiles_valid; ++b) {
            const int crt = (c_row0 + b * kTileRows) / kTileRows;
            bulk_g2s(st + Cfg::kPkRBytes + Cfg::kCPackedBytes + Cfg::kPkScaleRBytes + b * sc_bytes,
                     p.sC + (static_cast<size_t>(crt) * p.G + gfirst) * kTileRows, sc_bytes,
                     bar(bPkFull + s));
          }
        }
      }
    }
    // ========================================================================= MMA issuer
    else if (warp == 1 && lane == 0) {
      constexpr uint32_t idesc = umma_idesc_i8(kTileRows, NC);
      int acc_it = 0;
      for (int it = 0; it < nkb; ++it) {
        const int t = it % Cfg::kI8Stages;
        const uint32_t ph = (it / Cfg::kI8Stages) & 1;
        mbar_wait(bar(bI8Full + t), ph);
        tc_fence_after();
        const uint32_t i8 = smem_base + offI8 + t * Cfg::kI8StageBytes;
        const uint64_t adesc = umma_desc_sw128(i8);
        const uint64_t bdesc = umma_desc_sw128(i8 + Cfg::kI8RBytes);
        const int ks_per_sub = 4 / gpk;
        for (int sub = 0; sub < gpk; ++sub) {
          const bool first = (kbpg == 1) || (it % kbpg == 0);
          const bool last = (kbpg == 1) || (it % kbpg == kbpg - 1);
          const int buf = acc_it & 1;
          if (first) {
            mbar_wait(bar(bAccEmpty + buf), ((acc_it >> 1) & 1) ^ 1);
            tc_fence_after();
          }
          const uint32_t d = tmem_base + buf * Cfg::kTmemColsPerBuf;
          for (int ks = 0; ks < ks_per_sub; ++ks) {
            const uint32_t koff = (sub * ks_per_sub + ks) * 2;   // 32 bytes per K=32 slice, >>4
            mma_i8_ss(d, adesc + koff, bdesc + koff, idesc, (first && ks == 0) ? 0u : 1u);
          }
          if (last) {
            tc_commit(bar(bAccFull + buf));
            ++acc_it;
          }
        }
        tc_commit(bar(bI8Empty + t));
      }
    }
  }
  // =========================================================================== wideners
  else if (warp < 8) {
    if constexpr (Cfg::kRebalance) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(Cfg::kRegsWiden));
    const int w = threadIdx.x - 128;
    // a lane whose (lane>>2)&1 is set stores its hi chunk first: the two 16-byte stores of a quarter
    // warp then cover all 32 banks (32-byte stride would otherwise hit each bank twice)
    const uint32_t flip = ((lane >> 2) & 1) * 16;
    int grp = 0;
    for (int it = 0; it < nkb; ++it) {
      const int s = it % Cfg::kPkStages;
      const uint32_t phs = (it / Cfg::kPkStages) & 1;
      const int t = it % Cfg::kI8Stages;
      const uint32_t pht = (it / Cfg::kI8Stages) & 1;
      mbar_wait(bar(bPkFull + s), phs);
      mbar_wait(bar(bI8Empty + t), pht ^ 1);
      const uint8_t* pk = smem_gen + offPk + s * Cfg::kPkStageBytes;
      const uint32_t pk_addr = smem_base + offPk + s * Cfg::kPkStageBytes;
      const uint32_t i8_addr = smem_base + offI8 + t * Cfg::kI8StageBytes;
      // packed byte offset o -> INT8 byte offsets 2o (lo nibbles) and 2o+16 (hi nibbles); the R blob
      // and the C tile are adjacent in both buffers, so one linear loop covers both
      constexpr int kChunks = (Cfg::kPkRBytes + Cfg::kCPackedBytes) / 16;
#pragma unroll 4
      for (int ci = w; ci < kChunks; ci += 128) {
        uint32_t v0, v1, v2, v3;
        lds128(pk_addr + ci * 16, v0, v1, v2, v3);
        const uint32_t l0 = (v0 << 4) & 0xF0F0F0F0u, h0 = v0 & 0xF0F0F0F0u;
        const uint32_t l1 = (v1 << 4) & 0xF0F0F0F0u, h1 = v1 & 0xF0F0F0F0u;
        const uint32_t l2 = (v2 << 4) & 0xF0F0F0F0u, h2 = v2 & 0xF0F0F0F0u;
        const uint32_t l3 = (v3 << 4) & 0xF0F0F0F0u, h3 = v3 & 0xF0F0F0F0u;
        const uint32_t dst = i8_addr + ci * 32;
        if (flip) {   // warp-divergence free in effect: both sides are two 128-bit stores
          sts128(dst + 16, h0, h1, h2, h3);
          sts128(dst, l0, l1, l2, l3);
        } else {
          sts128(dst, l0, l1, l2, l3);
          sts128(dst + 16, h0, h1, h2, h3);
        }
      }
      fence_proxy_async_smem();
      mbar_arrive(bar(bI8Full + t));
      // scales of the groups that start in this k-block: FP16 -> FP32 (row scale carries the 2^-8)
      const bool has_scales = (kbpg == 1) || (it % kbpg == 0);
      if (has_scales) {
        const __half* sRh = reinterpret_cast<const __half*>(pk + Cfg::kPkRBytes + Cfg::kCPackedBytes);
        const __half* sCh = sRh + Cfg::kPkScaleRBytes / 2;
        for (int sub = 0; sub < gpk; ++sub, ++grp) {
          const int q = grp % Cfg::kScfSlots;
          mbar_wait(bar(bScfEmpty + q), ((grp / Cfg::kScfSlots) & 1) ^ 1);
          float* dstf = reinterpret_cast<float*>(smem_gen + offScf + q * Cfg::kScfSlotBytes);
          dstf[w] = __half2float(sRh[sub * kTileRows + w]) * 0.00390625f;
          for (int col = w; col < NC; col += 128) {
            float v;
            if (NC >= kTileRows) v = __half2float(sCh[((col >> 7) * gpk + sub) * kTileRows + (col & 127)]);
            else v = __half2float(sCh[sub * kTileRows + (c_row0 % kTileRows) + col]);
            dstf[kTileRows + col] = v;
          }
          mbar_arrive(bar(bScfFull + q));
        }
      }
      mbar_arrive(bar(bPkEmpty + s));
    }
  }
  // =========================================================================== epilogue
  else {
    if constexpr (Cfg::kRebalance) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(Cfg::kRegsEpi));
    constexpr int CPT = Cfg::kCPT;
    constexpr int CW = CPT >= 32 ? 32 : 16;             // columns per tcgen05.ld
    const int ch = (warp - 8) >> 2;                     // column half
    const int lq = warp & 3;                            // TMEM lane quarter this warp may access
    const int row = lq * 32 + lane;
    const int epi_tid = threadIdx.x - 256;
    const uint32_t lane_addr = static_cast<uint32_t>(lq * 32) << 16;
    uint64_t acc[CPT / 2];
#pragma unroll
    for (int i = 0; i < CPT / 2; ++i) acc[i] = 0ull;

    // (m, n) of this thread's row / first column
    const int r_glob = rt * kTileRows + row;
    const int c_glob0 = c_row0 + ch * CPT;

    for (int gi = 0; gi < ngroups; ++gi) {
      const int buf = gi & 1;
      const int q = gi % Cfg::kScfSlots;
      mbar_wait(bar(bScfFull + q), (gi / Cfg::kScfSlots) & 1);
      const float* scf = reinterpret_cast<const float*>(smem_gen + offScf + q * Cfg::kScfSlotBytes);
      const float sRv = scf[row];
      const uint64_t sR2 = pack_f2(sRv, sRv);
      const float* sCf = scf + kTileRows + ch * CPT;
      mbar_wait(bar(bAccFull + buf), (gi >> 1) & 1);
      tc_fence_after();
      const uint32_t tbase = tmem_base + lane_addr + buf * Cfg::kTmemColsPerBuf + ch * CPT;
#pragma unroll
      for (int chunk = 0; chunk < CPT / CW; ++chunk) {
        uint32_t v[CW];
        if constexpr (CW == 32) tmem_ld_32x32(tbase + chunk * CW, v);
        else tmem_ld_32x16(tbase + chunk * CW, v);
        tmem_ld_wait();
        if (chunk == CPT / CW - 1) {   // accumulator buffer fully read: hand it back to the MMA warp
          tc_fence_before();
          mbar_arrive(bar(bAccEmpty + buf));
        }
        if constexpr (DUMP) {
          const int gamma = (g < kBlockK ? kb0 * gpk : kb0 / kbpg) + gi;
#pragma unroll
          for (int j = 0; j < CW; ++j) {
            const int cg = c_glob0 + chunk * CW + j;
            const int m = p.swap ? cg : r_glob;
            const int n = p.swap ? r_glob : cg;
            if (m >= p.pm0 && m < p.pm1 && n >= p.pn0 && n < p.pn1)
              p.P_out[(static_cast<size_t>(m - p.pm0) * (p.pn1 - p.pn0) + (n - p.pn0)) * p.G + gamma] =
                  static_cast<int32_t>(v[j]) >> 8;
          }
        }
#pragma unroll
        for (int j = 0; j < CW; j += 4) {
          const float4 sc = *reinterpret_cast<const float4*>(sCf + chunk * CW + j);
          const uint64_t t0 = mul2(pack_f2(i2f(v[j]), i2f(v[j + 1])), pack_f2(sc.x, sc.y));
          const uint64_t t1 = mul2(pack_f2(i2f(v[j + 2]), i2f(v[j + 3])), pack_f2(sc.z, sc.w));
          acc[(chunk * CW + j) / 2] = fma2(t0, sR2, acc[(chunk * CW + j) / 2]);
          acc[(chunk * CW + j) / 2 + 1] = fma2(t1, sR2, acc[(chunk * CW + j) / 2 + 1]);
        }
      }
      mbar_arrive(bar(bScfEmpty + q));
    }

    // ---- a7 (cast + store) or a6 (split-K reduce)
    if (p.Y != nullptr) {
      const int Rlim = p.R, Clim = p.C;
      if (p.splits == 1) {
        if (!p.swap) {
          if (r_glob < Rlim) {
            if (p.out_f32) {
              float* y = static_cast<float*>(p.Y) + static_cast<size_t>(r_glob) * p.ldY + c_glob0;
#pragma unroll
              for (int j = 0; j < CPT; j += 4) {
                if (c_glob0 + j < Clim) {
                  float4 o;
                  unpack_f2(acc[j / 2], o.x, o.y);
                  unpack_f2(acc[j / 2 + 1], o.z, o.w);
                  *reinterpret_cast<float4*>(y + j) = o;
                }
              }
            } else {
              __half* y = static_cast<__half*>(p.Y) + static_cast<size_t>(r_glob) * p.ldY + c_glob0;
#pragma unroll
              for (int j = 0; j < CPT; j += 8) {
                if (c_glob0 + j < Clim) {
                  float f[8];
#pragma unroll
                  for (int e = 0; e < 4; ++e) unpack_f2(acc[j / 2 + e], f[2 * e], f[2 * e + 1]);
                  uint4 o;
                  __half2 h0 = __floats2half2_rn(f[0], f[1]), h1 = __floats2half2_rn(f[2], f[3]);
                  __half2 h2 = __floats2half2_rn(f[4], f[5]), h3 = __floats2half2_rn(f[6], f[7]);
                  o.x = *reinterpret_cast<uint32_t*>(&h0); o.y = *reinterpret_cast<uint32_t*>(&h1);
                  o.z = *reinterpret_cast<uint32_t*>(&h2); o.w = *reinterpret_cast<uint32_t*>(&h3);
                  *reinterpret_cast<uint4*>(y + j) = o;
                }
              }
            }
          }
        } else {   // swapped: Y[m = column, n = row]; lanes run along n -> coalesced
#pragma unroll
          for (int j = 0; j < CPT; j += 2) {
            float f0, f1;
            unpack_f2(acc[j / 2], f0, f1);
            const int m0 = c_glob0 + j;
            if (r_glob < Rlim) {
              if (p.out_f32) {
                float* y = static_cast<float*>(p.Y);
                if (m0 < Clim) y[static_cast<size_t>(m0) * p.ldY + r_glob] = f0;
                if (m0 + 1 < Clim) y[static_cast<size_t>(m0 + 1) * p.ldY + r_glob] = f1;
              } else {
                __half* y = static_cast<__half*>(p.Y);
                if (m0 < Clim) y[static_cast<size_t>(m0) * p.ldY + r_glob] = __float2half_rn(f0);
                if (m0 + 1 < Clim) y[static_cast<size_t>(m0 + 1) * p.ldY + r_glob] = __float2half_rn(f1);
              }
            }
          }
        }
      } else {
        // a6: FP32 partial sums meet in the workspace (red.add at L2); the last CTA of the tile
        // casts, stores and leaves the workspace zero-filled again ("inter-SM global
        // reduction").
#pragma unroll
        for (int j = 0; j < CPT; j += 2) {
          float f0, f1;
          unpack_f2(acc[j / 2], f0, f1);
          const int cg = c_glob0 + j;
          if (r_glob < Rlim) {
            if (cg < Clim)
              atomicAdd(p.ws + (p.swap ? static_cast<size_t>(cg) * p.ldY + r_glob
                                       : static_cast<size_t>(r_glob) * p.ldY + cg), f0);
            if (cg + 1 < Clim)
              atomicAdd(p.ws + (p.swap ? static_cast<size_t>(cg + 1) * p.ldY + r_glob
                                       : static_cast<size_t>(r_glob) * p.ldY + cg + 1), f1);
          }
        }
        __threadfence();
        int* flag = reinterpret_cast<int*>(smem_gen + offTmemPtr + 8);
        asm volatile("bar.sync 1, %0;" ::"n"(128 * Cfg::kColHalves) : "memory");
        if (epi_tid == 0) {
          const int tile = blockIdx.y * gridDim.x + blockIdx.x;
          const int prev = atomicAdd(p.counters + tile, 1);
          *flag = (prev == p.splits - 1);
          if (prev == p.splits - 1) p.counters[tile] = 0;
        }
        asm volatile("bar.sync 1, %0;" ::"n"(128 * Cfg::kColHalves) : "memory");
        if (*flag) {
          __threadfence();
#pragma unroll
          for (int j = 0; j < CPT; ++j) {
            const int cg = c_glob0 + j;
            if (r_glob < Rlim && cg < Clim) {
              const size_t idx = p.swap ? static_cast<size_t>(cg) * p.ldY + r_glob
                                        : static_cast<size_t>(r_glob) * p.ldY + cg;
              const float vsum = __ldcg(p.ws + idx);
              __stcg(p.ws + idx, 0.f);
              if (p.out_f32) static_cast<float*>(p.Y)[idx] = vsum;
              else static_cast<__half*>(p.Y)[idx] = __float2half_rn(vsum);
            }
          }
        }
      }
    }
    tc_fence_before();
  }

  // ---- teardown
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc<Cfg::kTmemCols>(tmem_base);
  }
}

// ------------------------------------------------------------------------------------ launcher
template <int NC, bool DUMP>
static cudaError_t launch_one(const GemmParams& p, cudaStream_t st) {
  using Cfg = GemmCfg<NC>;
  auto kern = w4a4_gemm_kernel<NC, DUMP>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::kSmemBytes);
  if (e != cudaSuccess) return e;
  dim3 grid((p.C + NC - 1) / NC, (p.R + kTileRows - 1) / kTileRows, p.splits);
  kern<<<grid, Cfg::kThreads, Cfg::kSmemBytes, st>>>(p);
  return cudaGetLastError();
}

cudaError_t launch_gemm(const GemmParams& p, int nc, bool dump, cudaStream_t st) {
  switch (nc) {
    case 16: return dump ? launch_one<16, true>(p, st) : launch_one<16, false>(p, st);
    case 32: return dump ? launch_one<32, true>(p, st) : launch_one<32, false>(p, st);
    case 64: return dump ? launch_one<64, true>(p, st) : launch_one<64, false>(p, st);
    case 128: return dump ? launch_one<128, true>(p, st) : launch_one<128, false>(p, st);
    case 256: return dump ? launch_one<256, true>(p, st) : launch_one<256, false>(p, st);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace apex4
