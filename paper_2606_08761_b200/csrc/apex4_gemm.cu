// apex4_gemm.cu -- a2..a7 of the hot path: the W4A4 group-dequant GEMM of Eq. 8
// for sm_100a.  Persistent kernel, one CTA per SM, 512 threads, warp-specialised:
//
//   warp 0       producer : 1-D bulk async copies (TMA engine, UBLKCP) of the packed INT4 blobs of
//                           both operands + FP16 scales into a shared-memory ring
//   warp 1       MMA      : one thread issues tcgen05.mma kind::i8 (K = 32 per instruction), A operand
//                           from TMEM, B operand from shared memory, into one of three TMEM
//                           accumulator buffers; tcgen05.commit hands stages / accumulators on
//   warps 4-7    wideners : INT4 -> INT8 (x16, sign kept).  Thread r widens weight row r in registers
//                           and stores it to TMEM (tcgen05.st) -- the widened weights never touch
//                           shared memory; the activation rows are widened smem -> smem straight into
//                           the 128B-swizzled UMMA layout.  Also FP16 -> FP32 scale preparation.
//   warps 8-15   epilogue : tcgen05.ld a finished group's tile, two FFMA2 per element pair
//                           (P*sW exactly rounded, then FMA with sA into the FP32 running sums kept in
//                           registers) while the tensor core works on the next groups (the overlap
//                           the paper says Ampere cannot do); cast + store at the end.
//
// Orientation: TMEM lanes = 128 weight rows n, accumulator columns = NT token rows m.
//
// Integer exactness: operands are 16*q, the accumulator holds 256*P_g (|256 P_g| <= 2^21 for
// g <= 128, < 2^31 for any K <= 32768).  INT32 -> FP32 without a conversion instruction (I2F runs
// at 63/clk/SM on B200, as slow as the whole MMA of a g=128 group): for g <= 128 every accumulator
// buffer is pre-loaded with 0x4B400000 by tcgen05.st, every MMA accumulates, so the TMEM word read
// back IS the float 12582912 + 256 P (exact), and fma(f, sW/256, -49152 sW) = P * sW rounded once.
#include "apex4_gemm.cuh"
#include "apex4_layout.cuh"
#include "apex4_ptx.cuh"

namespace apex4 {

constexpr uint32_t kMagicBits = 0x4B400000u;   // float 12582912 = 1.5 * 2^23
constexpr int kAccBufs = 3;
constexpr int kScfSlots = 8;
constexpr int kTmemA0 = 384;                   // first TMEM column of the A-operand stages
constexpr int kThreads = 512;

template <int NT>
struct GemmCfg {
  static constexpr int kHalves = NT == 256 ? 2 : 1;            // accumulator buffers per group
  static constexpr int NB = NT / kHalves;                      // MMA N = accumulator buffer width
  static constexpr int kEpiWGs = NT >= 128 ? 2 : 1;            // working epilogue warpgroups
  static constexpr int CPT = NT == 256 ? 128 : (NT == 128 ? 64 : NT);   // columns per epilogue thread
  static constexpr int kWGsPerUse = kHalves == 2 ? 1 : kEpiWGs;
  static constexpr int kOpStages = NT == 256 ? 3 : 4;          // widened-operand stages (TMEM A + smem B)
  static constexpr int kPkStages = NT == 256 ? 4 : NT == 128 ? 6 : NT == 64 ? 10 : 12;
  static constexpr int kATiles = (NT + 127) / 128;             // 128-row activation blobs per tile
  static constexpr int kPkWBytes = kBlobBytes;                 // packed weights of a k-block
  static constexpr int kPkABytes = NT * kRowBytes;             // packed activations of a k-block
  static constexpr int kPkSWBytes = 4 * 256;                   // up to 4 groups per k-block
  static constexpr int kPkSABytes = 4 * 256 * kATiles;
  static constexpr int kPkStageBytes = kPkWBytes + kPkABytes + kPkSWBytes + kPkSABytes;
  static constexpr int kI8StageBytes = NT * kBlockK;           // widened activations of a k-block
  static constexpr int kScfSlotBytes = kTileRows * 8 + NT * 4; // {sW/256, -49152 sW} per row + sA per column
  static constexpr int kRegsCtl = 40, kRegsWiden = 72, kRegsEpi = 200;
  static constexpr int kNumBars = 2 * kPkStages + 2 * kOpStages + 2 * kScfSlots + 2 * kAccBufs;
  static constexpr int kSmemBytes = 1024 /*align slack*/ + kOpStages * kI8StageBytes +
                                    kPkStages * kPkStageBytes + kScfSlots * kScfSlotBytes +
                                    kNumBars * 8 + 64;
  static_assert(kAccBufs * NB <= kTmemA0 && kTmemA0 + 32 * kOpStages <= 512, "TMEM columns");
  static_assert(kSmemBytes <= 232448, "shared memory");
};

// ------------------------------------------------------------------------------------ scheduling
struct Work {
  int nt, mt;      // weight-row tile, token tile
  int kb0, kb1;    // k-block range
  int partial;     // the range is not the whole K loop: reduce through the workspace
  int units;
};
struct WorkIter {
  long long u, u1;   // split = 1: unit range of this CTA
  int i;             // split = 0: iteration
};
__device__ __forceinline__ void work_begin(const GemmParams& p, WorkIter& it) {
  it.i = 0;
  const long long total = static_cast<long long>(p.tiles_m) * p.tiles_n * p.upt;
  it.u = total * blockIdx.x / gridDim.x;
  it.u1 = total * (blockIdx.x + 1) / gridDim.x;
}
// Tiles are numbered token-tile fastest: CTAs that run together share weight tiles in L2, and a
// weight matrix larger than L2 is still streamed from HBM once.
__device__ __forceinline__ bool work_next(const GemmParams& p, WorkIter& it, Work& w) {
  int tile;
  if (p.split == 0) {
    tile = blockIdx.x + it.i * gridDim.x;
    if (tile >= p.tiles_m * p.tiles_n) return false;
    ++it.i;
    w.kb0 = 0; w.kb1 = p.K / kBlockK; w.partial = 0; w.units = p.upt;
  } else {
    if (it.u >= it.u1) return false;
    tile = static_cast<int>(it.u / p.upt);
    const int off = static_cast<int>(it.u - static_cast<long long>(tile) * p.upt);
    const long long left = it.u1 - it.u;
    const int n = static_cast<int>(left < p.upt - off ? left : p.upt - off);
    w.kb0 = off * p.kbu; w.kb1 = (off + n) * p.kbu; w.partial = (n != p.upt); w.units = n;
    it.u += n;
  }
  w.mt = tile % p.tiles_m;
  w.nt = tile / p.tiles_m;
  return true;
}

__device__ __forceinline__ float i2f(uint32_t v) { return __int2float_rn(static_cast<int>(v)); }

template <int NT, bool BIAS, bool DUMP>
__global__ void __launch_bounds__(kThreads, 1) w4a4_gemm_kernel(const GemmParams p) {
  using Cfg = GemmCfg<NT>;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));

  // ---- carve-up (offsets from the 1024-aligned base)
  constexpr uint32_t offI8 = 0;
  constexpr uint32_t offPk = offI8 + Cfg::kOpStages * Cfg::kI8StageBytes;
  constexpr uint32_t offScf = offPk + Cfg::kPkStages * Cfg::kPkStageBytes;
  constexpr uint32_t offBar = offScf + kScfSlots * Cfg::kScfSlotBytes;
  constexpr uint32_t offTmemPtr = offBar + Cfg::kNumBars * 8;
  auto bar = [&](int i) { return smem_base + offBar + 8u * i; };
  constexpr int bPkFull = 0, bPkEmpty = bPkFull + Cfg::kPkStages, bOpFull = bPkEmpty + Cfg::kPkStages,
                bOpEmpty = bOpFull + Cfg::kOpStages, bScfFull = bOpEmpty + Cfg::kOpStages,
                bScfEmpty = bScfFull + kScfSlots, bAccFull = bScfEmpty + kScfSlots,
                bAccEmpty = bAccFull + kAccBufs;

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const int g = p.g;
  const int gpk = g < kBlockK ? kBlockK / g : 1;        // groups per k-block (1, 2, 4)
  const int kbpg = g > kBlockK ? g / kBlockK : 1;       // k-blocks per group
  const int KB = p.K / kBlockK;

  if (threadIdx.x == 0) {
    for (int i = 0; i < Cfg::kPkStages; ++i) { mbar_init(bar(bPkFull + i), 1); mbar_init(bar(bPkEmpty + i), 128); }
    for (int i = 0; i < Cfg::kOpStages; ++i) { mbar_init(bar(bOpFull + i), 128); mbar_init(bar(bOpEmpty + i), 1); }
    for (int i = 0; i < kScfSlots; ++i) { mbar_init(bar(bScfFull + i), 128); mbar_init(bar(bScfEmpty + i), 128 * Cfg::kEpiWGs); }
    for (int i = 0; i < kAccBufs; ++i) { mbar_init(bar(bAccFull + i), 1); mbar_init(bar(bAccEmpty + i), 128 * Cfg::kWGsPerUse); }
    fence_mbar_init();
  }
  if (warp == 1) tmem_alloc<512>(smem_base + offTmemPtr);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(smem_gen + offTmemPtr);

  WorkIter wit;
  Work w;
  work_begin(p, wit);

  // =========================================================================== producer
  if (warp < 4) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(Cfg::kRegsCtl));
    if (warp == 0 && lane == 0) {
      const int Mp = round_up(p.M, kTileRows);
      const uint32_t sc_bytes = gpk * 256;
      uint32_t kbc = 0;
      while (work_next(p, wit, w)) {
        const int a_row0 = w.mt * NT;
        const int a_rows = min(NT, Mp - a_row0);          // valid packed token rows of this tile
        const int a_tiles = (a_rows + kTileRows - 1) / kTileRows;
        for (int kb = w.kb0; kb < w.kb1; ++kb, ++kbc) {
          const int s = kbc % Cfg::kPkStages;
          mbar_wait(bar(bPkEmpty + s), ((kbc / Cfg::kPkStages) & 1) ^ 1);
          const uint32_t st = smem_base + offPk + s * Cfg::kPkStageBytes;
          const bool has_scales = (kb % kbpg) == 0;
          const int gfirst = g < kBlockK ? kb * gpk : kb / kbpg;
          uint32_t bytes = kBlobBytes + a_rows * kRowBytes;
          if (has_scales) bytes += sc_bytes * (1 + a_tiles);
          mbar_arrive_expect_tx(bar(bPkFull + s), bytes);
          bulk_g2s(st, p.qW + pt4_blob_offset(w.nt, kb, p.K), kBlobBytes, bar(bPkFull + s));
          for (int b = 0; b < a_tiles; ++b) {
            const int rows_b = min(kTileRows, a_rows - b * kTileRows);
            // NT < 128: the tile is rows a_row0 % 128 ... of its blob (NT divides 128)
            bulk_g2s(st + Cfg::kPkWBytes + b * kBlobBytes,
                     p.qA + pt4_blob_offset(a_row0 / kTileRows + b, kb, p.K) +
                         (a_row0 % kTileRows) * kRowBytes,
                     rows_b * kRowBytes, bar(bPkFull + s));
          }
          if (has_scales) {
            bulk_g2s(st + Cfg::kPkWBytes + Cfg::kPkABytes,
                     p.sW + (static_cast<size_t>(w.nt) * p.G + gfirst) * kTileRows, sc_bytes,
                     bar(bPkFull + s));
            for (int b = 0; b < a_tiles; ++b)
              bulk_g2s(st + Cfg::kPkWBytes + Cfg::kPkABytes + Cfg::kPkSWBytes + b * sc_bytes,
                       p.sA + (static_cast<size_t>(a_row0 / kTileRows + b) * p.G + gfirst) * kTileRows,
                       sc_bytes, bar(bPkFull + s));
          }
        }
      }
    }
    // ========================================================================= MMA issuer
    else if (warp == 1 && lane == 0) {
      constexpr uint32_t idesc = umma_idesc_i8(kTileRows, Cfg::NB);
      uint32_t kbc = 0, gc = 0;
      const int ks_per_sub = 4 / gpk;
      while (work_next(p, wit, w)) {
        for (int kb = w.kb0; kb < w.kb1; ++kb, ++kbc) {
          const int t = kbc % Cfg::kOpStages;
          mbar_wait(bar(bOpFull + t), (kbc / Cfg::kOpStages) & 1);
          tc_fence_after();
          const uint32_t a_tm = tmem_base + kTmemA0 + 32 * t;
          const uint32_t b_sm = smem_base + offI8 + t * Cfg::kI8StageBytes;
          const bool first = (kb % kbpg) == 0;
          const bool last = (kb % kbpg) == kbpg - 1;
          for (int sub = 0; sub < gpk; ++sub) {
#pragma unroll
            for (int h = 0; h < Cfg::kHalves; ++h) {
              const uint32_t u = (gc + sub) * Cfg::kHalves + h;
              const uint32_t buf = u % kAccBufs;
              if (first) {
                mbar_wait(bar(bAccEmpty + buf), (u / kAccBufs) & 1);
                tc_fence_after();
              }
              const uint32_t d = tmem_base + buf * Cfg::NB;
              const uint64_t bdesc = umma_desc_sw128(b_sm + h * (Cfg::NB * kBlockK));
              for (int ks = 0; ks < ks_per_sub; ++ks) {
                const uint32_t kq = sub * ks_per_sub + ks;     // K=32 slice of the k-block
                const uint32_t accum = BIAS ? 1u : ((first && ks == 0) ? 0u : 1u);
                mma_i8_ts(d, a_tm + 8 * kq, bdesc + 2 * kq, idesc, accum);
              }
              if (last) tc_commit(bar(bAccFull + buf));
            }
          }
          tc_commit(bar(bOpEmpty + t));
          if (last) gc += gpk;
        }
      }
    }
  }
  // =========================================================================== wideners
  else if (warp < 8) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(Cfg::kRegsWiden));
    const int r = threadIdx.x - 128;                    // weight row of the tile = TMEM lane
    const uint32_t lane_addr = static_cast<uint32_t>((warp & 3) * 32) << 16;
    const uint32_t wsw = (r >> 1) & 3;                  // chunk-slot swizzle of the packed row (PW4)
    // a lane whose (lane>>2)&1 is set stores its hi chunk first: the two 16-byte stores of a quarter
    // warp then cover all 32 banks (32-byte stride would otherwise hit each bank twice)
    const uint32_t flip = ((lane >> 2) & 1) * 16;
    uint32_t kbc = 0, gc = 0;
    while (work_next(p, wit, w)) {
      for (int kb = w.kb0; kb < w.kb1; ++kb, ++kbc) {
        const int s = kbc % Cfg::kPkStages;
        const int t = kbc % Cfg::kOpStages;
        mbar_wait(bar(bPkFull + s), (kbc / Cfg::kPkStages) & 1);
        mbar_wait(bar(bOpEmpty + t), ((kbc / Cfg::kOpStages) & 1) ^ 1);
        tc_fence_after();
        const uint8_t* pk = smem_gen + offPk + s * Cfg::kPkStageBytes;
        const uint32_t pk_addr = smem_base + offPk + s * Cfg::kPkStageBytes;
        // ---- weights: packed row r (64 bytes) -> 32 INT8 words -> TMEM columns of stage t
        {
          uint32_t o[32];
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            uint32_t v0, v1, v2, v3;
            lds128(pk_addr + r * kRowBytes + ((j ^ wsw) << 4), v0, v1, v2, v3);
            o[8 * j + 0] = (v0 << 4) & 0xF0F0F0F0u; o[8 * j + 4] = v0 & 0xF0F0F0F0u;
            o[8 * j + 1] = (v1 << 4) & 0xF0F0F0F0u; o[8 * j + 5] = v1 & 0xF0F0F0F0u;
            o[8 * j + 2] = (v2 << 4) & 0xF0F0F0F0u; o[8 * j + 6] = v2 & 0xF0F0F0F0u;
            o[8 * j + 3] = (v3 << 4) & 0xF0F0F0F0u; o[8 * j + 7] = v3 & 0xF0F0F0F0u;
          }
          tmem_st_32x32(tmem_base + lane_addr + kTmemA0 + 32 * t, o);
        }
        // ---- activations: packed byte offset o -> INT8 byte offsets 2o (lo nibbles), 2o+16 (hi)
        {
          const uint32_t src = pk_addr + Cfg::kPkWBytes;
          const uint32_t dst0 = smem_base + offI8 + t * Cfg::kI8StageBytes;
          constexpr int kChunks = Cfg::kPkABytes / 16;
#pragma unroll
          for (int ci0 = 0; ci0 < kChunks; ci0 += 128) {
            const int ci = ci0 + r;
            if (kChunks % 128 == 0 || ci < kChunks) {
              uint32_t v0, v1, v2, v3;
              lds128(src + ci * 16, v0, v1, v2, v3);
              const uint32_t l0 = (v0 << 4) & 0xF0F0F0F0u, h0 = v0 & 0xF0F0F0F0u;
              const uint32_t l1 = (v1 << 4) & 0xF0F0F0F0u, h1 = v1 & 0xF0F0F0F0u;
              const uint32_t l2 = (v2 << 4) & 0xF0F0F0F0u, h2 = v2 & 0xF0F0F0F0u;
              const uint32_t l3 = (v3 << 4) & 0xF0F0F0F0u, h3 = v3 & 0xF0F0F0F0u;
              const uint32_t dst = dst0 + ci * 32;
              if (flip) {   // both sides are two 128-bit stores
                sts128(dst + 16, h0, h1, h2, h3);
                sts128(dst, l0, l1, l2, l3);
              } else {
                sts128(dst, l0, l1, l2, l3);
                sts128(dst + 16, h0, h1, h2, h3);
              }
            }
          }
        }
        fence_proxy_async_smem();
        tmem_st_wait();
        tc_fence_before();
        mbar_arrive(bar(bOpFull + t));
        // ---- scales of the groups that start in this k-block: FP16 -> FP32
        if ((kb % kbpg) == 0) {
          const __half* sWh = reinterpret_cast<const __half*>(pk + Cfg::kPkWBytes + Cfg::kPkABytes);
          const __half* sAh = sWh + Cfg::kPkSWBytes / 2 + (w.mt * NT) % kTileRows;
          for (int sub = 0; sub < gpk; ++sub, ++gc) {
            const int q = gc % kScfSlots;
            mbar_wait(bar(bScfEmpty + q), ((gc / kScfSlots) & 1) ^ 1);
            float* dstf = reinterpret_cast<float*>(smem_gen + offScf + q * Cfg::kScfSlotBytes);
            const float sw = __half2float(sWh[sub * kTileRows + r]);
            // a = sW / 256 (the operands are 16 q each); b = -12582912 * a removes the magic bias
            reinterpret_cast<float2*>(dstf)[r] = make_float2(sw * 0.00390625f, sw * -49152.0f);
#pragma unroll
            for (int col0 = 0; col0 < NT; col0 += 128) {
              const int col = col0 + r;
              if (NT % 128 == 0 || col < NT)
                dstf[2 * kTileRows + col] = __half2float(sAh[((col >> 7) * gpk + sub) * kTileRows + (col & 127)]);
            }
            mbar_arrive(bar(bScfFull + q));
          }
        }
        mbar_arrive(bar(bPkEmpty + s));
      }
    }
  }
  // =========================================================================== epilogue
  else {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(Cfg::kRegsEpi));
    constexpr int CPT = Cfg::CPT;
    constexpr int CW = CPT >= 32 ? 32 : 16;             // columns per tcgen05.ld
    const int wg = (warp - 8) >> 2;                     // epilogue warpgroup
    const int lq = warp & 3;                            // TMEM lane quarter this warp may access
    const int row = lq * 32 + lane;
    const int epi_tid = threadIdx.x - 256;
    const uint32_t lane_addr = static_cast<uint32_t>(lq * 32) << 16;
    const bool active = wg < Cfg::kEpiWGs;
    // columns of an accumulator buffer this thread reads, and the tokens they are
    const int col0 = Cfg::kHalves == 2 ? 0 : wg * CPT;
    const int tok0 = Cfg::kHalves == 2 ? wg * Cfg::NB : wg * CPT;

    if (active) {
      // completion #0 of every accEmpty barrier: the buffers start out holding the magic bias
#pragma unroll
      for (int b = 0; b < kAccBufs; ++b) {
        if (Cfg::kHalves == 2 && (b & 1) != wg) continue;
        if (BIAS) {
#pragma unroll
          for (int c = 0; c < CPT; c += 16) tmem_fill_32x16(tmem_base + lane_addr + b * Cfg::NB + col0 + c, kMagicBits);
          tmem_st_wait();
        }
        tc_fence_before();
        mbar_arrive(bar(bAccEmpty + b));
      }

      uint32_t gc = 0;
      while (work_next(p, wit, w)) {
        const int nkb = w.kb1 - w.kb0;
        const int ngroups = g < kBlockK ? nkb * gpk : nkb / kbpg;
        uint64_t acc[CPT / 2];
#pragma unroll
        for (int i = 0; i < CPT / 2; ++i) acc[i] = 0ull;
        const int n_glob = w.nt * kTileRows + row;
        const int m_glob0 = w.mt * NT + tok0;

        for (int gi = 0; gi < ngroups; ++gi, ++gc) {
          const int q = gc % kScfSlots;
          const uint32_t u = gc * Cfg::kHalves + (Cfg::kHalves == 2 ? wg : 0);
          const uint32_t buf = u % kAccBufs;
          mbar_wait(bar(bScfFull + q), (gc / kScfSlots) & 1);
          const uint32_t scf = smem_base + offScf + q * Cfg::kScfSlotBytes;
          const uint64_t ab = lds64(scf + row * 8);
          float af, bf;
          unpack_f2(ab, af, bf);
          const uint64_t a2 = pack_f2(af, af), b2 = pack_f2(bf, bf);
          const uint32_t sAf = scf + 2 * kTileRows * 4 + tok0 * 4;
          mbar_wait(bar(bAccFull + buf), (u / kAccBufs) & 1);
          tc_fence_after();
          const uint32_t tbase = tmem_base + lane_addr + buf * Cfg::NB + col0;
#pragma unroll
          for (int chunk = 0; chunk < CPT / CW; ++chunk) {
            uint32_t v[CW];
            if constexpr (CW == 32) tmem_ld_32x32(tbase + chunk * CW, v);
            else tmem_ld_32x16(tbase + chunk * CW, v);
            tmem_ld_wait();
            if constexpr (BIAS) {   // re-arm the columns just read for the buffer's next group
#pragma unroll
              for (int c = 0; c < CW; c += 16) tmem_fill_32x16(tbase + chunk * CW + c, kMagicBits);
            }
            if (chunk == CPT / CW - 1) {   // buffer fully read (and re-armed): hand it back
              if constexpr (BIAS) tmem_st_wait();
              tc_fence_before();
              mbar_arrive(bar(bAccEmpty + buf));
            }
            if constexpr (DUMP) {
              const int gamma = (g < kBlockK ? w.kb0 * gpk : w.kb0 / kbpg) + gi;
#pragma unroll
              for (int j = 0; j < CW; ++j) {
                const int m = m_glob0 + chunk * CW + j;
                if (m >= p.pm0 && m < p.pm1 && n_glob >= p.pn0 && n_glob < p.pn1) {
                  const int32_t raw = static_cast<int32_t>(BIAS ? v[j] - kMagicBits : v[j]);
                  p.P_out[(static_cast<size_t>(m - p.pm0) * (p.pn1 - p.pn0) + (n_glob - p.pn0)) * p.G + gamma] = raw >> 8;
                }
              }
            }
#pragma unroll
            for (int j = 0; j < CW; j += 4) {
              uint64_t s01, s23;
              lds_2x64(sAf + (chunk * CW + j) * 4, s01, s23);
              uint64_t t0, t1;
              if constexpr (BIAS) {
                t0 = fma2(pack_u2(v[j], v[j + 1]), a2, b2);
                t1 = fma2(pack_u2(v[j + 2], v[j + 3]), a2, b2);
              } else {
                t0 = mul2(pack_f2(i2f(v[j]), i2f(v[j + 1])), a2);
                t1 = mul2(pack_f2(i2f(v[j + 2]), i2f(v[j + 3])), a2);
              }
              acc[(chunk * CW + j) / 2] = fma2(t0, s01, acc[(chunk * CW + j) / 2]);
              acc[(chunk * CW + j) / 2 + 1] = fma2(t1, s23, acc[(chunk * CW + j) / 2 + 1]);
            }
          }
          mbar_arrive(bar(bScfEmpty + q));
        }

        // ---- a7 (cast + store) or a6 (cross-CTA reduce).  Lanes run along n: coalesced in Y[m, n].
        if (p.Y != nullptr) {
          if (!w.partial) {
            if (n_glob < p.N) {
#pragma unroll
              for (int j = 0; j < CPT; j += 2) {
                float f0, f1;
                unpack_f2(acc[j / 2], f0, f1);
                const int m0 = m_glob0 + j;
                if (p.out_f32) {
                  float* y = static_cast<float*>(p.Y);
                  if (m0 < p.M) y[static_cast<size_t>(m0) * p.N + n_glob] = f0;
                  if (m0 + 1 < p.M) y[static_cast<size_t>(m0 + 1) * p.N + n_glob] = f1;
                } else {
                  __half* y = static_cast<__half*>(p.Y);
                  if (m0 < p.M) y[static_cast<size_t>(m0) * p.N + n_glob] = __float2half_rn(f0);
                  if (m0 + 1 < p.M) y[static_cast<size_t>(m0 + 1) * p.N + n_glob] = __float2half_rn(f1);
                }
              }
            }
          } else {
            // a6: FP32 partial sums meet in the workspace (red.add at L2); the CTA that completes the
            // tile casts, stores and leaves the workspace zero-filled again ("inter-SM
            // global reduction").
            if (n_glob < p.N) {
#pragma unroll
              for (int j = 0; j < CPT; j += 2) {
                float f0, f1;
                unpack_f2(acc[j / 2], f0, f1);
                const int m0 = m_glob0 + j;
                if (m0 < p.M) atomicAdd(p.ws + static_cast<size_t>(m0) * p.N + n_glob, f0);
                if (m0 + 1 < p.M) atomicAdd(p.ws + static_cast<size_t>(m0 + 1) * p.N + n_glob, f1);
              }
            }
            __threadfence();
            int* flag = reinterpret_cast<int*>(smem_gen + offTmemPtr + 8);
            asm volatile("bar.sync 1, %0;" ::"n"(128 * Cfg::kEpiWGs) : "memory");
            if (epi_tid == 0) {
              const int tile = w.nt * p.tiles_m + w.mt;
              const int prev = atomicAdd(p.counters + tile, w.units);
              const int done = (prev + w.units == p.upt);
              *flag = done;
              if (done) p.counters[tile] = 0;
            }
            asm volatile("bar.sync 1, %0;" ::"n"(128 * Cfg::kEpiWGs) : "memory");
            const int done = *flag;
            asm volatile("bar.sync 1, %0;" ::"n"(128 * Cfg::kEpiWGs) : "memory");   // flag may be rewritten next item
            if (done) {
              __threadfence();
              if (n_glob < p.N) {
#pragma unroll
                for (int j = 0; j < CPT; j += 2) {       // all loads first, then the stores
                  const int m = m_glob0 + j;
                  float f0 = 0.f, f1 = 0.f;
                  if (m < p.M) f0 = __ldcg(p.ws + static_cast<size_t>(m) * p.N + n_glob);
                  if (m + 1 < p.M) f1 = __ldcg(p.ws + static_cast<size_t>(m + 1) * p.N + n_glob);
                  acc[j / 2] = pack_f2(f0, f1);
                }
#pragma unroll
                for (int j = 0; j < CPT; ++j) {
                  const int m = m_glob0 + j;
                  if (m < p.M) {
                    const size_t idx = static_cast<size_t>(m) * p.N + n_glob;
                    float f0, f1;
                    unpack_f2(acc[j / 2], f0, f1);
                    const float vsum = (j & 1) ? f1 : f0;
                    __stcg(p.ws + idx, 0.f);
                    if (p.out_f32) static_cast<float*>(p.Y)[idx] = vsum;
                    else static_cast<__half*>(p.Y)[idx] = __float2half_rn(vsum);
                  }
                }
              }
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
    tmem_dealloc<512>(tmem_base);
  }
}

// ------------------------------------------------------------------------------------ launcher
template <int NT, bool BIAS, bool DUMP>
static cudaError_t launch_one(const GemmParams& p, int grid, cudaStream_t st) {
  using Cfg = GemmCfg<NT>;
  auto kern = w4a4_gemm_kernel<NT, BIAS, DUMP>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::kSmemBytes);
  if (e != cudaSuccess) return e;
  kern<<<grid, kThreads, Cfg::kSmemBytes, st>>>(p);
  return cudaGetLastError();
}

template <int NT>
static cudaError_t launch_nt(const GemmParams& p, bool bias, bool dump, int grid, cudaStream_t st) {
  if (bias) return dump ? launch_one<NT, true, true>(p, grid, st) : launch_one<NT, true, false>(p, grid, st);
  return dump ? launch_one<NT, false, true>(p, grid, st) : launch_one<NT, false, false>(p, grid, st);
}

cudaError_t launch_gemm(const GemmParams& p, int nt, bool bias, bool dump, int grid, cudaStream_t st) {
  switch (nt) {
    case 16: return launch_nt<16>(p, bias, dump, grid, st);
    case 32: return launch_nt<32>(p, bias, dump, grid, st);
    case 64: return launch_nt<64>(p, bias, dump, grid, st);
    case 128: return launch_nt<128>(p, bias, dump, grid, st);
    default: return cudaErrorInvalidValue;
  }
}

int gemm_max_ctas() {
  static int sms = 0;
  if (sms == 0) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0)
      sms = 148;
  }
  return sms;
}

}  // namespace apex4
