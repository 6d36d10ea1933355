// apex4_gemm_pair.cu -- a2..a7 of the hot path for the tensor-bound regime (M > 128): the W4A4
// group-dequant GEMM of Eq. 8 on a CTA PAIR (cluster of 2, tcgen05 cta_group::2).
//
// A pair owns a 256 (weight rows n) x 256 (tokens m) output tile.  CTA r of the pair holds weight
// rows 128 r .. 128 r + 127 of the tile on its 128 TMEM lanes and supplies one half of the token
// rows of every MMA from its own shared memory, so per SM and k-block (K = 128) only 8 KB of packed
// weights and 8 KB of packed activations are fetched, widened and read by the tensor core: half the
// L2 traffic, half the activation widening and half the shared-memory operand reads of a lone CTA
// (shared-memory read bandwidth is the scarce resource, profiles/r1_ubench_b200.md).
//
// Roles (512 threads per CTA):
//   warp 0      producer : 1-D bulk async copies (UBLKCP) of this CTA's packed INT4 rows + FP16 scales
//   warp 1      MMA      : leader CTA only; tcgen05.mma cta_group::2 kind::i8, M = 256, N = 128, K = 32,
//                          A (weights) from TMEM, B (tokens) from shared memory, three half-tile
//                          accumulator buffers of 128 columns; tcgen05.commit multicast to both CTAs
//   warps 4-7   wideners : INT4 -> INT8 (x16).  Thread r widens weight row r in registers and stores it
//                          to TMEM; 128 token rows are widened smem -> smem into the 128B-swizzled
//                          UMMA layout.  One elected arrive per warp on the LEADER's operand barrier.
//                          Also FP16 -> FP32 scale preparation.
//   warps 8-15  epilogue : warpgroup h owns the tokens of half h.  tcgen05.ld in the 16x256b shape
//                          (thread = 4 rows x 4 columns of a 16-column chunk, so one LDS.128 fetches
//                          the four token scales a chunk needs instead of sixteen), chunk c+1 is
//                          loaded while chunk c is in the FMA pipe and the buffer goes back to the
//                          MMA warp before the last chunk's arithmetic.  Two FFMA2 per element pair:
//                          fma(f, sW/256, -49152 sW) = P sW rounded once (magic-biased accumulators,
//                          see apex4_gemm.cu), then fma with sA into the FP32 running sums.
#include <cooperative_groups.h>

#include "apex4_gemm.cuh"
#include "apex4_layout.cuh"
#include "apex4_ptx.cuh"

namespace apex4 {

namespace pair {

constexpr uint32_t kMagicBits = 0x4B400000u;   // float 12582912 = 1.5 * 2^23
constexpr int kThreads = 512;
constexpr int kNT = 256;            // tokens per pair tile
constexpr int kNB = 128;            // tokens per half = MMA N = accumulator buffer width
constexpr int kAccBufs = 3;
constexpr int kOpStages = 4;        // widened operand stages (TMEM A + smem B)
constexpr int kPkStages = 5;        // packed (bulk copy) stages
constexpr int kScfSlots = 8;
constexpr int kTmemA0 = 384;        // first TMEM column of the A-operand stages
constexpr int kPkWBytes = kBlobBytes;             // 128 weight rows of a k-block
constexpr int kPkABytes = 2 * 64 * kRowBytes;     // 64 token rows of each half
constexpr int kPkSWBytes = 4 * 256;               // up to 4 groups per k-block, 128 FP16 each
constexpr int kPkSABytes = 2 * 4 * 256;           // two 128-token blobs
constexpr int kPkStageBytes = kPkWBytes + kPkABytes + kPkSWBytes + kPkSABytes;
constexpr int kI8StageBytes = 128 * kBlockK;      // widened tokens: [half][64 rows][128 B]
constexpr int kScfSlotBytes = kTileRows * 8 + kNT * 4;
constexpr int kRegsCtl = 32, kRegsWiden = 64, kRegsEpi = 208;
constexpr int kNumBars = 2 * kPkStages + 2 * kOpStages + 2 * kScfSlots + 2 * kAccBufs;
constexpr int kSmemBytes = 1024 + kOpStages * kI8StageBytes + kPkStages * kPkStageBytes +
                           kScfSlots * kScfSlotBytes + kNumBars * 8 + 64;
static_assert(kAccBufs * kNB <= kTmemA0 && kTmemA0 + 32 * kOpStages <= 512, "TMEM columns");
static_assert(kSmemBytes <= 232448, "shared memory");
static_assert(128 * kRegsCtl + 128 * kRegsWiden + 256 * kRegsEpi <= 65536, "registers");

struct Work {
  int nt, mt;      // pair tile: 256 weight rows, 256 tokens
  int kb0, kb1;
  int partial, units;
};
struct WorkIter {
  long long u, u1;
  int i;
};
__device__ __forceinline__ void work_begin(const GemmParams& p, WorkIter& it, int cp, int npairs) {
  it.i = 0;
  const long long total = static_cast<long long>(p.tiles_m) * p.tiles_n * p.upt;
  it.u = total * cp / npairs;
  it.u1 = total * (cp + 1) / npairs;
}
__device__ __forceinline__ bool work_next(const GemmParams& p, WorkIter& it, Work& w, int cp, int npairs) {
  int tile;
  if (p.split == 0) {
    tile = cp + it.i * npairs;
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

}  // namespace pair

using namespace pair;

template <bool BIAS, bool DUMP>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads, 1)
    w4a4_gemm_pair_kernel(const GemmParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));

  constexpr uint32_t offI8 = 0;
  constexpr uint32_t offPk = offI8 + kOpStages * kI8StageBytes;
  constexpr uint32_t offScf = offPk + kPkStages * kPkStageBytes;
  constexpr uint32_t offBar = offScf + kScfSlots * kScfSlotBytes;
  constexpr uint32_t offTmemPtr = offBar + kNumBars * 8;
  auto bar = [&](int i) { return smem_base + offBar + 8u * i; };
  constexpr int bPkFull = 0, bPkEmpty = bPkFull + kPkStages, bOpFull = bPkEmpty + kPkStages,
                bOpEmpty = bOpFull + kOpStages, bScfFull = bOpEmpty + kOpStages,
                bScfEmpty = bScfFull + kScfSlots, bAccFull = bScfEmpty + kScfSlots,
                bAccEmpty = bAccFull + kAccBufs;

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();      // 0 = leader
  const int cp = blockIdx.x >> 1;               // pair index
  const int npairs = gridDim.x >> 1;
  const int g = p.g;
  const int gpk = g < kBlockK ? kBlockK / g : 1;        // groups per k-block (1, 2, 4)
  const int kbpg = g > kBlockK ? g / kBlockK : 1;       // k-blocks per group

  if (threadIdx.x == 0) {
    for (int i = 0; i < kPkStages; ++i) { mbar_init(bar(bPkFull + i), 1); mbar_init(bar(bPkEmpty + i), 128); }
    // operand stage full: one elected arrive per widener warp of BOTH CTAs, on the leader's barrier
    for (int i = 0; i < kOpStages; ++i) { mbar_init(bar(bOpFull + i), 8); mbar_init(bar(bOpEmpty + i), 1); }
    for (int i = 0; i < kScfSlots; ++i) { mbar_init(bar(bScfFull + i), 128); mbar_init(bar(bScfEmpty + i), 8); }
    // accumulator buffer empty: one elected arrive per epilogue warp of the owning warpgroup, both CTAs
    for (int i = 0; i < kAccBufs; ++i) { mbar_init(bar(bAccFull + i), 1); mbar_init(bar(bAccEmpty + i), 8); }
    fence_mbar_init();
  }
  if (warp == 1) tmem_alloc_pair<512>(smem_base + offTmemPtr);
  tc_fence_before();
  cluster_sync_all();       // barriers of both CTAs initialised before any remote arrive / multicast
  tc_fence_after();
  const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(smem_gen + offTmemPtr);

  WorkIter wit;
  Work w;
  work_begin(p, wit, cp, npairs);

  // =========================================================================== producer
  if (warp < 4) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsCtl));
    if (warp == 0 && lane == 0) {
      const int n_blobs = round_up(p.N, kTileRows) / kTileRows;
      const int m_blobs = round_up(p.M, kTileRows) / kTileRows;
      const uint32_t sc_bytes = gpk * 256;
      uint32_t kbc = 0;
      while (work_next(p, wit, w, cp, npairs)) {
        const int wblob = 2 * w.nt + static_cast<int>(rank);
        const bool has_w = wblob < n_blobs;
        const int a_blobs = min(2, m_blobs - 2 * w.mt);      // 128-token blobs of this tile
        for (int kb = w.kb0; kb < w.kb1; ++kb, ++kbc) {
          const int s = kbc % kPkStages;
          mbar_wait(bar(bPkEmpty + s), ((kbc / kPkStages) & 1) ^ 1);
          const uint32_t st = smem_base + offPk + s * kPkStageBytes;
          const bool has_scales = (kb % kbpg) == 0;
          const int gfirst = g < kBlockK ? kb * gpk : kb / kbpg;
          uint32_t bytes = (has_w ? kBlobBytes : 0) + a_blobs * 64 * kRowBytes;
          if (has_scales) bytes += sc_bytes * ((has_w ? 1 : 0) + a_blobs);
          mbar_arrive_expect_tx(bar(bPkFull + s), bytes);
          if (has_w) bulk_g2s(st, p.qW + pt4_blob_offset(wblob, kb, p.K), kBlobBytes, bar(bPkFull + s));
          for (int h = 0; h < a_blobs; ++h)   // half h of the tile = blob 2 mt + h; this CTA's 64 rows
            bulk_g2s(st + kPkWBytes + h * 64 * kRowBytes,
                     p.qA + pt4_blob_offset(2 * w.mt + h, kb, p.K) + rank * 64 * kRowBytes,
                     64 * kRowBytes, bar(bPkFull + s));
          if (has_scales) {
            if (has_w)
              bulk_g2s(st + kPkWBytes + kPkABytes,
                       p.sW + (static_cast<size_t>(wblob) * p.G + gfirst) * kTileRows, sc_bytes,
                       bar(bPkFull + s));
            for (int h = 0; h < a_blobs; ++h)
              bulk_g2s(st + kPkWBytes + kPkABytes + kPkSWBytes + h * sc_bytes,
                       p.sA + (static_cast<size_t>(2 * w.mt + h) * p.G + gfirst) * kTileRows, sc_bytes,
                       bar(bPkFull + s));
          }
        }
      }
    }
    // ========================================================================= MMA issuer (leader)
    else if (warp == 1 && lane == 0 && rank == 0) {
      constexpr uint32_t idesc = umma_idesc_i8(256, kNB);
      uint32_t kbc = 0, gc = 0;
      const int ks_per_sub = 4 / gpk;
      while (work_next(p, wit, w, cp, npairs)) {
        for (int kb = w.kb0; kb < w.kb1; ++kb, ++kbc) {
          const int t = kbc % kOpStages;
          mbar_wait_cluster(bar(bOpFull + t), (kbc / kOpStages) & 1);
          tc_fence_after();
          const uint32_t a_tm = tmem_base + kTmemA0 + 32 * t;
          const uint32_t b_sm = smem_base + offI8 + t * kI8StageBytes;
          const bool first = (kb % kbpg) == 0;
          const bool last = (kb % kbpg) == kbpg - 1;
          for (int sub = 0; sub < gpk; ++sub) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              const uint32_t u = (gc + sub) * 2 + h;
              const uint32_t buf = u % kAccBufs;
              if (first) {
                mbar_wait_cluster(bar(bAccEmpty + buf), (u / kAccBufs) & 1);
                tc_fence_after();
              }
              const uint32_t d = tmem_base + buf * kNB;
              const uint64_t bdesc = umma_desc_sw128(b_sm + h * (64 * kBlockK));
              for (int ks = 0; ks < ks_per_sub; ++ks) {
                const uint32_t kq = sub * ks_per_sub + ks;     // K=32 slice of the k-block
                const uint32_t accum = BIAS ? 1u : ((first && ks == 0) ? 0u : 1u);
                mma_i8_ts_pair(d, a_tm + 8 * kq, bdesc + 2 * kq, idesc, accum);
              }
              if (last) tc_commit_pair(bar(bAccFull + buf), 3);
            }
          }
          tc_commit_pair(bar(bOpEmpty + t), 3);
          if (last) gc += gpk;
        }
      }
    }
  }
  // =========================================================================== wideners
  else if (warp < 8) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsWiden));
    const int r = threadIdx.x - 128;                    // weight row of this CTA's blob = TMEM lane
    const uint32_t lane_addr = static_cast<uint32_t>((warp & 3) * 32) << 16;
    const uint32_t wsw = (r >> 1) & 3;                  // chunk-slot swizzle of the packed row (PW4)
    const uint32_t flip = ((lane >> 2) & 1) * 16;       // see apex4_gemm.cu: bank spread of the two stores
    constexpr uint32_t kMask = 0xF0F0F0F0u;
    uint32_t kbc = 0, gc = 0;
    int pend_t = -1;                                    // operand stage written but not yet published
    // Publishing stage t (fences + one elected arrive on the leader's barrier) is deferred until the
    // loads of the next k-block are in flight, so the TMEM / shared-memory store drain overlaps them.
    auto publish = [&](int t) {
      fence_proxy_async_smem();
      tmem_st_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(bar(bOpFull + t), 0);
    };
    while (work_next(p, wit, w, cp, npairs)) {
      for (int kb = w.kb0; kb < w.kb1; ++kb, ++kbc) {
        const int s = kbc % kPkStages;
        const int t = kbc % kOpStages;
        mbar_wait(bar(bPkFull + s), (kbc / kPkStages) & 1);
        const uint32_t pk_addr = smem_base + offPk + s * kPkStageBytes;
        uint32_t wv[16];
#pragma unroll
        for (int j = 0; j < 4; ++j)
          lds128(pk_addr + r * kRowBytes + ((j ^ wsw) << 4), wv[4 * j], wv[4 * j + 1], wv[4 * j + 2], wv[4 * j + 3]);
        if (pend_t >= 0) publish(pend_t);
        mbar_wait(bar(bOpEmpty + t), ((kbc / kOpStages) & 1) ^ 1);
        tc_fence_after();
        // ---- weights: packed row r (64 bytes) -> 32 INT8 words -> TMEM columns of stage t
        {
          uint32_t o[32];
#pragma unroll
          for (int j = 0; j < 4; ++j) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              o[8 * j + i] = rotl4(wv[4 * j + i]) & kMask;
              o[8 * j + 4 + i] = wv[4 * j + i] & kMask;
            }
          }
          tmem_st_32x32(tmem_base + lane_addr + kTmemA0 + 32 * t, o);
        }
        // ---- tokens: packed byte offset o -> INT8 byte offsets 2o (lo nibbles), 2o+16 (hi)
        {
          uint32_t av[16];
#pragma unroll
          for (int x = 0; x < 4; ++x)
            lds128(pk_addr + kPkWBytes + (r + 128 * x) * 16, av[4 * x], av[4 * x + 1], av[4 * x + 2], av[4 * x + 3]);
          const uint32_t dst0 = smem_base + offI8 + t * kI8StageBytes;
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            const uint32_t dst = dst0 + (r + 128 * x) * 32;
            const uint32_t l0 = rotl4(av[4 * x]) & kMask, h0 = av[4 * x] & kMask;
            const uint32_t l1 = rotl4(av[4 * x + 1]) & kMask, h1 = av[4 * x + 1] & kMask;
            const uint32_t l2 = rotl4(av[4 * x + 2]) & kMask, h2 = av[4 * x + 2] & kMask;
            const uint32_t l3 = rotl4(av[4 * x + 3]) & kMask, h3 = av[4 * x + 3] & kMask;
            if (flip) {
              sts128(dst + 16, h0, h1, h2, h3);
              sts128(dst, l0, l1, l2, l3);
            } else {
              sts128(dst, l0, l1, l2, l3);
              sts128(dst + 16, h0, h1, h2, h3);
            }
          }
        }
        pend_t = t;
        // ---- scales of the groups that start in this k-block: FP16 -> FP32
        if ((kb % kbpg) == 0) {
          const uint8_t* pk = smem_gen + offPk + s * kPkStageBytes;
          const __half* sWh = reinterpret_cast<const __half*>(pk + kPkWBytes + kPkABytes);
          const __half* sAh = sWh + kPkSWBytes / 2;
          for (int sub = 0; sub < gpk; ++sub, ++gc) {
            const int q = gc % kScfSlots;
            mbar_wait(bar(bScfEmpty + q), ((gc / kScfSlots) & 1) ^ 1);
            float* dstf = reinterpret_cast<float*>(smem_gen + offScf + q * kScfSlotBytes);
            const float sw = __half2float(sWh[sub * kTileRows + r]);
            // a = sW / 256 (the operands are 16 q each); b = -12582912 * a removes the magic bias
            reinterpret_cast<float2*>(dstf)[r] = make_float2(sw * 0.00390625f, sw * -49152.0f);
            // token scales, permuted inside every 16-column chunk so that the four columns
            // {2t, 2t+1, 8+2t, 9+2t} an epilogue thread owns are one 16-byte vector: c -> 4t + 2j + e
#pragma unroll
            for (int x = 0; x < 2; ++x) {
              const int col = r + 128 * x;                       // token of the tile
              const int c = col & 15;
              const int pos = (col & ~15) | (((c >> 1) & 3) << 2) | ((c >> 3) << 1) | (c & 1);
              dstf[2 * kTileRows + pos] = __half2float(sAh[(x * gpk + sub) * kTileRows + r]);
            }
            mbar_arrive(bar(bScfFull + q));
          }
        }
        mbar_arrive(bar(bPkEmpty + s));
      }
    }
    if (pend_t >= 0) publish(pend_t);
  }
  // =========================================================================== epilogue
  else {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegsEpi));
    const int h = (warp - 8) >> 2;                      // warpgroup = token half
    const int lq = warp & 3;                            // TMEM lane quarter this warp may access
    const int q = lane >> 2, t = lane & 3;
    const int epi_tid = threadIdx.x - 256;
    const uint32_t lane_addr = static_cast<uint32_t>(lq * 32) << 16;
    const int row0 = lq * 32 + q;                       // rows row0 + 8 i, i = 0..3

    // completion #0 of every accEmpty barrier: buffer b is first used by unit u = b, half b & 1
#pragma unroll
    for (int b = 0; b < kAccBufs; ++b) {
      if ((b & 1) != h) continue;
      if (BIAS) {
#pragma unroll
        for (int c = 0; c < kNB; c += 16) tmem_fill_32x16(tmem_base + lane_addr + b * kNB + c, kMagicBits);
        tmem_st_wait();
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(bar(bAccEmpty + b), 0);
    }

    uint32_t gc = 0;
    while (work_next(p, wit, w, cp, npairs)) {
      const int nkb = w.kb1 - w.kb0;
      const int ngroups = g < kBlockK ? nkb * gpk : nkb / kbpg;
      uint64_t acc[64];                                 // [i][c][j] -> (i * 8 + c) * 2 + j
#pragma unroll
      for (int i = 0; i < 64; ++i) acc[i] = 0ull;
      const int n_glob0 = (2 * w.nt + static_cast<int>(rank)) * kTileRows + row0;
      const int m_glob0 = w.mt * kNT + h * kNB + 2 * t;   // + 16 c + 8 j + e

      for (int gi = 0; gi < ngroups; ++gi, ++gc) {
        const int slot = gc % kScfSlots;
        const uint32_t u = gc * 2 + h;
        const uint32_t buf = u % kAccBufs;
        mbar_wait(bar(bScfFull + slot), (gc / kScfSlots) & 1);
        const uint32_t scf = smem_base + offScf + slot * kScfSlotBytes;
        uint64_t a2[4], b2[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          float af, bf;
          unpack_f2(lds64(scf + (row0 + 8 * i) * 8), af, bf);
          a2[i] = pack_f2(af, af);
          b2[i] = pack_f2(bf, bf);
        }
        const uint32_t sAf = scf + 2 * kTileRows * 4 + (h * kNB) * 4 + t * 16;   // + 64 c
        mbar_wait(bar(bAccFull + buf), (u / kAccBufs) & 1);
        tc_fence_after();
        const uint32_t tb = tmem_base + lane_addr + buf * kNB;
        uint32_t v[2][16];
        tmem_ld_16x256b_x2(tb, v[0]);
        tmem_ld_16x256b_x2(tb + (16u << 16), v[0] + 8);
#pragma unroll
        for (int c = 0; c < 8; ++c) {
          uint32_t* vc = v[c & 1];
          tmem_ld_wait16(vc);
          if constexpr (BIAS) tmem_fill_32x16(tb + 16 * c, kMagicBits);   // re-arm the chunk just read
          if (c < 7) {
            tmem_ld_16x256b_x2(tb + 16 * (c + 1), v[(c + 1) & 1]);
            tmem_ld_16x256b_x2(tb + (16u << 16) + 16 * (c + 1), v[(c + 1) & 1] + 8);
          } else {                                       // buffer fully read (and re-armed): hand it back
            if constexpr (BIAS) tmem_st_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(bar(bAccEmpty + buf), 0);
          }
          if constexpr (DUMP) {
            const int gamma = (g < kBlockK ? w.kb0 * gpk : w.kb0 / kbpg) + gi;
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
              for (int j = 0; j < 2; ++j)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                  const int m = m_glob0 + 16 * c + 8 * j + e;
                  const int n = n_glob0 + 8 * i;
                  if (m >= p.pm0 && m < p.pm1 && n >= p.pn0 && n < p.pn1) {
                    const uint32_t x = vc[8 * (i >> 1) + 4 * j + 2 * (i & 1) + e];
                    const int32_t raw = static_cast<int32_t>(BIAS ? x - kMagicBits : x);
                    p.P_out[(static_cast<size_t>(m - p.pm0) * (p.pn1 - p.pn0) + (n - p.pn0)) * p.G + gamma] = raw >> 8;
                  }
                }
          }
          uint64_t s01, s23;
          lds_2x64(sAf + 64 * c, s01, s23);              // token scales of columns {2t,2t+1}, {8+2t,9+2t}
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int rb = 8 * (i >> 1) + 2 * (i & 1);
            uint64_t t0, t1;
            if constexpr (BIAS) {
              t0 = fma2(pack_u2(vc[rb], vc[rb + 1]), a2[i], b2[i]);
              t1 = fma2(pack_u2(vc[rb + 4], vc[rb + 5]), a2[i], b2[i]);
            } else {
              t0 = mul2(pack_f2(__int2float_rn(static_cast<int>(vc[rb])), __int2float_rn(static_cast<int>(vc[rb + 1]))), a2[i]);
              t1 = mul2(pack_f2(__int2float_rn(static_cast<int>(vc[rb + 4])), __int2float_rn(static_cast<int>(vc[rb + 5]))), a2[i]);
            }
            acc[(i * 8 + c) * 2] = fma2(t0, s01, acc[(i * 8 + c) * 2]);
            acc[(i * 8 + c) * 2 + 1] = fma2(t1, s23, acc[(i * 8 + c) * 2 + 1]);
          }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(bScfEmpty + slot));
      }

      // ---- a7 (cast + store) or a6 (cross-pair reduce through the FP32 workspace)
      if (p.Y != nullptr) {
        if (!w.partial) {
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int n = n_glob0 + 8 * i;
            if (n >= p.N) continue;
#pragma unroll
            for (int c = 0; c < 8; ++c)
#pragma unroll
              for (int j = 0; j < 2; ++j) {
                float f0, f1;
                unpack_f2(acc[(i * 8 + c) * 2 + j], f0, f1);
                const int m = m_glob0 + 16 * c + 8 * j;
                if (p.out_f32) {
                  float* y = static_cast<float*>(p.Y);
                  if (m < p.M) y[static_cast<size_t>(m) * p.N + n] = f0;
                  if (m + 1 < p.M) y[static_cast<size_t>(m + 1) * p.N + n] = f1;
                } else {
                  __half* y = static_cast<__half*>(p.Y);
                  if (m < p.M) y[static_cast<size_t>(m) * p.N + n] = __float2half_rn(f0);
                  if (m + 1 < p.M) y[static_cast<size_t>(m + 1) * p.N + n] = __float2half_rn(f1);
                }
              }
          }
        } else {
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int n = n_glob0 + 8 * i;
            if (n >= p.N) continue;
#pragma unroll
            for (int c = 0; c < 8; ++c)
#pragma unroll
              for (int j = 0; j < 2; ++j) {
                float f0, f1;
                unpack_f2(acc[(i * 8 + c) * 2 + j], f0, f1);
                const int m = m_glob0 + 16 * c + 8 * j;
                if (m < p.M) atomicAdd(p.ws + static_cast<size_t>(m) * p.N + n, f0);
                if (m + 1 < p.M) atomicAdd(p.ws + static_cast<size_t>(m + 1) * p.N + n, f1);
              }
          }
          __threadfence();
          int* flag = reinterpret_cast<int*>(smem_gen + offTmemPtr + 8);
          asm volatile("bar.sync 1, 256;" ::: "memory");
          if (epi_tid == 0) {
            const int tile = (w.nt * p.tiles_m + w.mt) * 2 + static_cast<int>(rank);
            const int prev = atomicAdd(p.counters + tile, w.units);
            const int done = (prev + w.units == p.upt);
            *flag = done;
            if (done) p.counters[tile] = 0;
          }
          asm volatile("bar.sync 1, 256;" ::: "memory");
          const int done = *flag;
          asm volatile("bar.sync 1, 256;" ::: "memory");   // flag may be rewritten by the next item
          if (done) {
            __threadfence();
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const int n = n_glob0 + 8 * i;
              if (n >= p.N) continue;
#pragma unroll 4
              for (int cj = 0; cj < 16; ++cj)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                  const int m = m_glob0 + 8 * cj + e;
                  if (m < p.M) {
                    const size_t idx = static_cast<size_t>(m) * p.N + n;
                    const float vsum = __ldcg(p.ws + idx);
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
    tc_fence_before();
  }

  // ---- teardown: nobody leaves while the peer may still signal this CTA's barriers or read its
  // shared memory / TMEM through the pair MMA
  cluster_sync_all();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc_pair<512>(tmem_base);
  }
}

// ------------------------------------------------------------------------------------ launcher
template <bool BIAS, bool DUMP>
static cudaError_t launch_pair_one(const GemmParams& p, int npairs, cudaStream_t st) {
  auto kern = w4a4_gemm_pair_kernel<BIAS, DUMP>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
  if (e != cudaSuccess) return e;
  kern<<<2 * npairs, kThreads, kSmemBytes, st>>>(p);
  return cudaGetLastError();
}

cudaError_t launch_gemm_pair(const GemmParams& p, bool bias, bool dump, int npairs, cudaStream_t st) {
  if (bias) return dump ? launch_pair_one<true, true>(p, npairs, st) : launch_pair_one<true, false>(p, npairs, st);
  return dump ? launch_pair_one<false, true>(p, npairs, st) : launch_pair_one<false, false>(p, npairs, st);
}

// CTA pairs that can be resident at once (one per TPC); queried once
int gemm_max_pairs() {
  static int pairs = 0;
  if (pairs == 0) {
    auto kern = w4a4_gemm_pair_kernel<true, false>;
    int n = 0;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(2 * 74);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = kSmemBytes;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes) != cudaSuccess ||
        cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess || n <= 0) {
      cudaGetLastError();
      n = gemm_max_ctas() / 2;
    }
    pairs = n;
  }
  return pairs;
}

}  // namespace apex4
