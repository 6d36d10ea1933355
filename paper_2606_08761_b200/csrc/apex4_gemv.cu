// apex4_gemv.cu -- a2..a7 of the hot path for the decode regime (M <= 32; g = 32 / 64 / 128 or per-channel):
// the weights are read once from HBM and every byte is used M times, so the kernel is a weight STREAM:
// warp-private bulk-copy stages in shared memory, no TMEM, no cross-CTA exchange, no workspace.
//
//   * A CTA (16 warps) owns a contiguous range of 8-row weight groups ("row blocks"), processed in
//     batches of RBB row blocks, and ALL of K.  Warp w owns the k-blocks [KB w / 16, KB (w+1) / 16).
//   * Operand staging is warp-private: for each of its k-blocks the warp's elected lane issues 1-D bulk
//     async copies (cp.async.bulk, TMA engine) of the batch's weight rows (RBB x 512 contiguous bytes of
//     the PW4 blob), the token rows, and both scale vectors into one of the warp's two shared-memory
//     stages, completion counted on an mbarrier.  16 warps x 2 stages x ~4.7 KB = 150 KB per SM are in
//     flight with no register cost (a register ring held only 57 KB and cost one HBM round trip per 7
//     units and warp: 15 us; profiles/r1_gemv_ncu.md).  No cross-warp hand-off: the warp that issued a
//     stage is the one that consumes it and re-arms it.
//   * Consumption: lane (q, t) reads the 16-byte packed chunk that holds K slice t of row q (one
//     conflict-free LDS.128 per row block), widens the four words with two logic ops each (16 x code,
//     apex4_layout.cuh) and feeds them to four mma.sync.m16n8k32.s8 (tokens = m16, 8 weight rows = n8).
//     MMA i takes word i of every lane: its 32 k are {32 t + 4 i + e, 32 t + 16 + 4 i + e}; any k order
//     inside a group gives the same exact INT32 sum and the token fragments (widened once per k-block,
//     reused by every row block) use the very same lane -> k assignment.
//   * Each k-block's INT32 sum is converted, multiplied by sW/256 (operands are 16 q) and sA and added
//     to the warp's FP32 partial sums (registers, one set per row block of the batch); once per batch
//     the partials of the 16 warps are reduced through shared memory, cast and stored (a6, a7).
// Tensor cores here are the legacy warp-level path on purpose: at M <= 64 the MMA work is < 2 % of the
// HBM time and a tcgen05 pipeline (bulk copy -> widen -> TMEM -> MMA -> TMEM load) only adds latency
// (round 1, first tcgen05 tile kernel: 48 us at M = 16 against 5.3 us of HBM time).
#include <type_traits>

#include "apex4_gemm.cuh"
#include "apex4_layout.cuh"
#include "apex4_ptx.cuh"

namespace apex4 {

namespace gemv {

constexpr int kWarps = 16;
constexpr int kThreads = 32 * kWarps;
constexpr uint32_t kMask = 0xF0F0F0F0u;
constexpr int kStages = 2;                              // warp-private operand stages

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

}  // namespace gemv

using namespace gemv;


// MT: m16 token tiles (M <= 16 MT).  p.tiles_n = 8-row row blocks; p.kbu = k-blocks per group.
// GS: groups per k-block (1: g >= 128; 2: g = 64; 4: g = 32)
template <int MT, int GS = 1>
struct GemvCfg {
  static constexpr int RBB = MT == 1 ? 7 : MT == 2 ? 4 : MT == 3 ? 2 : 1;         // row blocks per batch
  static constexpr int kWBytes = RBB * 8 * kRowBytes;                // weight rows of a k-block
  static constexpr int kABytes = MT * 16 * kRowBytes;                // token rows of a k-block
  static constexpr int kSWBytes = RBB * 16 * GS;                     // FP16 weight scales of the batch rows, [group][row]
  static constexpr int kSABytes = MT * 32 * GS;                      // FP16 token scales, [group][token]
  static constexpr int kStageBytes = kWBytes + kABytes + kSWBytes + kSABytes;
  static constexpr int kPartBytes = RBB * kWarps * MT * 512;         // FP32 partial sums of a batch
  static constexpr int kSmemBytes = 128 + kPartBytes + kWarps * kStages * kStageBytes + kWarps * kStages * 8;
  static_assert(kStageBytes % 16 == 0 && kSmemBytes <= 232448, "shared memory");
};

// GM (group mode): 0 = a group is a k-block or a part of one (g <= 128): every k-block is scaled on its own;
// 1 = a group is several k-blocks and a warp's k range is a whole number of groups (g = 256 .. with K / 16 a
//     multiple of g): the INT32 sums of a group stay in registers across its k-blocks and are scaled once;
// 2 = a warp's k range lies inside ONE group (per-channel g = K, or g a multiple of K / 16): see below.
// GM = 2, e.g. per-channel (one group = all of K).  The warps' k ranges are then parts of ONE group, so the
// partial sums stay INT32 through the k loop and through the cross-warp reduction (exact), and the two
// scales are applied once at the end -- one rounding per group as R12 wants, which the per-k-block FP32
// scaling of the g = 128 path cannot give for larger groups.  |256 P| <= 2^8 * 64 * 32768 = 2^29: no overflow.
// GS > 1 (g = 64 / 32): lane (q, t) takes word t of each of the row's four 16-byte chunks instead of chunk t,
// so that MMA c covers exactly k = 32 c .. 32 c + 31 of the k-block, i.e. one g = 32 group (half a g = 64
// group), and every group gets its own scales.
template <int MT, bool DUMP, int GM, int GS>
__global__ void __launch_bounds__(kThreads, 1) w4a4_gemv_kernel(const GemmParams p) {
  static_assert(GM == 0 || GS == 1, "groups of several k-blocks have no sub-k-block groups");
  constexpr bool CH = GM == 2;          // INT32 partial sums meet across warps
  const int kbpg = p.kbu;               // k-blocks per group (GM = 1, 2)
  using Cfg = GemvCfg<MT, GS>;
  constexpr int RBB = Cfg::RBB;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 127u) & ~127u;
  uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
  float4* part = reinterpret_cast<float4*>(smem_gen);                // [row block][warp][MT][lane]
  constexpr uint32_t offStage = Cfg::kPartBytes;
  constexpr uint32_t offBar = offStage + kWarps * kStages * Cfg::kStageBytes;

  // warp index through a shuffle: tells the compiler it is warp-uniform, so the copy descriptors of
  // issue_next live in uniform registers (per-thread operands cost an R2UR waterfall per UBLKCP)
  const int lane = threadIdx.x & 31, w = __shfl_sync(0xffffffffu, static_cast<int>(threadIdx.x >> 5), 0);
  const int q = lane >> 2, t = lane & 3;
  const int KB = p.K / kBlockK;
  const int kbw0 = KB * w / kWarps, kbw1 = KB * (w + 1) / kWarps;    // this warp's k-blocks
  const int nkw = kbw1 - kbw0;
  const int rb0 = static_cast<int>(static_cast<long long>(p.tiles_n) * blockIdx.x / gridDim.x);
  const int rb1 = static_cast<int>(static_cast<long long>(p.tiles_n) * (blockIdx.x + 1) / gridDim.x);
  const size_t row_pitch = static_cast<size_t>(KB) * kBlobBytes;
  const bool swap = (q & 1) != 0;                       // odd token rows: lo / hi nibbles exchanged (PT4)
  // byte offset of this lane's 16-byte chunk (K slice t of row q) inside an 8-row group
  const uint32_t lane_off = q * kRowBytes + ((t ^ ((q >> 1) & 3)) << 4);
  const uint32_t my_stage0 = smem_base + offStage + w * kStages * Cfg::kStageBytes;
  const uint32_t my_bar0 = smem_base + offBar + w * kStages * 8;
  if (lane == 0) {
    for (int s = 0; s < kStages; ++s) mbar_init(my_bar0 + 8 * s, 1);
    fence_mbar_init();
  }
  __syncwarp();

  // ---- issue cursor: (batch start row block, k-block index of this warp), flattened, k fastest.
  // The whole warp runs the bookkeeping on warp-uniform values and one elected lane issues: with the
  // cursor private to lane 0 the divergent block cost the warp ~185 issue slots per k-block (a third
  // of the loop), every copy sitting in an R2UR / BRA.U.ANY waterfall.
  const bool el = elect_one();
  // Source pointers advance by a blob (k-block) per stage and are set up once per batch: recomputing them
  // per stage cost ~120 (uniform-datapath) instructions per k-block.  One group per k-block (g = 128, the
  // only granularity the dispatcher sends here): group index = k-block index.
  int ib0 = rb0, ij = 0, islot = 0, ikin = 0;            // ikin: k-block inside its group (GM = 1)
  const uint8_t *w1 = nullptr, *w2 = nullptr, *aq = nullptr;
  const __half *s1 = nullptr, *s2 = nullptr, *sq = nullptr;
  uint32_t n1b = 0, n2b = 0, tx = 0;                    // rows x 64 bytes of the two pieces, bytes per stage
  auto batch_setup = [&]() {
    const int nb = min(RBB, rb1 - ib0);
    const int row_a = ib0 * 8, row_b = row_a + nb * 8;                 // weight rows of the batch
    const int tile_a = row_a >> 7;
    const int split_row = min(row_b, (tile_a + 1) << 7);               // rows [row_a, split_row) in tile_a
    const int n1 = split_row - row_a, n2 = row_b - split_row;
    w1 = p.qW + tile_a * row_pitch + static_cast<size_t>(kbw0) * kBlobBytes + (row_a & 127) * kRowBytes;
    w2 = p.qW + (tile_a + 1) * row_pitch + static_cast<size_t>(kbw0) * kBlobBytes;
    if constexpr (!CH && !DUMP) {   // the dump of the integer sums takes no scales (null pointers)
      const int g0 = GM == 1 ? kbw0 / kbpg : GS * kbw0;               // first group of this warp's k range
      s1 = p.sW + (static_cast<size_t>(tile_a) * p.G + g0) * kTileRows + (row_a & 127);
      s2 = p.sW + (static_cast<size_t>(tile_a + 1) * p.G + g0) * kTileRows;
      sq = p.sA + static_cast<size_t>(g0) * kTileRows;
    }
    ikin = 0;
    aq = p.qA + static_cast<size_t>(kbw0) * kBlobBytes;
    n1b = n1 * kRowBytes;
    n2b = n2 * kRowBytes;
    tx = (n1 + n2) * kRowBytes + Cfg::kABytes + ((CH || DUMP) ? 0 : GS * (n1 + n2) * 2 + Cfg::kSABytes);
  };
  if (rb0 < rb1 && nkw > 0) batch_setup();
  // The activation side of a stage (packed token rows + token scales): what the PREVIOUS kernel on the stream
  // (the online quantizer) writes.  The weight side is constant, so the first stages' weight copies are issued
  // before griddep_wait() and stream in while the predecessor drains (programmatic dependent launch).
  auto issue_tokens = [&](uint32_t st, uint32_t full, const uint8_t* aq_, const __half* sq_) {
    if (el) {
      bulk_g2s(st + Cfg::kWBytes, aq_, Cfg::kABytes, full);
      if constexpr (!CH && !DUMP) {
#pragma unroll
        for (int gs = 0; gs < GS; ++gs)
          bulk_g2s(st + Cfg::kWBytes + Cfg::kABytes + Cfg::kSWBytes + gs * (MT * 32), sq_ + gs * kTileRows, MT * 32, full);
      }
    }
  };
  const uint8_t* aq_pre[kStages] = {};
  const __half* sq_pre[kStages] = {};
  int n_pre = 0;
  auto issue_next = [&](bool tokens_now) {              // copies of one stage
    if (ib0 >= rb1 || nkw == 0) return;
    const uint32_t st = my_stage0 + islot * Cfg::kStageBytes;
    const uint32_t full = my_bar0 + 8 * islot;
    if (el) {
      mbar_arrive_expect_tx(full, tx);
      bulk_g2s(st, w1, n1b, full);
      if (n2b > 0) bulk_g2s(st + n1b, w2, n2b, full);
      if constexpr (!CH && !DUMP) {
#pragma unroll
        for (int gs = 0; gs < GS; ++gs) {               // 2 bytes per row and group
          const uint32_t dsw = st + Cfg::kWBytes + Cfg::kABytes + gs * (RBB * 16);
          bulk_g2s(dsw, s1 + gs * kTileRows, n1b >> 5, full);
          if (n2b > 0) bulk_g2s(dsw + (n1b >> 5), s2 + gs * kTileRows, n2b >> 5, full);
        }
      }
    }
    if (tokens_now) {
      issue_tokens(st, full, aq, sq);
    } else {                                            // prologue: after griddep_wait()
      aq_pre[n_pre] = aq;
      sq_pre[n_pre] = sq;
      ++n_pre;
    }
    w1 += kBlobBytes; w2 += kBlobBytes; aq += kBlobBytes;
    if constexpr (!CH && !DUMP) {
      // every k-block stage carries the scales of ITS group: the pointers move on at a group boundary
      if (GM == 0 || ++ikin == kbpg) { s1 += GS * kTileRows; s2 += GS * kTileRows; sq += GS * kTileRows; ikin = 0; }
    }
    islot = islot + 1 == kStages ? 0 : islot + 1;
    if (++ij == nkw) {
      ij = 0;
      ib0 += RBB;
      if (ib0 < rb1) batch_setup();
    }
  };
#pragma unroll
  for (int s = 0; s < kStages; ++s) issue_next(false);  // weight side of the first stages
  griddep_launch();                                     // the next kernel on the stream may start its own weight stream
  griddep_wait();                                       // the quantizer's output is complete and visible from here on
#pragma unroll
  for (int s = 0; s < kStages; ++s)
    if (s < n_pre) issue_tokens(my_stage0 + s * Cfg::kStageBytes, my_bar0 + 8 * s, aq_pre[s], sq_pre[s]);

  uint32_t par = 0;                                     // phase parity of the warp's stage barriers
  int cslot = 0;
  for (int b0 = rb0; b0 < rb1; b0 += RBB) {
    const int nb = min(RBB, rb1 - b0);
    float yf[RBB][MT][4];
#pragma unroll
    for (int i = 0; i < RBB; ++i)
#pragma unroll
      for (int mi = 0; mi < MT; ++mi)
#pragma unroll
        for (int e = 0; e < 4; ++e) yf[i][mi][e] = 0.f;
    int ia[RBB][MT][4];                                 // CH: 256 x the INT32 sums over this warp's k range
#pragma unroll
    for (int i = 0; i < RBB; ++i)
#pragma unroll
      for (int mi = 0; mi < MT; ++mi)
#pragma unroll
        for (int e = 0; e < 4; ++e) ia[i][mi][e] = 0;

    for (int j = 0; j < nkw; ++j) {
      const uint32_t st = my_stage0 + cslot * Cfg::kStageBytes;
      mbar_wait(my_bar0 + 8 * cslot, (par >> cslot) & 1);
      par ^= 1u << cslot;
      // ---- token fragments of this k-block (widened once, reused by every row block)
      uint32_t af[MT][4][4];
      float sa[MT][2];
      float sag[GS > 1 ? MT : 1][GS][2];                // GS > 1: token scales per group of the k-block
#pragma unroll
      for (int mi = 0; mi < MT; ++mi) {
        uint32_t x0[4], x1[4];
        if constexpr (GS > 1) {
#pragma unroll
          for (int c = 0; c < 4; ++c) {                 // word t of chunk c (stored at slot c ^ swizzle)
            const uint32_t off = q * kRowBytes + ((c ^ ((q >> 1) & 3)) << 4) + 4 * t;
            x0[c] = lds32(st + Cfg::kWBytes + (16 * mi) * kRowBytes + off);
            x1[c] = lds32(st + Cfg::kWBytes + (16 * mi + 8) * kRowBytes + off);
          }
          const __half* sah = reinterpret_cast<const __half*>(smem_gen + (st - smem_base) + Cfg::kWBytes + Cfg::kABytes + Cfg::kSWBytes);
#pragma unroll
          for (int gs = 0; gs < GS; ++gs) {
            sag[mi][gs][0] = __half2float(sah[gs * (16 * MT) + 16 * mi + q]);
            sag[mi][gs][1] = __half2float(sah[gs * (16 * MT) + 16 * mi + q + 8]);
          }
        } else {
        lds128(st + Cfg::kWBytes + (16 * mi) * kRowBytes + lane_off, x0[0], x0[1], x0[2], x0[3]);
        lds128(st + Cfg::kWBytes + (16 * mi + 8) * kRowBytes + lane_off, x1[0], x1[1], x1[2], x1[3]);
        }
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const uint32_t l0 = rotl4(x0[i]) & kMask, h0 = x0[i] & kMask;
          const uint32_t l1 = rotl4(x1[i]) & kMask, h1 = x1[i] & kMask;
          af[mi][i][0] = swap ? h0 : l0; af[mi][i][2] = swap ? l0 : h0;   // token q: k lo / hi half
          af[mi][i][1] = swap ? h1 : l1; af[mi][i][3] = swap ? l1 : h1;   // token q + 8
        }
        if constexpr (GM != 2 && GS == 1) {
          const __half* sah = reinterpret_cast<const __half*>(smem_gen + (st - smem_base) + Cfg::kWBytes + Cfg::kABytes + Cfg::kSWBytes);
          sa[mi][0] = __half2float(sah[16 * mi + q]);
          sa[mi][1] = __half2float(sah[16 * mi + q + 8]);
        }
      }
      const int gm = DUMP ? (kbw0 + j) / p.kbu : 0;
      const bool group_ends = GM == 1 && ((kbw0 + j + 1) % kbpg) == 0;   // warp ranges start on group boundaries
#pragma unroll
      for (int i = 0; i < RBB; ++i) {
        if (i < nb) {
          uint32_t x[4];
          if constexpr (GS > 1) {
            const uint32_t off = q * kRowBytes + 4 * t;
            const uint32_t swz = (q >> 1) & 3;
#pragma unroll
            for (int c = 0; c < 4; ++c) x[c] = lds32(st + i * 512 + off + ((c ^ swz) << 4));
            constexpr int MPG = 4 / GS;                   // MMAs per group
#pragma unroll
            for (int gs = 0; gs < GS; ++gs) {
              int acc[MT][4];
#pragma unroll
              for (int mi = 0; mi < MT; ++mi)
#pragma unroll
                for (int e = 0; e < 4; ++e) acc[mi][e] = 0;
#pragma unroll
              for (int c = gs * MPG; c < (gs + 1) * MPG; ++c) {
                const uint32_t b0w = rotl4(x[c]) & kMask, b1w = x[c] & kMask;
#pragma unroll
                for (int mi = 0; mi < MT; ++mi) mma_s8(acc[mi], af[mi][c], b0w, b1w);
              }
              const __half2 sw2 = *reinterpret_cast<const __half2*>(smem_gen + (st - smem_base) + Cfg::kWBytes + Cfg::kABytes + gs * (RBB * 16) + i * 16 + 4 * t);
              const float sw0 = __low2float(sw2) * 0.00390625f, sw1 = __high2float(sw2) * 0.00390625f;
#pragma unroll
              for (int mi = 0; mi < MT; ++mi) {
                yf[i][mi][0] = fmaf(__int2float_rn(acc[mi][0]) * sw0, sag[mi][gs][0], yf[i][mi][0]);
                yf[i][mi][1] = fmaf(__int2float_rn(acc[mi][1]) * sw1, sag[mi][gs][0], yf[i][mi][1]);
                yf[i][mi][2] = fmaf(__int2float_rn(acc[mi][2]) * sw0, sag[mi][gs][1], yf[i][mi][2]);
                yf[i][mi][3] = fmaf(__int2float_rn(acc[mi][3]) * sw1, sag[mi][gs][1], yf[i][mi][3]);
                if constexpr (DUMP) {
                  const int gmm = (kbw0 + j) * GS + gs;
#pragma unroll
                  for (int e = 0; e < 4; ++e) {
                    const int m = 16 * mi + q + 8 * (e >> 1), n = (b0 + i) * 8 + 2 * t + (e & 1);
                    if (m >= p.pm0 && m < p.pm1 && n >= p.pn0 && n < p.pn1)
                      atomicAdd(p.P_out + (static_cast<size_t>(m - p.pm0) * (p.pn1 - p.pn0) + (n - p.pn0)) * p.G + gmm,
                                acc[mi][e] >> 8);
                  }
                }
              }
            }
            continue;
          }
          lds128(st + i * 512 + lane_off, x[0], x[1], x[2], x[3]);
          if constexpr (GM != 0) {
#pragma unroll
            for (int k4 = 0; k4 < 4; ++k4) {
              const uint32_t b0w = rotl4(x[k4]) & kMask, b1w = x[k4] & kMask;
#pragma unroll
              for (int mi = 0; mi < MT; ++mi) mma_s8(ia[i][mi], af[mi][k4], b0w, b1w);
            }
            if constexpr (GM == 1) {
              if (group_ends) {     // the group's exact sum: INT32 -> FP32, x sW / 256, x sA, once (a5, R12)
                const __half2 sw2 = *reinterpret_cast<const __half2*>(smem_gen + (st - smem_base) + Cfg::kWBytes + Cfg::kABytes + i * 16 + 4 * t);
                const float sw0 = __low2float(sw2) * 0.00390625f, sw1 = __high2float(sw2) * 0.00390625f;
#pragma unroll
                for (int mi = 0; mi < MT; ++mi) {
                  yf[i][mi][0] = fmaf(__int2float_rn(ia[i][mi][0]) * sw0, sa[mi][0], yf[i][mi][0]);
                  yf[i][mi][1] = fmaf(__int2float_rn(ia[i][mi][1]) * sw1, sa[mi][0], yf[i][mi][1]);
                  yf[i][mi][2] = fmaf(__int2float_rn(ia[i][mi][2]) * sw0, sa[mi][1], yf[i][mi][2]);
                  yf[i][mi][3] = fmaf(__int2float_rn(ia[i][mi][3]) * sw1, sa[mi][1], yf[i][mi][3]);
                  if constexpr (DUMP) {
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                      const int m = 16 * mi + q + 8 * (e >> 1), n = (b0 + i) * 8 + 2 * t + (e & 1);
                      if (m >= p.pm0 && m < p.pm1 && n >= p.pn0 && n < p.pn1)
                        p.P_out[(static_cast<size_t>(m - p.pm0) * (p.pn1 - p.pn0) + (n - p.pn0)) * p.G + gm] = ia[i][mi][e] >> 8;
                    }
                  }
#pragma unroll
                  for (int e = 0; e < 4; ++e) ia[i][mi][e] = 0;
                }
              }
            }
            continue;
          }
          const __half2 sw2 = *reinterpret_cast<const __half2*>(smem_gen + (st - smem_base) + Cfg::kWBytes + Cfg::kABytes + i * 16 + 4 * t);
          int acc[MT][4];
#pragma unroll
          for (int mi = 0; mi < MT; ++mi)
#pragma unroll
            for (int e = 0; e < 4; ++e) acc[mi][e] = 0;
#pragma unroll
          for (int k4 = 0; k4 < 4; ++k4) {
            const uint32_t b0w = rotl4(x[k4]) & kMask, b1w = x[k4] & kMask;
#pragma unroll
            for (int mi = 0; mi < MT; ++mi) mma_s8(acc[mi], af[mi][k4], b0w, b1w);
          }
          // this k-block's sums: INT32 -> FP32, x sW / 256, x sA (a5)
          const float sw0 = __low2float(sw2) * 0.00390625f, sw1 = __high2float(sw2) * 0.00390625f;
#pragma unroll
          for (int mi = 0; mi < MT; ++mi) {
            yf[i][mi][0] = fmaf(__int2float_rn(acc[mi][0]) * sw0, sa[mi][0], yf[i][mi][0]);
            yf[i][mi][1] = fmaf(__int2float_rn(acc[mi][1]) * sw1, sa[mi][0], yf[i][mi][1]);
            yf[i][mi][2] = fmaf(__int2float_rn(acc[mi][2]) * sw0, sa[mi][1], yf[i][mi][2]);
            yf[i][mi][3] = fmaf(__int2float_rn(acc[mi][3]) * sw1, sa[mi][1], yf[i][mi][3]);
            if constexpr (DUMP) {
#pragma unroll
              for (int e = 0; e < 4; ++e) {
                const int m = 16 * mi + q + 8 * (e >> 1), n = (b0 + i) * 8 + 2 * t + (e & 1);
                if (m >= p.pm0 && m < p.pm1 && n >= p.pn0 && n < p.pn1)   // P_out is zero-filled by the caller
                  atomicAdd(p.P_out + (static_cast<size_t>(m - p.pm0) * (p.pn1 - p.pn0) + (n - p.pn0)) * p.G + gm,
                            acc[mi][e] >> 8);
              }
            }
          }
        }
      }
      __syncwarp();                                     // every lane is done reading the stage
      issue_next(true);                                 // re-arm it with the warp's next k-block
      cslot = cslot + 1 == kStages ? 0 : cslot + 1;
    }

    // ---- a6 / a7: the 16 warps' partials of the batch meet in shared memory; cast, store
#pragma unroll
    for (int i = 0; i < RBB; ++i)
#pragma unroll
      for (int mi = 0; mi < MT; ++mi)
        part[((i * kWarps + w) * MT + mi) * 32 + lane] =
            CH ? make_float4(__int_as_float(ia[i][mi][0]), __int_as_float(ia[i][mi][1]), __int_as_float(ia[i][mi][2]),
                             __int_as_float(ia[i][mi][3]))
               : make_float4(yf[i][mi][0], yf[i][mi][1], yf[i][mi][2], yf[i][mi][3]);
    __syncthreads();
    if (p.Y != nullptr || (CH && DUMP)) {
      for (int i = w; i < nb; i += kWarps) {
#pragma unroll
        for (int mi = 0; mi < MT; ++mi) {
          float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
          const int n = (b0 + i) * 8 + 2 * t;
          const int m = 16 * mi + q;
          if constexpr (CH) {
            // the warps [gamma wpg, (gamma + 1) wpg) hold the parts of group gamma (all 16 for per-channel)
            const int wpg = kWarps / p.G;
            for (int gamma = 0; gamma < p.G; ++gamma) {
              int s0 = 0, s1i = 0, s2i = 0, s3 = 0;         // exact: INT32 all the way
              for (int ww = gamma * wpg; ww < (gamma + 1) * wpg; ++ww) {
                const float4 xx = part[((i * kWarps + ww) * MT + mi) * 32 + lane];
                s0 += __float_as_int(xx.x); s1i += __float_as_int(xx.y); s2i += __float_as_int(xx.z); s3 += __float_as_int(xx.w);
              }
              s0 >>= 8; s1i >>= 8; s2i >>= 8; s3 >>= 8;       // operands were 16 q each
              if constexpr (DUMP) {
                const int sums[4] = {s0, s1i, s2i, s3};
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                  const int mm = m + 8 * (e >> 1), nn = n + (e & 1);
                  if (mm >= p.pm0 && mm < p.pm1 && nn >= p.pn0 && nn < p.pn1)
                    p.P_out[(static_cast<size_t>(mm - p.pm0) * (p.pn1 - p.pn0) + (nn - p.pn0)) * p.G + gamma] = sums[e];
                }
              }
              if constexpr (!DUMP) {   // the dump takes no scales (null pointers; the loads below may be hoisted)
                if (p.Y != nullptr && n < p.N) {
                  // Y += float(P) sW sA (a5), P exact in FP32 (|P| <= 64 K < 2^24): one rounding chain per group (R12)
                  const float sw0 = __half2float(__ldg(p.sW + st16_index(n, gamma, p.G))), sw1 = __half2float(__ldg(p.sW + st16_index(n + 1, gamma, p.G)));
                  const float sa0 = __half2float(__ldg(p.sA + st16_index(m, gamma, p.G))), sa1 = __half2float(__ldg(p.sA + st16_index(m + 8, gamma, p.G)));
                  v.x += __int2float_rn(s0) * sw0 * sa0; v.y += __int2float_rn(s1i) * sw1 * sa0;
                  v.z += __int2float_rn(s2i) * sw0 * sa1; v.w += __int2float_rn(s3) * sw1 * sa1;
                }
              }
            }
            if (p.Y == nullptr || n >= p.N) continue;
          } else {
#pragma unroll
          for (int ww = 0; ww < kWarps; ++ww) {
            const float4 xx = part[((i * kWarps + ww) * MT + mi) * 32 + lane];
            v.x += xx.x; v.y += xx.y; v.z += xx.z; v.w += xx.w;
          }
          }
          if (p.Y != nullptr && n < p.N) {
            if (p.push) {     // K-split tensor parallelism: add into the owner rank's FP32 buffer (see GemmParams)
              const int owner = n / p.push_cols;
              float* yo = p.push_y[owner] + (n - owner * p.push_cols);
              if (m < p.M) asm volatile("red.relaxed.sys.global.add.v2.f32 [%0], {%1, %2};" ::"l"(yo + static_cast<size_t>(m) * p.push_cols), "f"(v.x), "f"(v.y) : "memory");
              if (m + 8 < p.M) asm volatile("red.relaxed.sys.global.add.v2.f32 [%0], {%1, %2};" ::"l"(yo + static_cast<size_t>(m + 8) * p.push_cols), "f"(v.z), "f"(v.w) : "memory");
            } else if (p.out_f32) {
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
template <int MT, int GM, int GS>
static cudaError_t launch_gemv_m(const GemmParams& p, bool dump, int grid, cudaStream_t st) {
  constexpr int smem = GemvCfg<MT, GS>::kSmemBytes;
  cudaError_t e;
  if (dump) {
    auto kern = w4a4_gemv_kernel<MT, true, GM, GS>;
    if ((e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
    if ((e = launch_pdl(kern, dim3(grid), dim3(kThreads), smem, st, p)) != cudaSuccess) return e;
  } else {
    auto kern = w4a4_gemv_kernel<MT, false, GM, GS>;
    if ((e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
    if ((e = launch_pdl(kern, dim3(grid), dim3(kThreads), smem, st, p)) != cudaSuccess) return e;
  }
  return cudaGetLastError();
}
template <int MT>
static cudaError_t launch_gemv_g(const GemmParams& p, int gm, int gs, bool dump, int grid, cudaStream_t st) {
  if (gm == 2) return launch_gemv_m<MT, 2, 1>(p, dump, grid, st);
  if (gm == 1) return launch_gemv_m<MT, 1, 1>(p, dump, grid, st);
  if (gs == 4) return launch_gemv_m<MT, 0, 4>(p, dump, grid, st);
  if (gs == 2) return launch_gemv_m<MT, 0, 2>(p, dump, grid, st);
  return launch_gemv_m<MT, 0, 1>(p, dump, grid, st);
}

// Group mode of the decode kernel for (K, g), or -1 if it does not cover them (see the kernel's GM comment):
// 16 warps split the K / 128 k-blocks evenly; groups of several k-blocks must nest with those ranges.
int gemv_group_mode(int K, int g) {
  const int KB = K / kBlockK;
  if (g <= kBlockK) return (g == 32 || g == 64 || g == kBlockK) ? 0 : -1;
  if (g == K) return 2;                                   // per-channel: every warp inside the one group, any KB
  if (g % kBlockK != 0 || KB % gemv::kWarps != 0) return -1;
  const int q = KB / gemv::kWarps, kbpg = g / kBlockK;
  if (q % kbpg == 0) return 1;
  if (kbpg % q == 0 && gemv::kWarps % (K / g) == 0) return 2;
  return -1;
}

// mt: m16 token tiles (1 or 2)
cudaError_t launch_gemv(const GemmParams& p, int mt, bool dump, int grid, cudaStream_t st) {
  const int gm = gemv_group_mode(p.K, p.g);
  if (gm < 0) return cudaErrorInvalidValue;
  const int gs = p.g < kBlockK ? kBlockK / p.g : 1;     // groups per k-block (g = 64: 2, g = 32: 4)
  switch (mt) {
    case 1: return launch_gemv_g<1>(p, gm, gs, dump, grid, st);
    case 2: return launch_gemv_g<2>(p, gm, gs, dump, grid, st);
    default: return cudaErrorInvalidValue;
  }
}

int gemv_max_batch(int mt) { return mt == 1 ? 7 : 4; }

}  // namespace apex4
