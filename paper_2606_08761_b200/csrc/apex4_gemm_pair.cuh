// apex4_gemm_pair.cuh -- a2..a7 of the hot path (every shape but decode M <= 32): the W4A4 group-dequant
// GEMM of Eq. 8 on a CTA PAIR (cluster of 2, tcgen05 cta_group::2).  The kernel
// template lives here; apex4_gemm_pair_m{0,1,2,3}.cu instantiate it per granularity MODE so that the
// four variants compile in parallel.
//
// A pair owns a 256 (weight rows n) x NT (tokens m) output tile; NT = 192 below, 128 / 64 are the same
// kernel instantiated for small M (Tile<NT>).  CTA r of the pair holds weight rows 128 r .. 128 r + 127
// of the tile on its 128 TMEM lanes and supplies NT/2 of the token rows of every MMA from its own shared
// memory, so per SM and k-block (K = 128) only 8 KB of packed weights and 6 KB of packed activations
// are fetched, widened and read by the tensor core (shared-memory read bandwidth is the scarce resource).
//
// Why 192 tokens: (1) TMEM holds two full 192-column accumulator buffers plus four 32-column
// weight-operand stages (2 x 192 + 4 x 32 = 512), so the MMA of group g+1 runs while the epilogue
// drains group g; (2) an epilogue thread keeps 96 FP32 running sums, which leaves registers for a
// true software prefetch of the next TMEM chunk.
//
// MODE (compile time; every role's loop is specialised, no run-time granularity branches):
//   0  g = 128       one group per k-block; scale slots ride on the operand / accumulator barriers
//   1  g = 64        two groups per k-block       } one accumulator buffer per group, magic-biased
//   2  g = 32        four groups per k-block      } accumulators (see the epilogue)
//   3  g = 128 j > 128 (up to per-channel g = K): j k-blocks accumulate into one buffer, INT32 -> FP32
//                    by I2F once per group
//
// Roles (W widener warpgroups: 1 for MODE 0-2, 2 for MODE 3; the launch register count x threads is
// the pool that setmaxnreg redistributes: control 32, wideners 64, the rest to the epilogue):
//   warps 0..4W-1  wideners : k-blocks dealt alternately between the warpgroups.  INT4 -> INT8 (x16).
//                          Thread r widens weight row r in registers and stores it to TMEM; NT/2 token
//                          rows are widened smem -> smem into the 128B-swizzled UMMA layout.  All
//                          shared-memory loads of a k-block are issued up front and the barriers of the
//                          NEXT k-block are polled (test_wait) while this one is widened: the chain
//                          wait -> LDS -> LOP -> STS/STTM -> fence -> arrive was latency-bound.
//   next 8 warps   epilogue : warpgroup h owns tokens (NT/2) h .. (NT/2) h + NT/2 - 1.  tcgen05.ld.32x32b.x16:
//                          a thread holds one weight row (its TMEM lane) x 16 consecutive tokens per chunk.
//                          Two FFMA2 per element pair: fma(f, sW/256, -49152 sW) = P sW rounded once
//                          (magic-biased accumulators), then fma with the two token scales into the FP32
//                          sums.  Software-pipelined ACROSS groups: chunk c+1 is in flight while chunk c
//                          is in the FMA pipe, and the first chunk of group g+1 (barrier polled two
//                          chunks earlier) is requested before the last chunk's FMAs of group g.
//   then           producer : 1-D bulk async copies (UBLKCP) of this CTA's packed INT4 rows + FP16 scales
//   then           MMA      : leader CTA only; tcgen05.mma cta_group::2 kind::i8, M = 256, N = NT, K = 32,
//                          A (weights) from TMEM, B (tokens) from shared memory; tcgen05.commit
//                          multicast to both CTAs.  Producer and MMA loops run warp-uniform with one
//                          elected lane issuing (operands in uniform registers, no divisions).
#pragma once
#include <type_traits>

#include "apex4_gemm.cuh"
#include "apex4_layout.cuh"
#include "apex4_ptx.cuh"

namespace apex4 {

namespace pair {

// Biased accumulators (g <= 128).  kind::i8 delivers INT32 sums; turning 96 of them per thread and group into floats
// with I2F would cost the epilogue as much as its FMAs.  Instead every group's accumulator STARTS at a bias B, so that
// the word in TMEM, read as binary32, is affine in the group sum P (the operands are 16 q: the sums are 256 P), and the
// conversion is the FMA that scales anyway: t = fma(word, a, b), acc = fma(t, sA', acc).  Two ways to put the bias there:
//  * product: B = 0x4B400000 (float 12582912 + 256 P), re-written by the epilogue with tcgen05.st behind every load;
//    a = sW / 256, b = -49152 sW, sA' = sA;
//  * -DAPEX4_X_BIASSLICE (tuning build, bit-identical results): the tensor core writes it -- a fifth K = 32 MMA with
//    accumulate off whose operands are the constant byte 240 read as UNSIGNED 8-bit from 4 KB of shared memory,
//    32 x 240 x 240 = 1843200 = 256 x 7200 in every element.  256 P lies in [-256 x 7168, 256 x 8192], the word in
//    [8192, 3940352]: a SUBNORMAL binary32 number of value 2^-149 (1843200 + 256 P); a = sW 2^92, b = -7200 sW 2^-49
//    (exact), t = P sW 2^-49 rounded once (no underflow: sW >= 2^-24), sA' = sA 2^49.  No tcgen05.st, no constant
//    registers, the buffer goes back as soon as its last column is in registers -- for 5 tensor-core slices per group
//    instead of 4.  Measured within 2 % of the product (profiles/r2_gemm_pair_ncu.md): the epilogue is bound by what it
//    shares the sub-partition with, not by its own instruction stream.
constexpr uint32_t kMagicBits = 0x4B400000u;   // float 12582912 = 1.5 * 2^23
#ifdef APEX4_X_BIASSLICE
constexpr uint32_t kBiasByte = 240;
constexpr uint32_t kBiasInt = 32u * kBiasByte * kBiasByte;
constexpr float kBiasP = 7200.0f;
constexpr int kConstBytes = 4096;              // 128 rows x 32 bytes of the constant
static_assert(kBiasInt == 256u * 7200u && 7200u >= 7168u && 256u * (7200u + 8192u) < (1u << 23), "bias range");
#else
constexpr uint32_t kBiasInt = kMagicBits;
constexpr int kConstBytes = 0;
#endif
#ifndef APEX4_EPI_WGS_192
#define APEX4_EPI_WGS_192 2          // epilogue warpgroups of the 192-token tile (tuning builds: 3)
#endif
constexpr int kAccBufs = 2;
#ifndef APEX4_X_HALVES
#define APEX4_X_HALVES 1
#endif
// Tuning option (2): each accumulator buffer is produced as two independent column halves -- one MMA of N = NT / 2
// and one full / empty barrier pair per half -- so that the two epilogue warpgroups hand their halves back and
// get them refilled independently.  Measured slower than one MMA per buffer (profiles/r2_gemm_pair_ncu.md): the
// epilogue is bound by its own instruction stream, not by the hand-off.
constexpr int kHalves = APEX4_X_HALVES;
constexpr int kOpStages = 4;        // widened operand stages (TMEM A + smem B)
constexpr int kPkStages = 6;        // packed (bulk copy) stages
constexpr int kScfSlots = 8;
constexpr int kTmemA0 = 384;        // first TMEM column of the A-operand stages
constexpr int kPkWBytes = kBlobBytes;             // 128 weight rows of a k-block
constexpr int kPkSWBytes = 4 * 256;               // up to 4 groups per k-block, 128 FP16 each
constexpr int kPkSABytes = 2 * 4 * 256;           // the (up to) two 128-token blobs the tile touches
constexpr int kNumBars = 2 * kPkStages + 2 * kOpStages + 2 * kScfSlots + 2 * kAccBufs * kHalves;
static_assert((kScfSlots & (kScfSlots - 1)) == 0, "power-of-two wraps");
static_assert((kOpStages & (kOpStages - 1)) == 0, "stage index wraps with a mask");

// Granularity mode -> compile-time constants
template <int MODE>
struct Gran {
  static_assert(MODE >= 0 && MODE <= 3, "mode");
  static constexpr int kGpk = MODE == 1 ? 2 : MODE == 2 ? 4 : 1;   // groups per k-block
#ifdef APEX4_X_NOBIAS
  static constexpr bool kBias = false;
#else
  static constexpr bool kBias = MODE < 3;                          // magic-biased accumulators (g <= 128)
#endif
  static constexpr bool kMultiKb = MODE == 3;                      // several k-blocks per group (run-time count)
  // Scale-slot hand-shake.  At g = 128 (one group per k-block) it is implied by the operand / accumulator
  // barriers and skipped -- every mbarrier wait costs ~100 clk even when the phase is already complete:
  //  * full:  the wideners write slot k before they publish operand stage k, the MMA of group k is
  //           issued after that, so "accumulator k full" implies "scales k written";
  //  * empty: the widener of k-block k has waited for operand stage k % 4 = MMA k-4 done, which was
  //           issued after all epilogue warps released accumulator k-6, i.e. had finished group k-7's
  //           last read of its slot (the epilogue reads slot k+1's row scales at the end of group k);
  //           slot k % 8 was last used by group k-8.
  static constexpr bool kScfSync = MODE != 0;
#ifdef APEX4_X_WWG
  static constexpr int kWidenWGs = APEX4_X_WWG;
#else
  static constexpr int kWidenWGs = MODE == 3 ? 2 : 1;
#endif
};
inline int gran_mode(int g) { return g == kBlockK ? 0 : g == 64 ? 1 : g == 32 ? 2 : 3; }

// Everything that depends on the token width NT of the pair tile (MMA N = accumulator buffer width):
// 192 in the tensor-bound regime, 128 / 64 where M would leave most of a 192-token tile empty.
// Widener warpgroups for (MODE, NT): two where the wideners, not the epilogue, set the pace -- groups of several
// k-blocks (MODE 3), and (tuning switch APEX4_X_WWG_NT: token width up to which two are used) narrow token tiles, whose
// epilogue is short while a k-block's 128 weight rows cost the wideners the same ~750 clk whatever the token width is.
#ifndef APEX4_X_WWG_NT
#define APEX4_X_WWG_NT 0
#endif
template <int MODE, int NT>
__host__ __device__ constexpr int widen_wgs() { return (Gran<MODE>::kWidenWGs == 2 || NT <= APEX4_X_WWG_NT) ? 2 : Gran<MODE>::kWidenWGs; }

template <int NT>
struct Tile {
  static constexpr int kNT = NT;
  static constexpr int kHalf = NT / 2;                  // token rows per CTA (its half of the B operand)
  static constexpr int kEpiWGs = NT == 192 ? APEX4_EPI_WGS_192 : 2;   // epilogue warpgroups, each owns NT / kEpiWGs token columns
  static constexpr int kEpiWarps = 4 * kEpiWGs;
  static constexpr int kEpiCols = NT / kEpiWGs;         // accumulator columns per epilogue warpgroup
  static constexpr int kChunks = kEpiCols / 16;         // 16-column TMEM chunks per epilogue thread
  static constexpr int kTokIters = kHalf / 32;          // 16-byte token pieces per widener thread
  static constexpr int kPkABytes = kHalf * kRowBytes;   // packed token rows of a k-block
  static constexpr int kPkStageBytes = kPkWBytes + kPkABytes + kPkSWBytes + kPkSABytes;
  static constexpr int kI8StageBytes = kHalf * kBlockK; // widened tokens: [kHalf rows][128 B]
  static constexpr int kScfSlotBytes = kTileRows * 8 + NT * 4 + 256;   // {a,b} per row, sA per column (padded)
  static constexpr int kStoreBytes = kEpiCols * 64;     // per epilogue warp: [kEpiCols m][32 n] FP16 output staging
  static constexpr int kSmemBytes = 1024 + kOpStages * kI8StageBytes + kPkStages * kPkStageBytes +
                                    kScfSlots * kScfSlotBytes + kNumBars * 8 + 64 + 64 + kEpiWarps * kStoreBytes +
                                    (kConstBytes ? 128 + kConstBytes : 0);
  static_assert(NT % 64 == 0 && NT <= kPairTokens, "token width");
  static_assert(kAccBufs * NT <= kTmemA0 && kTmemA0 + 32 * kOpStages <= 512, "TMEM columns");
  static_assert(kI8StageBytes % 1024 == 0 && kPkStageBytes % 16 == 0, "alignment");
  static_assert(kSmemBytes <= 232448, "shared memory");
  static_assert(NT % (16 * kEpiWGs) == 0, "epilogue warpgroups own whole 16-column chunks");
  static_assert(kChunks % 2 == 0, "the cross-group prefetch lands in v[0] while the last (odd) chunk is in v[1]");
  static constexpr int kPieceRows = kHalf / kHalves;    // token rows per CTA and accumulator half
  static constexpr int kMmaN = NT / kHalves;
  static_assert(kHalves == 1 || kEpiWGs == kHalves, "one epilogue warpgroup per accumulator half");
  static_assert(kPieceRows % 8 == 0 && kMmaN % 16 == 0, "swizzle atoms / MMA N of a half");
};

// Warp layout for WWG widener warpgroups.  With one, the wideners of a CTA run one k-block at a time:
// fewer warps competing for issue slots, which is what the epilogue-heavy fine granularities want;
// with two, k-blocks are dealt alternately and the bulk copy -> widen -> MMA chain is shorter, which is
// what counts once the epilogue is rare (g >= 256).  The register pool is threads x launch registers
// (<= 64 K), redistributed by setmaxnreg: control 32, wideners 64, the rest to the epilogue.
template <int WWG, int EW>
struct Warps {
  static constexpr int kEpiWGs = EW;
  static constexpr int kEpiWarps = 4 * EW;
  static constexpr int kWidenWGs = WWG;                     // k-blocks dealt alternately
  static constexpr int kEpiWarp0 = 4 * WWG;                 // first epilogue warp
  static constexpr int kCtlWarp0 = kEpiWarp0 + kEpiWarps;   // producer warp; the MMA warp follows
  static constexpr int kThreads = 32 * (kCtlWarp0 + 4);     // warps are allocated in fours: two control warps idle
  static constexpr int kLaunchRegs = (65536 / kThreads) / 8 * 8;
  // control 24 (the minimum; the producer spills two work-iterator words, off the critical path), wideners 56:
  // with one widener warpgroup that leaves 216 for the epilogue, whose group loop (96 FP32 accumulators, two 16-column
  // TMEM chunks, 16 token scales, the magic bias) spills at 208 -- 414 us against 368 us at M = 4096, N = K = 8192
  // (with two widener warpgroups the epilogue gets 168 either way, and the control warps keep 32)
  static constexpr int kRegsCtl = WWG == 1 ? 24 : 32, kRegsWiden = 56;
  static constexpr int kRegsEpi = ((kThreads * kLaunchRegs - 128 * kRegsCtl - 128 * WWG * kRegsWiden) / (128 * kEpiWGs)) / 8 * 8;
  static_assert((WWG & (WWG - 1)) == 0, "k-blocks are dealt with a mask");
  static_assert(128 * kRegsCtl + 128 * WWG * kRegsWiden + 128 * kEpiWGs * kRegsEpi <= kThreads * kLaunchRegs, "registers");
  static_assert(kRegsEpi <= 232 && kThreads <= 1024, "register / thread limits");
};

// "a group follows" as a compile-time fact of one copy of the epilogue's group body
struct Always {
  __device__ constexpr operator bool() const { return true; }
};

struct Work {
  int nt, mt;      // pair tile: 256 weight rows x NT tokens
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
// Tiles are numbered token-tile fastest: pairs that run together share weight tiles in L2.
__device__ __forceinline__ bool work_next(const GemmParams& p, WorkIter& it, Work& w, int cp, int npairs) {
#ifdef APEX4_PAIR_EMPTY   // tuning builds only: launch + set-up + teardown cost
  return false;
#endif
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

template <int MODE, bool DUMP, int NT, bool PUSH = false>
__global__ void __cluster_dims__(2, 1, 1) __maxnreg__((Warps<widen_wgs<MODE, NT>(), Tile<NT>::kEpiWGs>::kLaunchRegs))
    w4a4_gemm_pair_kernel(const GemmParams p) {
  using GR = Gran<MODE>;
  using L = Warps<widen_wgs<MODE, NT>(), Tile<NT>::kEpiWGs>;
  using T = Tile<NT>;
  constexpr bool BIAS = GR::kBias;
  constexpr int GPK = GR::kGpk;
  constexpr bool kScfSync = GR::kScfSync;
  constexpr int kNT = T::kNT, kHalf = T::kHalf, kEpiCols = T::kEpiCols, kChunks = T::kChunks;
  constexpr int kEpiWarps = T::kEpiWarps;
  constexpr int kPieceRows = T::kPieceRows;
  constexpr int kPkABytes = T::kPkABytes, kPkStageBytes = T::kPkStageBytes, kI8StageBytes = T::kI8StageBytes;
  constexpr int kScfSlotBytes = T::kScfSlotBytes, kStoreBytes = T::kStoreBytes, kTokIters = T::kTokIters;
  constexpr int kWidenWGs = L::kWidenWGs, kEpiWarp0 = L::kEpiWarp0, kCtlWarp0 = L::kCtlWarp0;
  constexpr int kRegsCtl = L::kRegsCtl, kRegsWiden = L::kRegsWiden, kRegsEpi = L::kRegsEpi;
  extern __shared__ uint8_t smem_raw[];
  // opaque: otherwise ptxas re-derives the base (S2R SR_CgaCtaId + 4 integer ops) in front of every
  // barrier wait and shared-memory access instead of keeping it in a register
  uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  asm volatile("" : "+r"(smem_base));
  uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
#ifdef APEX4_TIMELINE   // event 18: kernel entry / set-up done / before / after the teardown barrier (thread 0 of CTA 0, 1)
  if (p.tl != nullptr && blockIdx.x < 2 && threadIdx.x == 0) p.tl[(blockIdx.x * 32 + 18) * 64 + 0] = clock64();
#endif

  constexpr uint32_t offI8 = 0;
  constexpr uint32_t offPk = offI8 + kOpStages * kI8StageBytes;
  constexpr uint32_t offScf = offPk + kPkStages * kPkStageBytes;
  constexpr uint32_t offBar = offScf + kScfSlots * kScfSlotBytes;
  constexpr uint32_t offTmemPtr = offBar + kNumBars * 8;
  constexpr uint32_t offMagic = offTmemPtr + 64;       // 8 words of the magic bias (see epilogue)
  constexpr uint32_t offStore = (offMagic + 64 + 15) / 16 * 16;   // 8 x kStoreBytes output staging
  auto bar = [&](int i) { return smem_base + offBar + 8u * i; };
  constexpr int bPkFull = 0, bPkEmpty = bPkFull + kPkStages, bOpFull = bPkEmpty + kPkStages,
                bOpEmpty = bOpFull + kOpStages, bScfFull = bOpEmpty + kOpStages,
                bScfEmpty = bScfFull + kScfSlots, bAccFull = bScfEmpty + kScfSlots,
                bAccEmpty = bAccFull + kAccBufs * kHalves;   // index: buffer * kHalves + half

  // warp index through a shuffle from lane 0: tells the compiler it is warp-uniform, so addresses derived
  // from it (TMEM lane quarter, barrier and stage addresses) live in uniform registers (no R2UR per use)
  const int warp = __shfl_sync(0xffffffffu, static_cast<int>(threadIdx.x >> 5), 0);
  int lane = threadIdx.x & 31;
  asm volatile("" : "+r"(lane));                // no S2R SR_TID.X inside the loops
  const uint32_t rank = cluster_ctarank();      // 0 = leader
  const int cp = blockIdx.x >> 1;               // pair index
  const int npairs = gridDim.x >> 1;
  const int kbpg = GR::kMultiKb ? p.g / kBlockK : 1;    // k-blocks per group (MODE 3 only)

  if (threadIdx.x == 0) {
    for (int i = 0; i < kPkStages; ++i) { mbar_init(bar(bPkFull + i), 1); mbar_init(bar(bPkEmpty + i), 128); }
    // operand stage full: one elected arrive per widener warp of BOTH CTAs, on the leader's barrier
    for (int i = 0; i < kOpStages; ++i) { mbar_init(bar(bOpFull + i), 8); mbar_init(bar(bOpEmpty + i), 1); }
    for (int i = 0; i < kScfSlots; ++i) { mbar_init(bar(bScfFull + i), 128); mbar_init(bar(bScfEmpty + i), kEpiWarps); }
    // accumulator buffer empty: one elected arrive per epilogue warp of BOTH CTAs, on the leader's barrier
    for (int i = 0; i < kAccBufs * kHalves; ++i) { mbar_init(bar(bAccFull + i), 1); mbar_init(bar(bAccEmpty + i), 2 * kEpiWarps / kHalves); }
    fence_mbar_init();
  }
  if (threadIdx.x < 8) reinterpret_cast<volatile uint32_t*>(smem_gen + offMagic)[threadIdx.x] = kMagicBits;
#ifdef APEX4_X_BIASSLICE
  constexpr uint32_t offConst = (offStore + kEpiWarps * kStoreBytes + 127) / 128 * 128;   // operands of the bias slice
  if constexpr (BIAS) {
    constexpr uint32_t kFill = kBiasByte * 0x01010101u;
    for (int i = threadIdx.x; i < kConstBytes / 16; i += L::kThreads)
      reinterpret_cast<uint4*>(smem_gen + offConst)[i] = make_uint4(kFill, kFill, kFill, kFill);
    fence_proxy_async_smem();     // read by the tcgen05.mma (async proxy) the leader issues, in both CTAs
  }
#endif
  if (warp == kCtlWarp0 + 1) tmem_alloc_pair<512>(smem_base + offTmemPtr);
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();       // barriers of both CTAs initialised before any remote arrive / multicast
  tc_fence_after();
  const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(smem_gen + offTmemPtr);
  if (tmem_base != 0) __trap();   // the whole TMEM (512 columns) is ours: lane 0, column 0
#ifndef APEX4_X_NOPDL
  // Programmatic dependent launch: the set-up above (barriers, TMEM, cluster rendezvous) overlapped the tail of the
  // predecessor on the stream (the online quantizer); from here on its output is complete and visible.  The successor
  // may be scheduled as soon as SMs free up; every kernel of this library waits before it reads or writes global memory.
  griddep_launch();
  griddep_wait();
#endif

#ifdef APEX4_TIMELINE
  if (p.tl != nullptr && blockIdx.x < 2 && threadIdx.x == 0) p.tl[(blockIdx.x * 32 + 18) * 64 + 1] = clock64();
#endif
  WorkIter wit;
  Work w;
  work_begin(p, wit, cp, npairs);
  auto stamp = [&](int ev, uint32_t k) {   // debug timeline: compiled in with -DAPEX4_TIMELINE only
#ifdef APEX4_TIMELINE
    if (p.tl != nullptr && blockIdx.x < 2 && k < 64) p.tl[(blockIdx.x * 32 + ev) * 64 + k] = clock64();
#endif
  };

  // =========================================================================== control warps
  if (warp >= kCtlWarp0) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsCtl));
    // ------------------------------------------------------------------------- producer
    // The whole warp runs the loop on warp-uniform values, one elected lane issues the copies;
    // source pointers advance by a blob per k-block (no division, no 64-bit multiplies).
    if (warp == kCtlWarp0) {
      const bool el = elect_one();
      const int n_blobs = round_up(p.N, kTileRows) / kTileRows;
      const int m_blobs = round_up(p.M, kTileRows) / kTileRows;
      constexpr uint32_t sc_bytes = GPK * 256;
      const size_t row_pitch = static_cast<size_t>(p.K / kBlockK) * kBlobBytes;   // bytes per blob row
      const size_t srow_pitch = static_cast<size_t>(p.G) * kTileRows;               // FP16 scales per blob row
      uint32_t s = 0, pkpar = 0;
      while (work_next(p, wit, w, cp, npairs)) {
        const int wblob = 2 * w.nt + static_cast<int>(rank);
        const bool has_w = wblob < n_blobs;
        // this CTA's token rows: accumulator half hh covers tile tokens [hh * kMmaN, (hh + 1) * kMmaN), of which
        // this CTA supplies kPieceRows (the MMA takes N / 2 rows of B from each CTA); a piece may straddle two blobs
        int ar0[kHalves], n1[kHalves], n2[kHalves];
        const uint8_t* asrc[kHalves];
        uint32_t arows = 0;
#pragma unroll
        for (int hh = 0; hh < kHalves; ++hh) {
          const int t0 = w.mt * kNT + hh * T::kMmaN + static_cast<int>(rank) * kPieceRows;
          const int ab0 = t0 >> 7;
          ar0[hh] = t0 & 127;
          n1[hh] = ab0 < m_blobs ? min(kPieceRows, kTileRows - ar0[hh]) : 0;
          n2[hh] = (ab0 + 1 < m_blobs) ? kPieceRows - min(kPieceRows, kTileRows - ar0[hh]) : 0;
          asrc[hh] = p.qA + ab0 * row_pitch + static_cast<size_t>(w.kb0) * kBlobBytes + ar0[hh] * kRowBytes;
          arows += n1[hh] + n2[hh];
        }
        // token scales: the two blobs the tile touches
        const int sb0 = (w.mt * kNT) >> 7;
        const int s_blobs = min((((w.mt * kNT) & 127) + kNT > kTileRows) ? 2 : 1, m_blobs - sb0);
        const int gfirst0 = GR::kMultiKb ? w.kb0 / kbpg : w.kb0 * GPK;
        const uint8_t* wsrc = p.qW + wblob * row_pitch + static_cast<size_t>(w.kb0) * kBlobBytes;
        const __half* swsrc = p.sW + wblob * srow_pitch + static_cast<size_t>(gfirst0) * kTileRows;
        const __half* sasrc = p.sA + sb0 * srow_pitch + static_cast<size_t>(gfirst0) * kTileRows;
        const uint32_t bytes_data = (has_w ? kBlobBytes : 0) + arows * kRowBytes;
        const uint32_t bytes_scales = sc_bytes * ((has_w ? 1 : 0) + s_blobs);
        int kig = 0;
        for (int kb = w.kb0; kb < w.kb1; ++kb) {
          mbar_wait(bar(bPkEmpty + s), ((pkpar >> s) & 1) ^ 1);
          pkpar ^= 1u << s;
          const uint32_t st = smem_base + offPk + s * kPkStageBytes;
          const uint32_t full = bar(bPkFull + s);
          const bool has_scales = !DUMP && kig == 0;   // the dump of the integer sums takes no scales (null pointers)
          if (el) {
            mbar_arrive_expect_tx(full, bytes_data + (has_scales ? bytes_scales : 0));
            if (has_w) bulk_g2s(st, wsrc, kBlobBytes, full);
#pragma unroll
            for (int hh = 0; hh < kHalves; ++hh) {
              const uint32_t dst = st + kPkWBytes + hh * kPieceRows * kRowBytes;
              if (n1[hh] > 0) bulk_g2s(dst, asrc[hh], n1[hh] * kRowBytes, full);
              if (n2[hh] > 0)   // rows 0.. of the next blob
                bulk_g2s(dst + n1[hh] * kRowBytes, asrc[hh] + row_pitch - ar0[hh] * kRowBytes, n2[hh] * kRowBytes, full);
            }
            if (has_scales) {
              if (has_w) bulk_g2s(st + kPkWBytes + kPkABytes, swsrc, sc_bytes, full);
              if (s_blobs > 0) bulk_g2s(st + kPkWBytes + kPkABytes + kPkSWBytes, sasrc, sc_bytes, full);
              if (s_blobs > 1)
                bulk_g2s(st + kPkWBytes + kPkABytes + kPkSWBytes + sc_bytes, sasrc + srow_pitch, sc_bytes, full);
            }
          }
          wsrc += kBlobBytes;
#pragma unroll
          for (int hh = 0; hh < kHalves; ++hh) asrc[hh] += kBlobBytes;
          if (kig == 0) { swsrc += sc_bytes / 2; sasrc += sc_bytes / 2; }
          if constexpr (GR::kMultiKb) kig = (kig == kbpg - 1) ? 0 : kig + 1;
          s = (s == kPkStages - 1) ? 0 : s + 1;
        }
      }
    }
    // ------------------------------------------------------------------------- MMA issuer (leader)
    // Whole warp, warp-uniform values, one elected lane issues.  No division, no 64-bit descriptor
    // arithmetic, stage / buffer parities kept as bit masks.
    else if (warp == kCtlWarp0 + 1 && rank == 0) {
      const bool el = elect_one();
      const uint32_t desc_lo0 = (((smem_base + offI8) & 0x3FFFFu) >> 4) | (1u << 16);
#ifdef APEX4_X_BIASSLICE   // the constant operands: any 128 (A) / kHalf (B) rows x 32 bytes inside the 4 KB region
      const uint64_t cdesc = umma_desc_noswizzle(smem_base + offConst, 128, 256);
#endif
      uint32_t kbc = 0, t = 0, oppar = 0, accpar = 0;
      while (work_next(p, wit, w, cp, npairs)) {
        int kig = 0;                                     // k-block inside the group (MODE 3)
        uint32_t buf0 = 0;                               // group i of a work item uses accumulator buffer i & 1
        for (int kb = w.kb0; kb < w.kb1; ++kb, ++kbc) {
          mbar_wait(bar(bOpFull + t), (oppar >> t) & 1);
          oppar ^= 1u << t;
          tc_fence_after();
          if (el) stamp(4, kbc);
          const bool first = kig == 0;
          const bool last = !GR::kMultiKb || kig == kbpg - 1;
          const uint32_t a_tm = kTmemA0 + 32 * t;        // the 512-column allocation starts at column 0
          const uint32_t blo = desc_lo0 + t * (kI8StageBytes >> 4);
          constexpr int KS = 4 / GPK;
#pragma unroll
          for (int sub = 0; sub < GPK; ++sub) {
            const uint32_t buf = (buf0 + sub) & 1;       // one accumulator buffer per group
#pragma unroll
            for (int hh = 0; hh < kHalves; ++hh) {
              const uint32_t ab = buf * kHalves + hh;
              if (first) {
                mbar_wait(bar(bAccEmpty + ab), (accpar >> ab) & 1);
                accpar ^= 1u << ab;
                tc_fence_after();
                if (el) stamp(8, kbc);
              }
              const uint32_t d_tm = buf * kNT + hh * T::kMmaN;
              const uint32_t bh = blo + hh * (kPieceRows * kBlockK >> 4);   // B rows of this half
#if defined(APEX4_X_BIASSLICE) && !defined(APEX4_X_NOMMA)
              if (BIAS && el) mma_u8_ss_pair_overwrite<T::kMmaN>(d_tm, cdesc, cdesc);   // the group starts at the bias
#endif
#pragma unroll
              for (int ks = 0; ks < KS; ++ks) {
                const int kq = sub * KS + ks;            // K=32 slice of the k-block
#ifndef APEX4_X_NOMMA   // experiment builds: the barrier protocol without the tensor work
                if (el) {
                  if (BIAS || ks != 0) mma_i8_ts_pair_lohi<true, T::kMmaN>(d_tm, a_tm + 8 * kq, bh + 2 * kq, 1u);
                  else mma_i8_ts_pair_lohi<false, T::kMmaN>(d_tm, a_tm + 8 * kq, bh + 2 * kq, first ? 0u : 1u);
                }
#endif
              }
              if (last && el) tc_commit_pair(bar(bAccFull + ab), 3);
            }
          }
          if (el) tc_commit_pair(bar(bOpEmpty + t), 3);
          if (el) stamp(5, kbc);
          t = (t + 1) & (kOpStages - 1);
          if (last) { buf0 = (buf0 + GPK) & 1; kig = 0; } else { ++kig; }
        }
      }
    }
  }
  // =========================================================================== wideners
  else if (warp < kEpiWarp0) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsWiden));
    const int wwg = warp >> 2;                          // widener warpgroup
    const int r = threadIdx.x & 127;                    // weight row of this CTA's blob = TMEM lane
    const uint32_t lane_addr = static_cast<uint32_t>((warp & 3) * 32) << 16;
    const uint32_t wsw = (r >> 1) & 3;                  // chunk-slot swizzle of the packed row (PW4)
    const uint32_t flip = ((lane >> 2) & 1) * 16;       // order of the two 16-byte stores: spreads them over the banks
    constexpr uint32_t kMask = 0xF0F0F0F0u;
    // per-thread offsets inside a packed stage / an operand stage, computed once
    uint32_t w_off0 = r * kRowBytes + ((0 ^ wsw) << 4), w_off1 = r * kRowBytes + ((1 ^ wsw) << 4);
    uint32_t w_off2 = r * kRowBytes + ((2 ^ wsw) << 4), w_off3 = r * kRowBytes + ((3 ^ wsw) << 4);
    uint32_t a_off = kPkWBytes + r * 16;                // + 2048 x
    uint32_t d_off = offI8 + r * 32;                    // + 4096 x
    asm volatile("" : "+r"(w_off0), "+r"(w_off1), "+r"(w_off2), "+r"(w_off3), "+r"(a_off), "+r"(d_off));
    uint32_t kbc = 0, gc = 0;
    // this warpgroup's cursor: k-block index kbc -> packed stage kbc % 6, operand stage kbc % 4
    uint32_t s = wwg % kPkStages, t = wwg & (kOpStages - 1), pk_ph = 0, op_ph = 0;
    uint32_t ok_pk = 0, ok_op = 0;                      // the NEXT own k-block's barriers, polled ahead
    while (work_next(p, wit, w, cp, npairs)) {
      const int sa_row = (w.mt * kNT) & 127;            // tile token 0 inside its first scale blob
      // token-scale sources of this thread inside a stage's scale area (FP16 index): columns r and r + 128
      const int mm0 = sa_row + r, mm1 = sa_row + r + 128;
      const uint32_t sa_src0 = ((mm0 >> 7) * GPK) * kTileRows + (mm0 & 127);   // + sub * 128
      const uint32_t sa_src1 = ((mm1 >> 7) * GPK) * kTileRows + (mm1 & 127);
      int kig = 0;
      for (int kb = w.kb0; kb < w.kb1; ++kb, ++kbc) {
        const bool starts_group = kig == 0;
        if constexpr (GR::kMultiKb) kig = (kig == kbpg - 1) ? 0 : kig + 1;
        if (kWidenWGs > 1 && static_cast<int>(kbc & (kWidenWGs - 1)) != wwg) {   // the other warpgroup's k-block
          if (starts_group) gc += GPK;
          continue;
        }
        const uint32_t s_cur = s, t_cur = t;
        if (!ok_pk) mbar_wait(bar(bPkFull + s_cur), pk_ph);
        if (r == 0) stamp(1, kbc);
        const uint32_t pk_addr = smem_base + offPk + s_cur * kPkStageBytes;
        // ---- all shared-memory loads of the k-block up front
        uint32_t wv[16], av[4 * kTokIters];
        lds128(pk_addr + w_off0, wv[0], wv[1], wv[2], wv[3]);
        lds128(pk_addr + w_off1, wv[4], wv[5], wv[6], wv[7]);
        lds128(pk_addr + w_off2, wv[8], wv[9], wv[10], wv[11]);
        lds128(pk_addr + w_off3, wv[12], wv[13], wv[14], wv[15]);
#pragma unroll
        for (int x = 0; x < kTokIters; ++x)
          lds128(pk_addr + a_off + 2048 * x, av[4 * x], av[4 * x + 1], av[4 * x + 2], av[4 * x + 3]);
        if (!ok_op) mbar_wait(bar(bOpEmpty + t_cur), op_ph ^ 1);
        tc_fence_after();
        if (r == 0) stamp(2, kbc);
        // ---- advance the cursor and poll the next own k-block's barriers: their latency hides behind
        // the widening below (a completed mbarrier wait still costs ~100 clk)
        {
          s += kWidenWGs;
          if (s >= kPkStages) { s -= kPkStages; pk_ph ^= 1; }
          const uint32_t t_new = (t + kWidenWGs) & (kOpStages - 1);
          if (t_new < t) op_ph ^= 1;
          t = t_new;
          ok_pk = mbar_test_wait(bar(bPkFull + s), pk_ph);
          ok_op = mbar_test_wait(bar(bOpEmpty + t), op_ph ^ 1);
        }
#ifndef APEX4_X_NOWIDEN   // experiment builds: wideners only pass the barriers on
        // ---- weights: packed row r (64 bytes) -> 32 INT8 words -> TMEM columns of stage t
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
          uint32_t o[16];
#pragma unroll
          for (int j = 0; j < 2; ++j) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              o[8 * j + i] = rotl4(wv[8 * hh + 4 * j + i]) & kMask;
              o[8 * j + 4 + i] = wv[8 * hh + 4 * j + i] & kMask;
            }
          }
          tmem_st_32x16(tmem_base + lane_addr + kTmemA0 + 32 * t_cur + 16 * hh, o);
        }
        if (r == 0) stamp(9, kbc);
        // ---- tokens: kHalf rows x 4 packed chunks; byte offset o -> INT8 offsets 2o (lo), 2o+16 (hi)
        {
          const uint32_t dst0 = smem_base + d_off + t_cur * kI8StageBytes;
#pragma unroll
          for (int x = 0; x < kTokIters; ++x) {
            const uint32_t dst = dst0 + 4096 * x;
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
        // ---- scales of the groups that start in this k-block: FP16 -> FP32, BEFORE the stage is published:
        // at g = 128 the epilogue takes "accumulator full" as "scales written" (Gran<MODE>::kScfSync)
        if (starts_group) {
          const uint8_t* pk = smem_gen + offPk + s_cur * kPkStageBytes;
          const __half* sWh = reinterpret_cast<const __half*>(pk + kPkWBytes + kPkABytes);
          const __half* sAh = sWh + kPkSWBytes / 2;     // [blob 0/1][sub][128]
#pragma unroll
          for (int sub = 0; sub < GPK; ++sub, ++gc) {
            const int q = gc % kScfSlots;
            if (kScfSync) mbar_wait(bar(bScfEmpty + q), ((gc / kScfSlots) & 1) ^ 1);
            float* dstf = reinterpret_cast<float*>(smem_gen + offScf + q * kScfSlotBytes);
            const float sw = __half2float(sWh[sub * kTileRows + r]);
            float sa0 = __half2float(sAh[sa_src0 + sub * kTileRows]);
            float sa1 = 0.f;
            if (kNT > kTileRows && r + kTileRows < kNT) sa1 = __half2float(sAh[sa_src1 + sub * kTileRows]);
#ifdef APEX4_X_BIASSLICE
            reinterpret_cast<float2*>(dstf)[r] = BIAS ? make_float2(sw * 0x1p92f, sw * (-kBiasP * 0x1p-49f)) : make_float2(sw * 0.00390625f, 0.f);
            if (BIAS) { sa0 *= 0x1p49f; sa1 *= 0x1p49f; }
#else
            // a = sW / 256 (the operands are 16 q each); b = -12582912 * a removes the magic bias
            reinterpret_cast<float2*>(dstf)[r] = make_float2(sw * 0.00390625f, sw * -49152.0f);
#endif
            // token scales, in tile order (an epilogue thread reads the 16 of a chunk as four 16-byte vectors)
            if (r < kNT) dstf[2 * kTileRows + r] = sa0;
            if (kNT > kTileRows && r + kTileRows < kNT) dstf[2 * kTileRows + r + kTileRows] = sa1;
            if (kScfSync) mbar_arrive(bar(bScfFull + q));
          }
        }
#endif
        // ---- publish stage t: one elected arrive per warp on the leader's barrier
        if (r == 0) stamp(10, kbc);
        fence_proxy_async_smem();
        tmem_st_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(bar(bOpFull + t_cur), 0);
        if (r == 0) stamp(3, kbc);
        mbar_arrive(bar(bPkEmpty + s_cur));
        if (r == 0) stamp(13, kbc);
      }
    }
  }
  // =========================================================================== epilogue
  else {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegsEpi));
    const int h = (warp - kEpiWarp0) >> 2;              // warpgroup = slice of kEpiCols token columns
    const int hsel = kHalves == 1 ? 0 : h;              // which full / empty barrier pair of a buffer is ours
    const int lq = warp & 3;                            // TMEM lane quarter this warp may access
    const int epi_tid = threadIdx.x - 32 * kEpiWarp0;
    const uint32_t lane_addr = static_cast<uint32_t>(lq * 32) << 16;
    const int row0 = lq * 32 + lane;                    // weight row of the CTA's blob = TMEM lane
    // per-thread address parts of the group loop, made opaque so that ptxas keeps them in registers
    // instead of re-deriving them from %tid in every group (11 S2R + ~40 integer ops per group)
    const uint32_t tm_rd = lane_addr + h * kEpiCols;                                   // + buf * kNT
    uint32_t ab_off = offScf + row0 * 8;                                      // {a, b} of row row0
    uint32_t sa_off = offScf + kTileRows * 8 + (h * kEpiCols) * 4;            // token scales (+ 64 c)
    asm volatile("" : "+r"(ab_off), "+r"(sa_off));   // tm_rd stays warp-uniform (uniform registers)
    // the magic bias in 8 registers, read through a volatile load so that ptxas keeps them resident
    // instead of re-materialising 16 constants per tcgen05.st (IMAD.MOV on the FMA pipe)
    uint32_t mg[8];
#ifndef APEX4_X_BIASSLICE
    {
      const uint32_t ma = smem_base + offMagic;
      asm volatile("ld.volatile.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(mg[0]), "=r"(mg[1]), "=r"(mg[2]), "=r"(mg[3]) : "r"(ma));
      asm volatile("ld.volatile.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(mg[4]), "=r"(mg[5]), "=r"(mg[6]), "=r"(mg[7]) : "r"(ma + 16));
    }
#endif
    // completion #0 of the accEmpty barriers: both buffers start out holding the magic bias
#pragma unroll
    for (int b = 0; b < kAccBufs; ++b) {
#ifndef APEX4_X_BIASSLICE
      if (BIAS) {
#pragma unroll
        for (int c = 0; c < kEpiCols; c += 8) tmem_st_32x8(tmem_base + lane_addr + b * kNT + h * kEpiCols + c, mg);
        tmem_st_wait();
      }
#endif
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(bar(bAccEmpty + b * kHalves + hsel), 0);
    }

    uint32_t gc = 0, item = 0;
    uint32_t fullph = 0;                                // bit b: parity of the next "accumulator b full" phase
    while (work_next(p, wit, w, cp, npairs)) {
      if (epi_tid == 0) stamp(15, item * 4);
      const int nkb = w.kb1 - w.kb0;
      const int ngroups = GR::kMultiKb ? nkb / kbpg : nkb * GPK;
      uint64_t acc[8 * kChunks];                        // FP32 pairs: tokens 2 x, 2 x + 1 of the slice
#pragma unroll
      for (int i = 0; i < 8 * kChunks; ++i) acc[i] = 0ull;
      const int n_glob0 = (2 * w.nt + static_cast<int>(rank)) * kTileRows + row0;
      const int m_glob0 = w.mt * kNT + h * kEpiCols;        // + 16 c + j
      const int gamma0 = GR::kMultiKb ? w.kb0 / kbpg : w.kb0 * GPK;

      // The group loop is software-pipelined and unrolled by two (group i of the work item lives in
      // accumulator buffer i & 1, so every TMEM address is a compile-time offset from a warp-uniform base
      // and the rotating registers -- the chunk buffers, the row scales -- need no moves): on entry to a
      // group body the group's barriers have been waited for, its row scales {a, b} are in `ab` and its
      // first TMEM chunk is in flight in v[0].
      constexpr int kVBufs = T::kEpiWGs >= 3 ? 1 : 2;   // three warpgroups hide the TMEM latency by themselves
      uint32_t v[kVBufs][16];
      float ab0[2], ab1[2];                              // row scales {a, b} of the even / odd group in flight
      // blocking = false: the barriers were polled earlier (ok != 0: complete)
      auto group_begin = [&](auto bufc, uint32_t gcx, float (&ab)[2], bool blocking, uint32_t ok) {
        constexpr uint32_t BUF = decltype(bufc)::value;
        const int slot = gcx % kScfSlots;
        // the polled flag becomes warp-uniform HERE (a vote right behind the poll would expose its latency):
        // the branch does not diverge, so TMEM addresses stay in uniform registers across it
        if (blocking || !__all_sync(0xffffffffu, ok)) {
          if (kScfSync) mbar_wait_warp(bar(bScfFull + slot), (gcx / kScfSlots) & 1);
          mbar_wait_warp(bar(bAccFull + BUF * kHalves + hsel), (fullph >> BUF) & 1);
        }
        fullph ^= 1u << BUF;
        unpack_f2(lds64(smem_base + slot * kScfSlotBytes + ab_off), ab[0], ab[1]);
        tc_fence_after();
#ifndef APEX4_X_NOLDTM
        tmem_ld_32x16(tm_rd + BUF * kNT, v[0]);
#endif
      };
      auto group_body = [&](auto bufc, auto morec, int gi, const float (&ab)[2], float (&ab_next)[2]) {
        constexpr uint32_t BUF = decltype(bufc)::value;
        const bool more = morec;                         // another group of this work item follows (Always: statically)
        const int slot = gc % kScfSlots;
        const uint32_t sAf = smem_base + slot * kScfSlotBytes + sa_off;   // + 64 c
        const uint32_t tb = tm_rd + BUF * kNT;
        if (epi_tid == 0) stamp(6, gc);
        uint64_t sq[8];                                  // token scales of the chunk, as pairs
        // both halves of a packed operand from one register: ptxas uses the broadcast form of FFMA2 (two registers
        // per group for the row scales instead of four)
        const uint64_t a2 = pack_f2(ab[0], ab[0]), b2 = pack_f2(ab[1], ab[1]);
        uint32_t ok_next = 0;
#ifndef APEX4_X_NOEPI   // experiment builds: the epilogue only hands the buffer back
#pragma unroll
        for (int c = 0; c < kChunks; ++c) {
          uint32_t* vc = v[c % kVBufs];
          // the scales of chunk c (those of chunk c - 1 have been consumed): in flight during the wait
#ifndef APEX4_X_NOLDS
          lds_2x64(sAf + 64 * c, sq[0], sq[1]);
          lds_2x64(sAf + 64 * c + 16, sq[2], sq[3]);
          lds_2x64(sAf + 64 * c + 32, sq[4], sq[5]);
          lds_2x64(sAf + 64 * c + 48, sq[6], sq[7]);
#else
          if (c == 0) { lds_2x64(sAf, sq[0], sq[1]); sq[2] = sq[0]; sq[3] = sq[1]; sq[4] = sq[0]; sq[5] = sq[1]; sq[6] = sq[0]; sq[7] = sq[1]; }
#endif
          if (c == (kChunks >= 3 ? kChunks - 3 : 0) && more) {
            // poll the next group's barriers well ahead of their use
            const uint32_t gn = gc + 1;
            ok_next = mbar_test_wait(bar(bAccFull + (BUF ^ 1) * kHalves + hsel), (fullph >> (BUF ^ 1)) & 1);
            if (kScfSync) ok_next &= mbar_test_wait(bar(bScfFull + gn % kScfSlots), (gn / kScfSlots) & 1);
          }
#ifndef APEX4_X_NOLDTM
          tmem_ld_wait16(vc);
          if (kVBufs == 2 && c < kChunks - 1) tmem_ld_32x16(tb + 16 * (c + 1), v[(c + 1) % kVBufs]);
#endif
#if !defined(APEX4_X_NOSTTM) && !defined(APEX4_X_BIASSLICE)
          if constexpr (BIAS) {
            tmem_st_32x8(tb + 16 * c, mg);
            tmem_st_32x8(tb + 16 * c + 8, mg);
          }
#endif
          if (c == kChunks - 1) {                        // buffer fully read (and re-armed): hand it back
#ifndef APEX4_X_BIASSLICE
            if constexpr (BIAS) tmem_st_wait();
#endif
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(bar(bAccEmpty + BUF * kHalves + hsel), 0);
            if (epi_tid == 0) stamp(16, gc);
            // the next group's first chunk goes into v[0] (chunk kChunks - 2 has been consumed) while the
            // FMAs of this group's last chunk run
            if (kVBufs == 2 && more) group_begin(std::integral_constant<uint32_t, (BUF ^ 1)>{}, gc + 1, ab_next, false, ok_next);
          }
          if (c == 0 && epi_tid == 0) stamp(17, gc);
          if constexpr (DUMP) {
            const int gamma = gamma0 + gi;
#pragma unroll
            for (int j = 0; j < 16; ++j) {
              const int m = m_glob0 + 16 * c + j;
              const int n = n_glob0;
              if (m >= p.pm0 && m < p.pm1 && n >= p.pn0 && n < p.pn1) {
                const uint32_t x = vc[j];
                const int32_t raw = static_cast<int32_t>(BIAS ? x - kBiasInt : x);
                p.P_out[(static_cast<size_t>(m - p.pm0) * (p.pn1 - p.pn0) + (n - p.pn0)) * p.G + gamma] = raw >> 8;
              }
            }
          }
#ifdef APEX4_X_NOFMA
          acc[c * 8] ^= pack_u2(vc[0] ^ vc[5] ^ vc[10] ^ vc[15], vc[3]) ^ sq[0] ^ sq[7];
#else
#pragma unroll
          for (int jj = 0; jj < 8; ++jj) {
            uint64_t t0;
            if constexpr (BIAS) {
              t0 = fma2v(pack_u2(vc[2 * jj], vc[2 * jj + 1]), a2, b2);
            } else {
#ifdef APEX4_X_IADDMAGIC   // tuning build: unbiased accumulators, the magic bias added in registers (one integer add per element)
              t0 = fma2v(pack_u2(vc[2 * jj] + kMagicBits, vc[2 * jj + 1] + kMagicBits), a2, b2);
#else
              t0 = mul2(pack_f2(__int2float_rn(static_cast<int>(vc[2 * jj])), __int2float_rn(static_cast<int>(vc[2 * jj + 1]))), a2);
#endif
            }
            fma2_acc(acc[c * 8 + jj], t0, sq[jj]);   // tokens 16 c + 2 jj, + 1
          }
#endif
#ifndef APEX4_X_NOLDTM
          if (kVBufs == 1 && c < kChunks - 1) tmem_ld_32x16(tb + 16 * (c + 1), v[0]);
#endif
          if (kVBufs == 1 && c == kChunks - 1 && more)
            group_begin(std::integral_constant<uint32_t, (BUF ^ 1)>{}, gc + 1, ab_next, false, ok_next);
        }
#else
        (void)sq; (void)sAf; (void)tb; (void)ok_next;
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(bar(bAccEmpty + BUF * kHalves + hsel), 0);
        if (more) group_begin(std::integral_constant<uint32_t, (BUF ^ 1)>{}, gc + 1, ab_next, true, 0);
#endif
        if (kScfSync) {
          __syncwarp();
          if (lane == 0) mbar_arrive(bar(bScfEmpty + slot));
        }
#ifdef APEX4_X_EPIDELAY   // experiment: N idle clocks after every group -- absorbed where the epilogue waits for the MMA warp anyway
        { const long long t_end = clock64() + APEX4_X_EPIDELAY; while (clock64() < t_end) {} }
#endif
        if (epi_tid == 0) stamp(7, gc);
        ++gc;
      };
      if (ngroups > 0) group_begin(std::integral_constant<uint32_t, 0>{}, gc, ab0, true, 0);
      {
        // "a group follows" is a compile-time property of each copy of the body: the steady-state pair of
        // groups is straight-line code (apart from the rare blocking wait), the last one or two are peeled
        constexpr std::integral_constant<uint32_t, 0> B0{};
        constexpr std::integral_constant<uint32_t, 1> B1{};
        int gi = 0;
        if constexpr (!GR::kMultiKb) {                   // (with groups of several k-blocks the epilogue is off the critical path)
          for (; gi + 4 < ngroups; gi += 4) {
            group_body(B0, Always{}, gi, ab0, ab1);
            group_body(B1, Always{}, gi + 1, ab1, ab0);
            group_body(B0, Always{}, gi + 2, ab0, ab1);
            group_body(B1, Always{}, gi + 3, ab1, ab0);
          }
          for (; gi + 2 < ngroups; gi += 2) {
            group_body(B0, Always{}, gi, ab0, ab1);
            group_body(B1, Always{}, gi + 1, ab1, ab0);
          }
        }
        for (; gi < ngroups; gi += 2) {                  // the last one to four groups: "more" at run time
          group_body(B0, gi + 1 < ngroups, gi, ab0, ab1);
          if (gi + 1 < ngroups) group_body(B1, gi + 2 < ngroups, gi + 1, ab1, ab0);
        }
      }

      // ---- a7 (cast + store) or a6 (cross-pair reduce through the FP32 workspace)
      if (epi_tid == 0) stamp(15, item * 4 + 1);
      if (p.Y != nullptr) {
        auto store_tile = [&]() {
          if (!p.out_f32) {
            // FP16 output: the warp's 32 (n) x kEpiCols (m) sub-tile goes through a private shared-memory
            // tile [m][32 n] (16-byte part p of row m stored at p ^ ((m >> 1) & 3)), then out as 16-byte
            // row pieces: 12 STG.128 per thread instead of 96 STG.U16 with 64-bit address arithmetic
            const uint32_t stg = smem_base + offStore + (warp - kEpiWarp0) * kStoreBytes;
#pragma unroll
            for (int x = 0; x < 8 * kChunks; ++x) {       // tokens m = 2 x, 2 x + 1 of the warpgroup's slice, n = lane
              float f0, f1;
              unpack_f2(acc[x], f0, f1);
              const uint32_t a0 = stg + (2 * x) * 64 + (((lane >> 3) ^ (x & 3)) << 4) + 2 * (lane & 7);
              asm volatile("st.shared.b16 [%0], %1;" ::"r"(a0), "h"(__half_as_ushort(__float2half_rn(f0))) : "memory");
              asm volatile("st.shared.b16 [%0], %1;" ::"r"(a0 + 64), "h"(__half_as_ushort(__float2half_rn(f1))) : "memory");
            }
            __syncwarp();
            const int n = (2 * w.nt + static_cast<int>(rank)) * kTileRows + lq * 32 + (lane & 3) * 8;
            __half* ybase = static_cast<__half*>(p.Y) + n;
#pragma unroll
            for (int ps = 0; ps < kEpiCols / 8; ++ps) {
              const int row = ps * 8 + (lane >> 2);
              uint32_t x0, x1, x2, x3;
              lds128(stg + row * 64 + (((lane & 3) ^ ((row >> 1) & 3)) << 4), x0, x1, x2, x3);
              const int m = w.mt * kNT + h * kEpiCols + row;
              if (m < p.M && n < p.N)
                *reinterpret_cast<uint4*>(ybase + static_cast<size_t>(m) * p.N) = make_uint4(x0, x1, x2, x3);
            }
            __syncwarp();
            return;
          }
          float* y = static_cast<float*>(p.Y);      // FP32 output: lanes = consecutive n, coalesced rows
          if (n_glob0 < p.N) {
            if constexpr (PUSH) {   // (its own instantiation: the product kernel's code is untouched)
              // K-split tensor parallelism: the partial tile is added into the buffer of the rank that owns these
              // columns (possibly over NVLink), tile by tile as the GEMM proceeds -- GEMM and reduce-scatter in one kernel
              const int owner = n_glob0 / p.push_cols;
              float* yo = p.push_y[owner] + (n_glob0 - owner * p.push_cols);
#pragma unroll
              for (int x = 0; x < 8 * kChunks; ++x) {
                float f0, f1;
                unpack_f2(acc[x], f0, f1);
                const int m = m_glob0 + 2 * x;
                if (m < p.M) asm volatile("red.relaxed.sys.global.add.f32 [%0], %1;" ::"l"(yo + static_cast<size_t>(m) * p.push_cols), "f"(f0) : "memory");
                if (m + 1 < p.M) asm volatile("red.relaxed.sys.global.add.f32 [%0], %1;" ::"l"(yo + static_cast<size_t>(m + 1) * p.push_cols), "f"(f1) : "memory");
              }
              return;
            }
#pragma unroll
            for (int x = 0; x < 8 * kChunks; ++x) {
              float f0, f1;
              unpack_f2(acc[x], f0, f1);
              const int m = m_glob0 + 2 * x;
              if (m < p.M) y[static_cast<size_t>(m) * p.N + n_glob0] = f0;
              if (m + 1 < p.M) y[static_cast<size_t>(m + 1) * p.N + n_glob0] = f1;
            }
          }
        };
        if (!w.partial) {
          store_tile();
        } else {
          // a6: FP32 partial sums meet in the workspace ("inter-SM global reduction").  The
          // workspace holds one CTA tile per SLOT in FRAGMENT order -- [slot][CTA][j][thread][4 floats] --
          // so a partial tile is fully coalesced red.global.add.v4.f32 per thread (not scalar atomics),
          // and the CTA that completes the tile reads it back with the same thread mapping,
          // leaves it zero-filled, casts and stores.
          // Slot of a shared tile = the pair whose unit range holds the tile's FIRST unit.  Ranges are contiguous, so
          // two shared tiles never have the same first-unit owner (the earlier one would lie wholly inside that
          // pair's range and not be shared): npairs slots suffice, whatever M and N are.
          const long long first_unit = static_cast<long long>(w.nt * p.tiles_m + w.mt) * p.upt;
          const long long total_units = static_cast<long long>(p.tiles_m) * p.tiles_n * p.upt;
          const int slot = static_cast<int>(((first_unit + 1) * static_cast<int>(gridDim.x >> 1) - 1) / total_units);
          float* wst = p.ws + static_cast<size_t>(slot * 2 + static_cast<int>(rank)) * (kTileRows * kNT) + epi_tid * 4;
#pragma unroll
          for (int j = 0; j < 4 * kChunks; ++j) {
            float f0, f1, f2, f3;
            unpack_f2(acc[2 * j], f0, f1);
            unpack_f2(acc[2 * j + 1], f2, f3);
            asm volatile("red.relaxed.gpu.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(wst + j * (128 * kEpiWarps)), "f"(f0),
                         "f"(f1), "f"(f2), "f"(f3)
                         : "memory");
          }
          __threadfence();
          if (epi_tid == 0) stamp(15, item * 4 + 2);
          int* flag = reinterpret_cast<int*>(smem_gen + offTmemPtr + 8);
          asm volatile("bar.sync 1, %0;" ::"n"(32 * kEpiWarps) : "memory");
          if (epi_tid == 0) {
            const int cslot = slot * 2 + static_cast<int>(rank);
            const int prev = atomicAdd(p.counters + cslot, w.units);
            const int done = (prev + w.units == p.upt);
            *flag = done;
            if (done) p.counters[cslot] = 0;
          }
          asm volatile("bar.sync 1, %0;" ::"n"(32 * kEpiWarps) : "memory");
          const int done = *flag;
          asm volatile("bar.sync 1, %0;" ::"n"(32 * kEpiWarps) : "memory");   // flag may be rewritten by the next item
          if (done) {
            __threadfence();
#pragma unroll
            for (int j = 0; j < 4 * kChunks; ++j) {       // all loads first, then the zero stores
              const float4 x = __ldcg(reinterpret_cast<const float4*>(wst + j * (128 * kEpiWarps)));
              acc[2 * j] = pack_f2(x.x, x.y);
              acc[2 * j + 1] = pack_f2(x.z, x.w);
            }
#pragma unroll
            for (int j = 0; j < 4 * kChunks; ++j) __stcg(reinterpret_cast<float4*>(wst + j * (128 * kEpiWarps)), make_float4(0.f, 0.f, 0.f, 0.f));
            store_tile();
          }
        }
      }
      if (epi_tid == 0) stamp(15, item * 4 + 3);
      ++item;
    }
    tc_fence_before();
  }

  // ---- teardown: nobody leaves while the peer may still signal this CTA's barriers or read its
  // shared memory / TMEM through the pair MMA
#ifdef APEX4_TIMELINE
  if (p.tl != nullptr && blockIdx.x < 2 && (threadIdx.x & 31) == 0) p.tl[(blockIdx.x * 32 + 19) * 64 + (threadIdx.x >> 5)] = clock64();   // per warp: done
#endif
  cluster_sync_all();
#ifdef APEX4_TIMELINE
  if (p.tl != nullptr && blockIdx.x < 2 && threadIdx.x == 0) p.tl[(blockIdx.x * 32 + 18) * 64 + 3] = clock64();
#endif
  if (warp == kCtlWarp0 + 1) {
    tc_fence_after();
    tmem_dealloc_pair<512>(tmem_base);
  }
}

// ------------------------------------------------------------------------------------ launcher
template <int MODE, bool DUMP, int NT, bool PUSH = false>
static cudaError_t launch_pair_one(const GemmParams& p, int npairs, cudaStream_t st) {
  auto kern = w4a4_gemm_pair_kernel<MODE, DUMP, NT, PUSH>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Tile<NT>::kSmemBytes);
  if (e != cudaSuccess) return e;
#ifdef APEX4_X_NOPDL
  kern<<<2 * npairs, Warps<widen_wgs<MODE, NT>(), Tile<NT>::kEpiWGs>::kThreads, Tile<NT>::kSmemBytes, st>>>(p);
  return cudaGetLastError();
#else
  e = launch_pdl(kern, dim3(2 * npairs), dim3(Warps<widen_wgs<MODE, NT>(), Tile<NT>::kEpiWGs>::kThreads), Tile<NT>::kSmemBytes, st, p);
  return e != cudaSuccess ? e : cudaGetLastError();
#endif
}

// defined (explicitly instantiated) in apex4_gemm_pair_m<MODE>.cu
template <int MODE>
cudaError_t launch_pair_mode(const GemmParams& p, bool dump, int npairs, cudaStream_t st);

#define APEX4_PAIR_INSTANTIATE(MODE)                                                                     \
  template <>                                                                                            \
  cudaError_t launch_pair_mode<MODE>(const GemmParams& p, bool dump, int npairs, cudaStream_t st) {      \
    if (p.push && !dump) {                                                                               \
      switch (p.pair_nt) {                                                                               \
        case 64: return launch_pair_one<MODE, false, 64, true>(p, npairs, st);                           \
        case 128: return launch_pair_one<MODE, false, 128, true>(p, npairs, st);                         \
        case kPairTokens: return launch_pair_one<MODE, false, kPairTokens, true>(p, npairs, st);         \
        default: return cudaErrorInvalidValue;                                                           \
      }                                                                                                  \
    }                                                                                                    \
    switch (p.pair_nt) {                                                                                 \
      case 64: return dump ? launch_pair_one<MODE, true, 64>(p, npairs, st) : launch_pair_one<MODE, false, 64>(p, npairs, st);   \
      case 128: return dump ? launch_pair_one<MODE, true, 128>(p, npairs, st) : launch_pair_one<MODE, false, 128>(p, npairs, st); \
      case kPairTokens:                                                                                  \
        return dump ? launch_pair_one<MODE, true, kPairTokens>(p, npairs, st) : launch_pair_one<MODE, false, kPairTokens>(p, npairs, st); \
      default: return cudaErrorInvalidValue;                                                             \
    }                                                                                                    \
  }

}  // namespace apex4
