// apex4_gemm.cuh -- parameters shared by the GEMM kernel file and the C-ABI dispatch.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace apex4 {

// Both GEMM kernels run "weights on the rows": the pair kernel puts 256 weight rows (n) on the TMEM lanes
// of a CTA pair and NT token rows (m) on the accumulator columns; weights (PW4/ST16) are the tcgen05 A
// operand (widened in registers, stored to TMEM), activations (PT4/ST16) the B operand (widened in shared
// memory).  The decode kernel streams 8-row weight groups against one or two m16 token tiles.
struct GemmParams {
  const uint8_t* qW;   // PW4  [Np/128][K/128][8192]
  const __half* sW;    // ST16 [Np/128][G][128]
  const uint8_t* qA;   // PT4  [Mp/128][K/128][8192]
  const __half* sA;    // ST16 [Mp/128][G][128]
  void* Y;             // [M, N] row-major, FP16 or FP32; nullptr for the debug dump
  int out_f32;
  int M, N, K, g, G;
  int tiles_m, tiles_n;   // pair kernel: ceil(M / pair_nt), ceil(N / 256); decode: 1, ceil(N / 8)
  // work distribution (a6 / PAPER.md:226-230): split = 0 -> CTA c owns whole tiles c, c + grid, ...;
  // split = 1 -> the K loop of all tiles is one line of `units` dealt to the CTAs in equal contiguous
  // ranges (stream-K); a unit is kbu k-blocks (one group when g >= 128), a tile has upt units.
  int split, upt, kbu;
  int pair_nt;         // pair kernel: tokens per tile (64 / 128 / kPairTokens)
  float* ws;           // split = 1: FP32 partial sums, every pair tile in fragment order; zero on entry, zero on exit
  int* counters;       // split = 1: finished units per tile, zero on entry/exit
  int32_t* P_out;      // debug dump of the per-group INT32 sums (DUMP kernels only)
  int pm0, pm1, pn0, pn1;
  long long* tl;       // -DAPEX4_TIMELINE builds only: clock64 stamps of CTA 0, [event][64]; else unused
  // Tensor-parallel K-split (apex4_w4a4_gemm_tp_push): instead of storing Y the epilogue ADDS its FP32 partial tile
  // into the owner's accumulation buffer -- output column n belongs to rank n / push_cols, whose buffer
  // push_y[rank] is [M, push_cols] FP32 row-major and may be peer memory mapped over NVLink (red.global.add.f32).
  int push, push_cols;
  float* push_y[8];
};
constexpr int kMaxPushRanks = 8;

// Launch with programmatic stream serialization (PDL): the kernel may start while its predecessor on the
// stream drains; it calls griddep_wait() (apex4_ptx.cuh) before it touches anything the predecessor wrote.
template <class... KArgs, class... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, args...);
}

constexpr int kPairTokens = 192;   // tokens per CTA-pair tile (the widest; 128 / 64 where M is small)

// Tensor-bound regime (apex4_gemm_pair.cu): CTA pairs (cluster of 2, cta_group::2), work tile = 256
// weight rows x p.pair_nt tokens; tiles_m / tiles_n / counters are in units of pair tiles (counters: two per
// tile, one per CTA of the pair).  npairs <= gemm_max_pairs().
cudaError_t launch_gemm_pair(const GemmParams& p, bool dump, int npairs, cudaStream_t st);
int gemm_max_pairs();

// Decode regime (apex4_gemv.cu): M <= 32 at g = 32 / 64 / 128 or per-channel, no workspace.  tiles_n = 8-row
// row blocks, upt = row blocks per shared-memory batch (<= gemv_max_batch(mt)), kbu = k-blocks per group.
cudaError_t launch_gemv(const GemmParams& p, int mt, bool dump, int grid, cudaStream_t st);
int gemv_max_batch(int mt);
int gemv_group_mode(int K, int g);   // >= 0: the decode kernel covers this (K, g); -1: it does not

}  // namespace apex4
