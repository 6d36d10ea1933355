// apex4_layout.cuh -- the two opaque device layouts of include/apex4.h, stated once.
//
// PT4 (packed INT4 codes).  Operand Q[R,K], rows padded to Rp = roundup(R,128), K % 128 == 0.
//   blob(rt, kb) = 128 rows x 128 k, 8192 contiguous bytes at ((rt * K/128 + kb) * 8192).
//   Row rr of a blob = 64 bytes = 4 chunks of 16 bytes = 16 words of 32 bits.
//   The GEMM widens a packed word w into two INT8 words  lo = (w << 4) & 0xF0F0F0F0  and
//   hi = w & 0xF0F0F0F0  (each byte = 16 * code, sign correct) and stores chunk j's four lo words as
//   physical 16-byte chunk 2j and its four hi words as physical chunk 2j+1 of the row's 128-byte
//   INT8 line.  The tensor core reads that line through the 128-byte swizzle, which maps logical
//   chunk c of row rr to physical chunk c ^ (rr & 7).  The packer pre-applies the inverse so that
//   logical INT8 byte p of the line is element k = kb*128 + p for every row:
//       c = p >> 4, y = p & 15, pc = c ^ (rr & 7), j = pc >> 1, h = pc & 1
//       code(rr, kb*128 + p) lives in blob byte  rr*64 + j*16 + y,  nibble h (0 = low, 1 = high).
//   (Any order inside a K=32 slice would give the same integer sums; identity keeps g=32 simple.)
//
// PW4 (packed INT4 weight codes).  Same blobs, same sizes.  The GEMM's widener thread r reads its own
//   64-byte row, widens it in registers and stores the 32 INT8 words to TMEM, where the tensor core
//   reads the A operand as: 32-bit column c of lane r = k bytes 4c..4c+3 of the k-block.  Logical
//   chunk j (= the K=32 slice j of the k-block) holds element k = kb*128 + 32j + p in byte p & 15,
//   nibble p >> 4.  Only the 16-byte chunk SLOT is permuted, slot = j ^ ((rr >> 1) & 3), so that the
//   128-bit loads of eight consecutive rows cover all 32 banks.
//
// ST16 (FP16 scales).  [Rp/128][G][128]: element (r, gamma) at ((r/128)*G + gamma)*128 + r%128, so
//   the scales of one 128-row tile for consecutive groups are one contiguous bulk copy.
#pragma once
#include <stddef.h>
#include <stdint.h>

namespace apex4 {

constexpr int kTileRows = 128;   // rows per blob / per TMEM lane set
constexpr int kBlockK = 128;     // k per blob = one 128-byte INT8 swizzle line
constexpr int kBlobBytes = kTileRows * kBlockK / 2;   // 8192
constexpr int kRowBytes = kBlockK / 2;                // 64

__host__ __device__ inline int round_up(int x, int m) { return (x + m - 1) / m * m; }

__host__ __device__ inline size_t pt4_bytes(int R, int K) {
  return static_cast<size_t>(round_up(R, kTileRows) / kTileRows) * (K / kBlockK) * kBlobBytes;
}
__host__ __device__ inline size_t pt4_blob_offset(int rt, int kb, int K) {
  return (static_cast<size_t>(rt) * (K / kBlockK) + kb) * kBlobBytes;
}
__host__ __device__ inline size_t st16_elems(int R, int G) {
  return static_cast<size_t>(round_up(R, kTileRows)) * G;
}
__host__ __device__ inline size_t st16_index(int r, int gamma, int G) {
  return (static_cast<size_t>(r / kTileRows) * G + gamma) * kTileRows + (r % kTileRows);
}

}  // namespace apex4
