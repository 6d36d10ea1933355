// apex4_gemm.cuh -- parameters shared by the GEMM kernel file and the C-ABI dispatch.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace apex4 {

// The kernel works on two abstract operands, both in PT4/ST16 layout:
//   "R side" = tcgen05 A operand: 128-row tiles -> TMEM lanes (one epilogue thread per row)
//   "C side" = tcgen05 B operand: NC-row tiles  -> TMEM columns
// Normal orientation (swap = 0): R = activations (rows m), C = weights (rows n), Y[r, c].
// Swapped (swap = 1, decode-sized M): R = weights (rows n), C = activations (rows m), Y[c, r].
struct GemmParams {
  const uint8_t* qR;
  const __half* sR;
  const uint8_t* qC;
  const __half* sC;
  void* Y;
  int out_f32;
  int R, C;        // logical row counts of the two operands
  int K, g, G;
  int ldY;         // N (row pitch of Y in elements)
  int swap;
  int splits;      // split-K factor (grid.z); 1 = direct store
  int kb_per_split;
  float* ws;       // split-K: FP32 partial sums [M, N], zero on entry, zero on exit
  int* counters;   // split-K: one arrival counter per (r tile, c tile), zero on entry/exit
  int32_t* P_out;  // debug dump of per-group INT32 sums (DUMP kernels only)
  int pm0, pm1, pn0, pn1;
};

cudaError_t launch_gemm(const GemmParams& p, int nc, bool dump, cudaStream_t st);

}  // namespace apex4
