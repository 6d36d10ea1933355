// apex4_gemm_pair_m3.cu -- the CTA-pair kernel of apex4_gemm_pair.cuh instantiated for granularity MODE 3
// (g = 128 j > 128, up to per-channel); one translation unit per mode so that they compile in parallel.
#include "apex4_gemm_pair.cuh"

namespace apex4 {
APEX4_PAIR_INSTANTIATE(3)

int gemm_max_pairs_query() {
  auto kern = w4a4_gemm_pair_kernel<3, false, kPairTokens>;   // one CTA per SM whatever the mode
  int n = 0;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(2 * 74);
  cfg.blockDim = dim3(Warps<Gran<3>::kWidenWGs, Tile<kPairTokens>::kEpiWGs>::kThreads);
  cfg.dynamicSmemBytes = Tile<kPairTokens>::kSmemBytes;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Tile<kPairTokens>::kSmemBytes) != cudaSuccess ||
      cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess || n <= 0) {
    cudaGetLastError();
    n = 74;   // B200: 148 SMs, one CTA pair per TPC
  }
  return n;
}
}  // namespace apex4
