// apex4_gemm_pair.cu -- host side of the CTA-pair kernel (apex4_gemm_pair.cuh): picks the granularity MODE
// instantiation and answers how many CTA pairs can be resident.
#include "apex4_gemm_pair.cuh"

namespace apex4 {

cudaError_t launch_gemm_pair(const GemmParams& p, bool dump, int npairs, cudaStream_t st) {
  switch (gran_mode(p.g)) {
    case 0: return launch_pair_mode<0>(p, dump, npairs, st);
    case 1: return launch_pair_mode<1>(p, dump, npairs, st);
    case 2: return launch_pair_mode<2>(p, dump, npairs, st);
    default: return launch_pair_mode<3>(p, dump, npairs, st);
  }
}

// declared here, defined in apex4_gemm_pair_m3.cu (it needs a kernel symbol for the occupancy query)
int gemm_max_pairs_query();

// CTA pairs that can be resident at once (one per TPC); queried once
int gemm_max_pairs() {
  static int pairs = 0;
  if (pairs == 0) pairs = gemm_max_pairs_query();
  return pairs;
}

}  // namespace apex4
