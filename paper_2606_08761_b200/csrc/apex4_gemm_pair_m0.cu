// apex4_gemm_pair_m0.cu -- the CTA-pair kernel of apex4_gemm_pair.cuh instantiated for granularity MODE 0
// (g = 128); one translation unit per mode so that they compile in parallel.
#include "apex4_gemm_pair.cuh"

namespace apex4 {
APEX4_PAIR_INSTANTIATE(0)
}  // namespace apex4
