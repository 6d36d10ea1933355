// apex4_gemm_pair_m1.cu -- the CTA-pair kernel of apex4_gemm_pair.cuh instantiated for granularity MODE 1
// (g = 64); one translation unit per mode so that they compile in parallel.
#include "apex4_gemm_pair.cuh"

namespace apex4 {
APEX4_PAIR_INSTANTIATE(1)
}  // namespace apex4
