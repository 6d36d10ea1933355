// apex4_api.cu -- the C ABI of include/apex4.h: argument validation, granularity policy (a8),
// choice of token-tile width and work distribution (whole tiles / stream-K) for the GEMM kernel.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "../../include/apex4.h"
#include "apex4_gemm.cuh"
#include "apex4_layout.cuh"

namespace apex4 {
cudaError_t launch_quantize(const void* x, int R, int K, int g, void* q, void* s, int weights,
                            cudaStream_t st);
bool quantize_supports_group(int g);
cudaError_t launch_rmsnorm_quantize(const void* x, const void* gamma, float eps, int R, int K, int g, void* q, void* s, void* y_out,
                                    cudaStream_t st);
cudaError_t launch_silu_mul_quantize(const void* gate, const void* up, int ld, int R, int K, int g, void* q, void* s, void* y_out,
                                     cudaStream_t st);
cudaError_t launch_pack_codes(const int8_t* codes, int R, int K, void* q, int weights, cudaStream_t st);
cudaError_t launch_unpack_codes(const void* q, int R, int K, int8_t* codes, int weights, cudaStream_t st);
cudaError_t launch_scales_from_natural(const void* nat, int R, int G, void* tiled, cudaStream_t st);
cudaError_t launch_scales_to_natural(const void* tiled, int R, int G, void* nat, cudaStream_t st);
int measure_rho(double* out, cudaStream_t st);
int measure_epilogue_pipes(double* out, cudaStream_t st);
int measure_epilogue_stream(double* out, cudaStream_t st);
int e4m3_exactness(int K, int pattern, int encoding, uint32_t seed, double* out, cudaStream_t st);
}  // namespace apex4

using namespace apex4;

namespace {

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

int check_arch() {
  static int cached = -1;
  if (cached >= 0) return cached;
  int dev = 0, major = 0, minor = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return APEX4_ERR_CUDA;
  if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev) != cudaSuccess)
    return APEX4_ERR_CUDA;
  cached = (major == 10 && minor == 0) ? APEX4_OK : APEX4_ERR_ARCH;
  return cached;
}

// a8: group size from (K, group_size, gran, layer).  PAPER.md:162-166, 183; reading R11.
int resolve_g(int K, int group_size, int gran, int layer) {
  if (K <= 0 || K % kBlockK != 0) return -APEX4_ERR_UNSUPPORTED_SHAPE;
  if (layer < APEX4_LAYER_OTHER || layer > APEX4_LAYER_DOWN) return -APEX4_ERR_INVALID_ARG;
  int g;
  switch (gran) {
    case APEX4_GRAN_GROUP: g = group_size; break;
    case APEX4_GRAN_CHANNEL: g = K; break;
    case APEX4_GRAN_MIXED:
      g = (layer == APEX4_LAYER_V || layer == APEX4_LAYER_DOWN) ? 32 : K;
      break;
    case APEX4_GRAN_MIXED_G128:
      g = (layer == APEX4_LAYER_V || layer == APEX4_LAYER_DOWN) ? 128 : K;
      break;
    default: return -APEX4_ERR_INVALID_ARG;
  }
  if (g <= 0) return -APEX4_ERR_INVALID_ARG;
  const bool ok = (g == 32 || g == 64 || (g % kBlockK == 0)) && (K % g == 0);
  if (!ok) return -APEX4_ERR_UNSUPPORTED_SHAPE;
  if (!quantize_supports_group(g)) return -APEX4_ERR_UNSUPPORTED_SHAPE;
  return g;
}

struct Dispatch {
  int kernel;  // 0 = decode (weight-stream) kernel, 1 = CTA-pair tcgen05 kernel
  int split;   // pair kernel: stream-K work distribution (needs the workspace)
  int grid;    // CTAs (decode) or CTA pairs (pair kernel)
  int upt, kbu, tiles_m, tiles_n;
  int mt;      // decode kernel: m16 token tiles
  int pnt;     // pair kernel: tokens per pair tile (64 / 128 / kPairTokens)
};

// "automatic" values of apex4_debug_opts
const apex4_debug_opts kAuto = {-1, 0, -1, 0, 0, nullptr};

// Tokens per pair tile: columns past M are wasted epilogue / MMA work, but a 128-token tile costs ~1.1 x
// a 192-token tile per token (measured at N = K = 8192, g = 128: M = 1024 110.1 vs 111.5 us, M = 512 60.3 vs 65.4 us,
// M = 256 32.6 vs 41.6 us, M = 4096 the 192-token tile).  M <= 64: the 64-token tile; up to 128 tokens it also wins
// while all its tiles still fit one wave (M = 128, N = 8192: 24.6 us against 26.0 us on one 128-token tile row).
// Groups of several k-blocks (g > 128) are tensor-bound, not epilogue-bound: there a 128-token tile costs ~1.2 x a
// 192-token tile per token (M = 1024 per-channel: 78.2 vs 71.6 us), so it is taken only when it saves more than that.
int pair_tokens(int M, int N, int g, const apex4_debug_opts& o) {
  if (o.pair_tokens > 0) return o.pair_tokens;
  if (M <= 64) return 64;
  const int tiles_n = (N + 2 * kTileRows - 1) / (2 * kTileRows);
  if (M <= 128 && 2 * tiles_n <= gemm_max_pairs()) return 64;
  const int r128 = (M + 127) / 128 * 128, r192 = (M + kPairTokens - 1) / kPairTokens * kPairTokens;
  return (g > kBlockK ? 6 * r128 < 5 * r192 : 11 * r128 < 10 * r192) ? 128 : kPairTokens;
}

// The decode kernel covers M <= 32 at g = 32 / 64 / 128, per-channel, and the group sizes in between whose
// groups nest with its 16 warps' k ranges (one rounding per group, R12: their INT32 sums are combined before scaling).
bool decode_supported(int M, int K, int g) {
  if (M > 32) return false;
  if (g == K && K <= kBlockK) return g == kBlockK;
  return gemv_group_mode(K, g) >= 0;
}

int sm_count() {
  static int sms = 0;
  if (sms == 0) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0)
      sms = 148;
  }
  return sms;
}

// Pure function of the problem and the (per-call) debug options: no process-global state.
// Returns false when the options ask for a kernel that does not cover the problem.
bool choose_dispatch(int M, int N, int K, int g, const apex4_debug_opts& o, Dispatch& d) {
  memset(&d, 0, sizeof(d));
  const int KB = K / kBlockK;
  d.kbu = g > kBlockK ? g / kBlockK : 1;   // indivisible k unit: a whole group, at least a k-block
  d.upt = KB / d.kbu;
  const bool dec_ok = decode_supported(M, K, g);
  if (o.kernel == 0 && !dec_ok) return false;
  if (o.kernel > 1 || o.kernel < -1) return false;
  d.kernel = o.kernel >= 0 ? o.kernel : (dec_ok ? 0 : 1);
  if (d.kernel == 0) {
    // a CTA owns a contiguous range of 8-row row blocks and all of K; no workspace
    d.mt = (M + 15) / 16;
    d.tiles_m = 1;
    d.tiles_n = (N + 7) / 8;
    d.grid = o.grid > 0 ? o.grid : sm_count();
    if (d.grid > d.tiles_n) d.grid = d.tiles_n;
    const int per_cta = (d.tiles_n + d.grid - 1) / d.grid;
    const int max_batch = gemv_max_batch(d.mt);
    d.upt = per_cta < max_batch ? per_cta : max_batch;     // row blocks per shared-memory batch
    if (o.decode_batch > 0 && o.decode_batch < d.upt) d.upt = o.decode_batch;
    return true;
  }
  d.pnt = pair_tokens(M, N, g, o);
  if (d.pnt != 64 && d.pnt != 128 && d.pnt != kPairTokens) return false;
  d.tiles_m = (M + d.pnt - 1) / d.pnt;
  d.tiles_n = (N + 2 * kTileRows - 1) / (2 * kTileRows);
  const long long tiles = static_cast<long long>(d.tiles_m) * d.tiles_n;
  const long long units = tiles * d.upt;
  const int max_grid = gemm_max_pairs();
  const int sms = (o.grid > 0 && o.grid < max_grid) ? o.grid : max_grid;
  d.grid = static_cast<int>(units < sms ? units : sms);
  // whole tiles per CTA pair when the last wave is reasonably full, stream-K otherwise
  const long long waves = (tiles + d.grid - 1) / d.grid;
  const double eff = static_cast<double>(tiles) / static_cast<double>(waves * d.grid);
  // a single, reasonably full wave is cheaper as whole tiles than as stream-K ranges (each partial range
  // pays a reduction and a pipeline restart: M = 256, N = K = 8192 57.7 us whole vs 61.5 us split)
  d.split = (o.split >= 0) ? (o.split ? 1 : 0) : ((eff < 0.93 && !(waves == 1 && eff >= 0.8)) ? 1 : 0);
  if (d.upt == 1) d.split = 0;                      // nothing to split
  if (!d.split && tiles < d.grid) d.grid = static_cast<int>(tiles);
  return true;
}

// Stream-K workspace: one slot per CTA pair (a shared tile's slot is the pair that owns its first unit, see the
// kernel), each an arrival counter per CTA and a 256 x pnt FP32 tile -- independent of M and N.
size_t counters_bytes(const Dispatch& d) {
  return (static_cast<size_t>(d.grid) * 2 * 4 + 255) / 256 * 256;
}

cudaError_t launch_dispatch(const GemmParams& p, const Dispatch& d, bool dump, cudaStream_t st) {
  const cudaError_t e = d.kernel == 1 ? launch_gemm_pair(p, dump, d.grid, st) : launch_gemv(p, d.mt, dump, d.grid, st);
  if (e != cudaSuccess && getenv("APEX4_VERBOSE"))
    fprintf(stderr, "apex4: GEMM launch (kernel %d, grid %d) failed: %s\n", d.kernel, d.grid, cudaGetErrorString(e));
  return e;
}
size_t workspace_need(const Dispatch& d) {
  if (!d.split) return 0;
  // per slot a 256 x pnt pair tile as FP32 in fragment order, after the arrival counters
  return counters_bytes(d) + static_cast<size_t>(d.grid) * 256 * d.pnt * 4;
}

int validate_gemm_shape(int M, int N, int K) {
  if (M < 1 || N < 1 || K < 1) return APEX4_ERR_INVALID_ARG;
  if (K % kBlockK != 0 || N % 8 != 0 || K > 32768) return APEX4_ERR_UNSUPPORTED_SHAPE;
  return APEX4_OK;
}

}  // namespace

extern "C" {

const char* apex4_status_string(int status) {
  switch (status) {
    case APEX4_OK: return "ok";
    case APEX4_ERR_INVALID_ARG: return "invalid argument";
    case APEX4_ERR_UNSUPPORTED_SHAPE: return "unsupported shape or group size";
    case APEX4_ERR_ALIGNMENT: return "pointer not 16-byte aligned";
    case APEX4_ERR_WORKSPACE: return "workspace missing or too small";
    case APEX4_ERR_CUDA: return "CUDA error";
    case APEX4_ERR_ARCH: return "device is not sm_100a (compute capability 10.0)";
    default: return "unknown status";
  }
}

int apex4_resolve_group_size(int K, int group_size, int gran, int layer) {
  return resolve_g(K, group_size, gran, layer);
}

size_t apex4_packed_bytes(int R, int K) {
  if (R < 1 || K < 1 || K % kBlockK != 0) return 0;
  return pt4_bytes(R, K);
}
size_t apex4_scale_elems(int R, int K, int g) {
  if (R < 1 || K < 1 || g < 1 || K % g != 0) return 0;
  return st16_elems(R, K / g);
}

size_t apex4_workspace_bytes_ex(int M, int N, int K, int group_size, int gran, int layer,
                                const apex4_debug_opts* opts) {
  if (validate_gemm_shape(M, N, K) != APEX4_OK) return 0;
  const int g = resolve_g(K, group_size, gran, layer);
  if (g < 0) return 0;
  Dispatch d;
  if (!choose_dispatch(M, N, K, g, opts ? *opts : kAuto, d)) return 0;
  return workspace_need(d);
}
size_t apex4_workspace_bytes(int M, int N, int K, int group_size, int gran, int layer) {
  return apex4_workspace_bytes_ex(M, N, K, group_size, gran, layer, nullptr);
}

static int quantize_common(const void* x, int R, int K, int group_size, int gran, int layer, void* q,
                           void* s, int weights, void* stream) {
  if (!x || !q || !s || R < 1 || K < 1) return APEX4_ERR_INVALID_ARG;
  if (K > 32768) return APEX4_ERR_UNSUPPORTED_SHAPE;
  const int g = resolve_g(K, group_size, gran, layer);
  if (g < 0) return -g;
  if (!aligned16(x) || !aligned16(q) || !aligned16(s)) return APEX4_ERR_ALIGNMENT;
  const int a = check_arch();
  if (a != APEX4_OK) return a;
  return launch_quantize(x, R, K, g, q, s, weights, static_cast<cudaStream_t>(stream)) == cudaSuccess
             ? APEX4_OK
             : APEX4_ERR_CUDA;
}

int apex4_quantize_act(const void* x_f16, int M, int K, int group_size, int gran, int layer,
                       void* qA_packed, void* sA_f16, void* stream) {
  return quantize_common(x_f16, M, K, group_size, gran, layer, qA_packed, sA_f16, 0, stream);
}
int apex4_pack_weights(const void* w_f16, int N, int K, int group_size, int gran, int layer,
                       void* qW_packed, void* sW_f16, void* stream) {
  return quantize_common(w_f16, N, K, group_size, gran, layer, qW_packed, sW_f16, 1, stream);
}

int apex4_rmsnorm_quantize(const void* x_f16, const void* gamma_f16, float eps, int M, int K, int group_size, int gran,
                           int layer, void* qA_packed, void* sA_f16, void* y_f16_out, void* stream) {
  if (!x_f16 || !gamma_f16 || !qA_packed || !sA_f16 || M < 1 || K < 1 || !(eps >= 0.f)) return APEX4_ERR_INVALID_ARG;
  if (K > 32768) return APEX4_ERR_UNSUPPORTED_SHAPE;
  const int g = resolve_g(K, group_size, gran, layer);
  if (g < 0) return -g;
  if (!aligned16(x_f16) || !aligned16(gamma_f16) || !aligned16(qA_packed) || !aligned16(sA_f16) || !aligned16(y_f16_out))
    return APEX4_ERR_ALIGNMENT;
  const int a = check_arch();
  if (a != APEX4_OK) return a;
  return launch_rmsnorm_quantize(x_f16, gamma_f16, eps, M, K, g, qA_packed, sA_f16, y_f16_out, static_cast<cudaStream_t>(stream)) ==
                 cudaSuccess
             ? APEX4_OK
             : APEX4_ERR_CUDA;
}

int apex4_silu_mul_quantize(const void* gate_f16, const void* up_f16, int ld, int M, int K, int group_size, int gran, int layer,
                            void* qA_packed, void* sA_f16, void* y_f16_out, void* stream) {
  if (!gate_f16 || !up_f16 || !qA_packed || !sA_f16 || M < 1 || K < 1 || ld < K) return APEX4_ERR_INVALID_ARG;
  if (K > 32768) return APEX4_ERR_UNSUPPORTED_SHAPE;
  const int g = resolve_g(K, group_size, gran, layer);
  if (g < 0) return -g;
  if (!aligned16(gate_f16) || !aligned16(up_f16) || (ld % 8) != 0 || !aligned16(qA_packed) || !aligned16(sA_f16) ||
      !aligned16(y_f16_out))
    return APEX4_ERR_ALIGNMENT;
  const int a = check_arch();
  if (a != APEX4_OK) return a;
  return launch_silu_mul_quantize(gate_f16, up_f16, ld, M, K, g, qA_packed, sA_f16, y_f16_out, static_cast<cudaStream_t>(stream)) ==
                 cudaSuccess
             ? APEX4_OK
             : APEX4_ERR_CUDA;
}

int apex4_pack_codes(const int8_t* codes, int R, int K, int operand, void* q_packed, void* stream) {
  if (!codes || !q_packed || R < 1 || K < 1) return APEX4_ERR_INVALID_ARG;
  if (operand != APEX4_OPERAND_ACT && operand != APEX4_OPERAND_WEIGHT) return APEX4_ERR_INVALID_ARG;
  if (K % kBlockK != 0) return APEX4_ERR_UNSUPPORTED_SHAPE;
  if (!aligned16(codes) || !aligned16(q_packed)) return APEX4_ERR_ALIGNMENT;
  const int a = check_arch();
  if (a != APEX4_OK) return a;
  return launch_pack_codes(codes, R, K, q_packed, operand, static_cast<cudaStream_t>(stream)) == cudaSuccess
             ? APEX4_OK
             : APEX4_ERR_CUDA;
}
int apex4_unpack_codes(const void* q_packed, int R, int K, int operand, int8_t* codes, void* stream) {
  if (!codes || !q_packed || R < 1 || K < 1) return APEX4_ERR_INVALID_ARG;
  if (operand != APEX4_OPERAND_ACT && operand != APEX4_OPERAND_WEIGHT) return APEX4_ERR_INVALID_ARG;
  if (K % kBlockK != 0) return APEX4_ERR_UNSUPPORTED_SHAPE;
  if (!aligned16(codes) || !aligned16(q_packed)) return APEX4_ERR_ALIGNMENT;
  const int a = check_arch();
  if (a != APEX4_OK) return a;
  return launch_unpack_codes(q_packed, R, K, codes, operand, static_cast<cudaStream_t>(stream)) == cudaSuccess
             ? APEX4_OK
             : APEX4_ERR_CUDA;
}
int apex4_scales_from_natural(const void* s_nat, int R, int G, void* s_tiled, void* stream) {
  if (!s_nat || !s_tiled || R < 1 || G < 1) return APEX4_ERR_INVALID_ARG;
  const int a = check_arch();
  if (a != APEX4_OK) return a;
  return launch_scales_from_natural(s_nat, R, G, s_tiled, static_cast<cudaStream_t>(stream)) ==
                 cudaSuccess
             ? APEX4_OK
             : APEX4_ERR_CUDA;
}
int apex4_scales_to_natural(const void* s_tiled, int R, int G, void* s_nat, void* stream) {
  if (!s_nat || !s_tiled || R < 1 || G < 1) return APEX4_ERR_INVALID_ARG;
  const int a = check_arch();
  if (a != APEX4_OK) return a;
  return launch_scales_to_natural(s_tiled, R, G, s_nat, static_cast<cudaStream_t>(stream)) ==
                 cudaSuccess
             ? APEX4_OK
             : APEX4_ERR_CUDA;
}

static void fill_params(GemmParams& p, const Dispatch& d, const void* qA, const void* sA,
                        const void* qW, const void* sW, int M, int N, int K, int g) {
  memset(&p, 0, sizeof(p));
  p.qW = static_cast<const uint8_t*>(qW); p.sW = static_cast<const __half*>(sW);
  p.qA = static_cast<const uint8_t*>(qA); p.sA = static_cast<const __half*>(sA);
  p.M = M; p.N = N; p.K = K; p.g = g; p.G = K / g;
  p.tiles_m = d.tiles_m; p.tiles_n = d.tiles_n;
  p.split = d.split; p.upt = d.upt; p.kbu = d.kbu; p.pair_nt = d.pnt;
}

int apex4_w4a4_gemm_ex(const void* qA_packed, const void* sA_f16, const void* qW_packed,
                       const void* sW_f16, void* Y, int out_dtype, int M, int N, int K, int group_size,
                       int gran, int layer, void* workspace, size_t workspace_bytes, void* stream,
                       const apex4_debug_opts* opts) {
  if (!qA_packed || !sA_f16 || !qW_packed || !sW_f16 || !Y) return APEX4_ERR_INVALID_ARG;
  if (out_dtype != APEX4_OUT_F16 && out_dtype != APEX4_OUT_F32) return APEX4_ERR_INVALID_ARG;
  int v = validate_gemm_shape(M, N, K);
  if (v != APEX4_OK) return v;
  const int g = resolve_g(K, group_size, gran, layer);
  if (g < 0) return -g;
  if (!aligned16(qA_packed) || !aligned16(sA_f16) || !aligned16(qW_packed) || !aligned16(sW_f16) ||
      !aligned16(Y))
    return APEX4_ERR_ALIGNMENT;
  const int a = check_arch();
  if (a != APEX4_OK) return a;
  Dispatch d;
  if (!choose_dispatch(M, N, K, g, opts ? *opts : kAuto, d)) return APEX4_ERR_INVALID_ARG;
  GemmParams p;
  fill_params(p, d, qA_packed, sA_f16, qW_packed, sW_f16, M, N, K, g);
  p.Y = Y; p.out_f32 = (out_dtype == APEX4_OUT_F32);
  p.tl = opts ? static_cast<long long*>(opts->timeline) : nullptr;   // read by -DAPEX4_TIMELINE builds only
  if (d.split) {
    if (!workspace || workspace_bytes < workspace_need(d) || !aligned16(workspace))
      return APEX4_ERR_WORKSPACE;
    p.counters = static_cast<int*>(workspace);
    p.ws = reinterpret_cast<float*>(static_cast<uint8_t*>(workspace) + counters_bytes(d));
  }
  return launch_dispatch(p, d, false, static_cast<cudaStream_t>(stream)) == cudaSuccess
             ? APEX4_OK
             : APEX4_ERR_CUDA;
}

int apex4_w4a4_gemm_tp_push(const void* qA_packed, const void* sA_f16, const void* qW_packed, const void* sW_f16,
                            void* const* owner_y_f32, int world, int M, int N, int K_local, int group_size, int gran,
                            int layer, void* workspace, size_t workspace_bytes, void* stream) {
  if (!qA_packed || !sA_f16 || !qW_packed || !sW_f16 || !owner_y_f32) return APEX4_ERR_INVALID_ARG;
  if (world < 1 || world > kMaxPushRanks) return APEX4_ERR_INVALID_ARG;
  int v = validate_gemm_shape(M, N, K_local);
  if (v != APEX4_OK) return v;
  if (N % world != 0 || (N / world) % 8 != 0) return APEX4_ERR_UNSUPPORTED_SHAPE;   // whole 8-column pieces per owner
  const int g = resolve_g(K_local, group_size, gran, layer);
  if (g < 0) return -g;
  if (!aligned16(qA_packed) || !aligned16(sA_f16) || !aligned16(qW_packed) || !aligned16(sW_f16)) return APEX4_ERR_ALIGNMENT;
  for (int r = 0; r < world; ++r)
    if (!owner_y_f32[r] || !aligned16(owner_y_f32[r])) return owner_y_f32[r] ? APEX4_ERR_ALIGNMENT : APEX4_ERR_INVALID_ARG;
  const int a = check_arch();
  if (a != APEX4_OK) return a;
  Dispatch d;
  if (!choose_dispatch(M, N, K_local, g, kAuto, d)) return APEX4_ERR_INVALID_ARG;
  GemmParams p;
  fill_params(p, d, qA_packed, sA_f16, qW_packed, sW_f16, M, N, K_local, g);
  p.Y = owner_y_f32[0];   // non-null: "there is an output"; the push path never stores through it
  p.out_f32 = 1;
  p.push = 1;
  p.push_cols = N / world;
  for (int r = 0; r < world; ++r) p.push_y[r] = static_cast<float*>(owner_y_f32[r]);
  if (d.split) {
    if (!workspace || workspace_bytes < workspace_need(d) || !aligned16(workspace)) return APEX4_ERR_WORKSPACE;
    p.counters = static_cast<int*>(workspace);
    p.ws = reinterpret_cast<float*>(static_cast<uint8_t*>(workspace) + counters_bytes(d));
  }
  return launch_dispatch(p, d, false, static_cast<cudaStream_t>(stream)) == cudaSuccess ? APEX4_OK : APEX4_ERR_CUDA;
}

int apex4_w4a4_gemm(const void* qA_packed, const void* sA_f16, const void* qW_packed,
                    const void* sW_f16, void* Y, int out_dtype, int M, int N, int K, int group_size,
                    int gran, int layer, void* workspace, size_t workspace_bytes, void* stream) {
  return apex4_w4a4_gemm_ex(qA_packed, sA_f16, qW_packed, sW_f16, Y, out_dtype, M, N, K, group_size, gran,
                            layer, workspace, workspace_bytes, stream, nullptr);
}

int apex4_debug_group_sums(const void* qA_packed, const void* qW_packed, int M, int N, int K,
                           int group_size, int gran, int layer, int m0, int m1, int n0, int n1,
                           int32_t* P_out, void* stream, const apex4_debug_opts* opts) {
  if (!qA_packed || !qW_packed || !P_out) return APEX4_ERR_INVALID_ARG;
  int v = validate_gemm_shape(M, N, K);
  if (v != APEX4_OK) return v;
  if (m0 < 0 || m1 > M || m0 >= m1 || n0 < 0 || n1 > N || n0 >= n1) return APEX4_ERR_INVALID_ARG;
  const int g = resolve_g(K, group_size, gran, layer);
  if (g < 0) return -g;
  const int a = check_arch();
  if (a != APEX4_OK) return a;
  Dispatch d;
  if (!choose_dispatch(M, N, K, g, opts ? *opts : kAuto, d)) return APEX4_ERR_INVALID_ARG;
  d.split = 0;   // the dump needs every tile's groups in one CTA (pair); the decode kernel never splits
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  // the decode kernel adds its warps' partial group sums into P_out
  if (cudaMemsetAsync(P_out, 0, static_cast<size_t>(m1 - m0) * (n1 - n0) * (K / g) * sizeof(int32_t), st) != cudaSuccess)
    return APEX4_ERR_CUDA;
  GemmParams p;
  // no scales: the DUMP kernels neither copy nor read them
  fill_params(p, d, qA_packed, nullptr, qW_packed, nullptr, M, N, K, g);
  p.Y = nullptr; p.P_out = P_out; p.pm0 = m0; p.pm1 = m1; p.pn0 = n0; p.pn1 = n1;
  return launch_dispatch(p, d, true, st) == cudaSuccess ? APEX4_OK : APEX4_ERR_CUDA;
}

static size_t align256(size_t x) { return (x + 255) / 256 * 256; }

static size_t host_ws_bytes(int M, int N, int K, int g) {
  Dispatch d;
  if (!choose_dispatch(M, N, K, g, kAuto, d)) return 0;
  return align256(workspace_need(d));
}

size_t apex4_linear_host_scratch_bytes(int M, int N, int K, int group_size, int gran, int layer) {
  if (validate_gemm_shape(M, N, K) != APEX4_OK) return 0;
  const int g = resolve_g(K, group_size, gran, layer);
  if (g < 0) return 0;
  return host_ws_bytes(M, N, K, g) + align256(static_cast<size_t>(M) * K * 2) + align256(pt4_bytes(M, K)) +
         align256(st16_elems(M, K / g) * 2) + align256(static_cast<size_t>(M) * N * 4);
}

int apex4_w4a4_linear_host(const void* x_host_f16, const void* qW_packed, const void* sW_f16,
                           void* y_host, int M, int N, int K, int group_size, int gran, int layer,
                           int out_dtype, void* scratch, size_t scratch_bytes, void* stream) {
  if (!x_host_f16 || !qW_packed || !sW_f16 || !y_host || !scratch) return APEX4_ERR_INVALID_ARG;
  int v = validate_gemm_shape(M, N, K);
  if (v != APEX4_OK) return v;
  const int g = resolve_g(K, group_size, gran, layer);
  if (g < 0) return -g;
  if (scratch_bytes < apex4_linear_host_scratch_bytes(M, N, K, group_size, gran, layer) ||
      !aligned16(scratch))
    return APEX4_ERR_WORKSPACE;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  uint8_t* base = static_cast<uint8_t*>(scratch);
  uint8_t* ws = base;   // the GEMM workspace comes first so that it stays zero-filled across calls
  const size_t ws_bytes = host_ws_bytes(M, N, K, g);
  uint8_t* xd = ws + ws_bytes;
  uint8_t* qa = xd + align256(static_cast<size_t>(M) * K * 2);
  uint8_t* sa = qa + align256(pt4_bytes(M, K));
  uint8_t* yd = sa + align256(st16_elems(M, K / g) * 2);
  const size_t ybytes = static_cast<size_t>(M) * N * (out_dtype == APEX4_OUT_F32 ? 4 : 2);
  if (cudaMemcpyAsync(xd, x_host_f16, static_cast<size_t>(M) * K * 2, cudaMemcpyHostToDevice, st) != cudaSuccess)
    return APEX4_ERR_CUDA;
  int rc = apex4_quantize_act(xd, M, K, group_size, gran, layer, qa, sa, stream);
  if (rc != APEX4_OK) return rc;
  rc = apex4_w4a4_gemm(qa, sa, qW_packed, sW_f16, yd, out_dtype, M, N, K, group_size, gran, layer,
                       ws_bytes ? ws : nullptr, ws_bytes, stream);
  if (rc != APEX4_OK) return rc;
  if (cudaMemcpyAsync(y_host, yd, ybytes, cudaMemcpyDeviceToHost, st) != cudaSuccess) return APEX4_ERR_CUDA;
  return APEX4_OK;
}

int apex4_debug_get_dispatch(int M, int N, int K, int group_size, int gran, int layer,
                             const apex4_debug_opts* opts, int* out5) {
  if (!out5) return APEX4_ERR_INVALID_ARG;
  if (validate_gemm_shape(M, N, K) != APEX4_OK) return APEX4_ERR_UNSUPPORTED_SHAPE;
  const int g = resolve_g(K, group_size, gran, layer);
  if (g < 0) return -g;
  Dispatch d;
  if (!choose_dispatch(M, N, K, g, opts ? *opts : kAuto, d)) return APEX4_ERR_INVALID_ARG;
  out5[0] = d.kernel; out5[1] = d.kernel == 1 ? d.pnt : 16 * d.mt; out5[2] = d.split; out5[3] = d.grid; out5[4] = d.upt;
  return APEX4_OK;
}

int apex4_e4m3_exactness(int K, int pattern, int encoding, unsigned seed, double* out_host, void* stream) {
  if (!out_host || pattern < 0 || pattern > 5 || (encoding != 0 && encoding != 1)) return APEX4_ERR_INVALID_ARG;
  if (K < kBlockK || K % kBlockK != 0 || K > 32768) return APEX4_ERR_UNSUPPORTED_SHAPE;
  const int a = check_arch();
  if (a != APEX4_OK) return a;
  return e4m3_exactness(K, pattern, encoding, seed, out_host, static_cast<cudaStream_t>(stream));
}

int apex4_measure_epilogue_pipes(double* out_host, void* stream) {
  if (!out_host) return APEX4_ERR_INVALID_ARG;
  const int a = check_arch();
  if (a != APEX4_OK) return a;
  return measure_epilogue_pipes(out_host, static_cast<cudaStream_t>(stream));
}

int apex4_measure_epilogue_stream(double* out_host, void* stream) {
  if (!out_host) return APEX4_ERR_INVALID_ARG;
  const int a = check_arch();
  if (a != APEX4_OK) return a;
  return measure_epilogue_stream(out_host, static_cast<cudaStream_t>(stream));
}

int apex4_measure_rho(double* out_host, void* stream) {
  if (!out_host) return APEX4_ERR_INVALID_ARG;
  const int a = check_arch();
  if (a != APEX4_OK) return a;
  return measure_rho(out_host, static_cast<cudaStream_t>(stream));
}

}  // extern "C"
