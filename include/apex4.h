/* apex4.h -- C ABI of the B200-native APEX4 W4A4 hot path (arxiv/paper_2606_08761).
 *
 * What the library computes (citations are /root/reference/PAPER.md lines):
 *   Eq. 7  symmetric INT4 group quantizer
 *        S = fp16(absmax / 7),  q = clamp(rne(x / S), -8, 7),  scales kept in FP16
 *   Eq. 8  group-dequantised GEMM
 *        Y[m,n] = sum_g sA[m,g] * sW[n,g] * (sum_{k in g} qA[m,k] * qW[n,k])
 *        exact INT32 partial sums per K-group on the tensor cores (tcgen05.mma kind::i8,
 *        operands widened INT4->INT8 on chip because sm_100a has no 4-bit integer MMA kind:
 *        weights in registers -> TMEM, activations shared -> shared memory), INT32->FP32 + scale
 *        multiply on the CUDA cores, FP32 accumulation.
 *   3.2.2  granularity: uniform g, per-channel (g = K), mixed policy.
 *
 * Conventions
 *   - Every pointer is a DEVICE pointer unless its comment says HOST.  The caller allocates and owns
 *     every buffer; the library never allocates, frees or keeps a pointer after the call returns.
 *   - Every call only enqueues work on `stream` (a cudaStream_t passed as void*, NULL = default
 *     stream) and never synchronises (except apex4_measure_rho and the *_host helpers, which say so).
 *   - Return value: an apex4_status.  Arguments are validated before anything is launched; a failed
 *     launch returns APEX4_ERR_CUDA.  Nothing aborts the host and nothing is printed unless the
 *     environment variable APEX4_VERBOSE is set (one stderr line per failed launch).  Every in-kernel
 *     barrier wait is bounded: a phase bug traps silently and surfaces as APEX4_ERR_CUDA / a sticky CUDA
 *     error, never as a hang.
 *   - No process-global state: the library keeps only two lazily filled read-only caches (SM count,
 *     resident CTA pairs).  Every call is a pure function of its arguments; concurrent calls on
 *     different streams are safe when they use different workspaces.
 *   - Determinism: integer stages are exact.  FP32 summation order is fixed except where three or more
 *     stream-K ranges meet in one output tile (FP32 atomics): such outputs can differ in the last bits
 *     between runs, inside the R12 tolerance of DESIGN.md.
 *   - Shapes: X[M,K], W[N,K], Y[M,N] dense row-major (last index contiguous).  K % 128 == 0,
 *     N % 8 == 0, M >= 1.  Group size g: 32, 64, or a multiple of 128 that divides K (128, 256, 512,
 *     1024, ..., K).  Pointers 16-byte aligned.  (SURVEY 8(b) asks for K % 32; the blob layout below
 *     is built from 128-k blocks, and every K of BASELINE.json's configs is a multiple of 128.)
 *   - Device layouts (opaque to the caller; sizes from the *_bytes queries below):
 *       packed codes  "PT4": rows padded to Rp = roundup(R,128); blob (rt, kb) of 128 rows x 128 k
 *                     = 8192 contiguous bytes at ((rt * K/128 + kb) * 8192); inside a blob row r
 *                     occupies 64 bytes and its 16-byte chunks / nibbles are permuted so that the
 *                     in-kernel widening lands directly in the 128B-swizzled UMMA operand layout
 *                     (see csrc/apex4_layout.cuh).  apex4_unpack_codes inverts it.
 *                     "PW4" (weights): same blobs and sizes, a different permutation inside a row
 *                     (the weights are widened in registers and stored to TMEM).  A buffer packed
 *                     as one operand kind must be used as that kind.
 *       scales        "ST16": FP16, tile-major [Rp/128][G][128], G = K/g: element (r, gamma) at
 *                     ((r/128) * G + gamma) * 128 + r % 128.  apex4_scales_to_natural inverts it.
 */
#ifndef APEX4_H_
#define APEX4_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  APEX4_OK = 0,
  APEX4_ERR_INVALID_ARG = 1,       /* null pointer, non-positive size, unknown enum */
  APEX4_ERR_UNSUPPORTED_SHAPE = 2, /* K % 128, N % 8, group size not supported / not dividing K */
  APEX4_ERR_ALIGNMENT = 3,         /* a pointer is not 16-byte aligned */
  APEX4_ERR_WORKSPACE = 4,         /* workspace NULL or smaller than apex4_workspace_bytes() */
  APEX4_ERR_CUDA = 5,              /* a CUDA runtime call / kernel launch failed */
  APEX4_ERR_ARCH = 6               /* device is not compute capability 10.0 (sm_100a) */
} apex4_status;

/* granularity mode: how group_size is resolved */
typedef enum {
  APEX4_GRAN_GROUP = 0,      /* g = group_size */
  APEX4_GRAN_CHANNEL = 1,    /* g = K (one scale per token row / per output channel), group_size ignored */
  APEX4_GRAN_MIXED = 2,      /* paper's mix: down_proj, v_proj -> 32; every other layer -> K */
  APEX4_GRAN_MIXED_G128 = 3  /* BASELINE.json wording: the fine layers at 128, others per-channel */
} apex4_gran;

typedef enum {
  APEX4_LAYER_OTHER = 0, APEX4_LAYER_Q = 1, APEX4_LAYER_K = 2, APEX4_LAYER_V = 3, APEX4_LAYER_QKV = 4,
  APEX4_LAYER_O = 5, APEX4_LAYER_GATE = 6, APEX4_LAYER_UP = 7, APEX4_LAYER_GATE_UP = 8,
  APEX4_LAYER_DOWN = 9
} apex4_layer;

typedef enum { APEX4_OUT_F16 = 0, APEX4_OUT_F32 = 1 } apex4_out;

/* which GEMM operand a packed-code buffer belongs to (selects the PT4 or the PW4 layout) */
typedef enum { APEX4_OPERAND_ACT = 0, APEX4_OPERAND_WEIGHT = 1 } apex4_operand;

/* Per-call verification / tuning options of the *_ex and debug exports (NULL = automatic everywhere).
 * They replace any global "force this kernel" switch: the library has no mutable state. */
typedef struct {
  int kernel;        /* -1 automatic, 0 decode (weight-stream) kernel, 1 CTA-pair tcgen05 kernel */
  int pair_tokens;   /* 0 automatic, else 64 / 128 / 192 tokens per pair tile */
  int split;         /* -1 automatic, 0 whole tiles per CTA pair, 1 stream-K (a6) */
  int grid;          /* 0 automatic, else CTAs (decode) / CTA pairs to launch (capped at what fits) */
  int decode_batch;  /* 0 automatic, else 8-row weight blocks per shared-memory batch of the decode kernel */
  void* timeline;    /* device buffer for clock stamps; read only by -DAPEX4_TIMELINE builds */
} apex4_debug_opts;

/* ---- host-side queries (no kernel launches; the first call of apex4_workspace_bytes reads two device
 *      attributes) ----------------------------------------------------------------------------- */

/* Group size a call with these arguments runs at, or a negative apex4_status on invalid input.
 * PAPER.md:162-166, 183.  Pure host function. */
int apex4_resolve_group_size(int K, int group_size, int gran, int layer);

/* Bytes of the PT4 packed-code buffer for an operand with R rows (M for activations, N for weights).
 * (SURVEY 8(b) calls this apex4_packed_weight_bytes; one query serves both operands here.) */
size_t apex4_packed_bytes(int R, int K);
/* Number of FP16 elements of the ST16 scale buffer for R rows at resolved group size g. */
size_t apex4_scale_elems(int R, int K, int g);
/* Bytes of DEVICE workspace apex4_w4a4_gemm needs for this problem.  0 when every output tile is
 * computed by one CTA (pair) alone: the decode kernels (M <= 32 at g <= 128 or per-channel) and any tile count that
 * fills the SMs evenly.  Otherwise (stream-K, a6) it holds, per CTA pair of the launch, two arrival counters and
 * one 256 x tile-width FP32 tile for the output tile that pair shares with its successors: at most ~14.6 MB on a
 * B200 (74 pairs x 256 x 192 x 4 B), independent of M and N.  The workspace must be zero-filled
 * once by the caller before its first use; every call leaves it zero-filled again, so one buffer
 * serves any sequence of calls on one stream.  Concurrent calls on different streams need their own. */
size_t apex4_workspace_bytes(int M, int N, int K, int group_size, int gran, int layer);
/* The same for a call that passes `opts` to apex4_w4a4_gemm_ex. */
size_t apex4_workspace_bytes_ex(int M, int N, int K, int group_size, int gran, int layer,
                                const apex4_debug_opts* opts);

const char* apex4_status_string(int status);

/* ---- a1: online activation quantizer (Eq. 7) -------------------------- */
/* x_f16 [M,K] FP16 -> qA_packed (PT4, apex4_packed_bytes(M,K)) + sA_f16 (ST16, apex4_scale_elems). */
int apex4_quantize_act(const void* x_f16, int M, int K, int group_size, int gran, int layer,
                       void* qA_packed, void* sA_f16, void* stream);

/* ---- a1 fused into its producer ("quantized online") ------------------------- */
/* The two ops that feed the linears of a Llama / Qwen block, with the quantizer of Eq. 7 applied to their FP16
 * result before it ever reaches HBM.  Outputs are exactly apex4_quantize_act of that FP16 result (same layouts,
 * same sizes); y_f16_out, if not NULL, also receives the FP16 result [M,K] (verification, residual paths).
 *   apex4_rmsnorm_quantize:  y = fp16( (x * inv) * gamma ),  inv = 1.0f / sqrtf( float(sum_k x^2 / K) + eps ),
 *       the sum of squares exact, every other step one IEEE binary32 operation (R17).  gamma_f16 [K].
 *   apex4_silu_mul_quantize: y = fp16( silu(gate) * up ), silu(g) = g / (1 + exp(-g)), the real-valued product
 *       rounded once (R18).  gate_f16 / up_f16 [M,K] with row stride ld >= K elements (ld % 8 == 0), so
 *       the two halves of a fused gate+up GEMM output [M, 2K] can be passed as (Y, Y + K, ld = 2K). */
int apex4_rmsnorm_quantize(const void* x_f16, const void* gamma_f16, float eps, int M, int K, int group_size,
                           int gran, int layer, void* qA_packed, void* sA_f16, void* y_f16_out, void* stream);
int apex4_silu_mul_quantize(const void* gate_f16, const void* up_f16, int ld, int M, int K, int group_size,
                            int gran, int layer, void* qA_packed, void* sA_f16, void* y_f16_out, void* stream);

/* ---- a0: offline weight quantize + pack (Eq. 7) --------------------------- */
/* w_f16 [N,K] FP16 -> qW_packed (PW4) + sW_f16 (ST16). Same arithmetic as the activation quantizer. */
int apex4_pack_weights(const void* w_f16, int N, int K, int group_size, int gran, int layer,
                       void* qW_packed, void* sW_f16, void* stream);
/* Offline-calibrated path (Alg. 1 output): codes [R,K] int8 in [-8,7] (row-major)
 * -> PT4 (operand = APEX4_OPERAND_ACT) or PW4 (APEX4_OPERAND_WEIGHT).  Values outside [-8,7] are
 * taken modulo 16 (low nibble).  (apex4_pack_weights_from_codes; its scales go through
 * apex4_scales_from_natural.  apex4_unpack_codes below is SURVEY 8(b)'s apex4_unpack_weights.) */
int apex4_pack_codes(const int8_t* codes, int R, int K, int operand, void* q_packed, void* stream);
/* natural FP16 scales [R,G] row-major -> ST16 (padding rows zero-filled), and back. */
int apex4_scales_from_natural(const void* s_nat_f16, int R, int G, void* s_tiled_f16, void* stream);
int apex4_scales_to_natural(const void* s_tiled_f16, int R, int G, void* s_nat_f16, void* stream);
/* PT4 / PW4 (per `operand`) -> codes [R,K] int8 (verification twin of the packers). */
int apex4_unpack_codes(const void* q_packed, int R, int K, int operand, int8_t* codes, void* stream);

/* ---- a2..a7: the W4A4 group-dequant GEMM (Eq. 8) ----------------------------- */
/* Y [M,N] (FP16 or FP32 per out_dtype) = sum_g sA sW P_g.  qA/sA from apex4_quantize_act, qW/sW
 * from apex4_pack_weights, both at the same resolved group size (G_a = G_w).
 * workspace: apex4_workspace_bytes() bytes of DEVICE memory (may be NULL when that is 0); it is used
 * when the K loop of an output tile is shared between CTAs (a6: a tile count that
 * does not fill the SMs evenly).  A smaller workspace_bytes returns APEX4_ERR_WORKSPACE and launches
 * nothing. */
int apex4_w4a4_gemm(const void* qA_packed, const void* sA_f16, const void* qW_packed,
                    const void* sW_f16, void* Y, int out_dtype, int M, int N, int K, int group_size,
                    int gran, int layer, void* workspace, size_t workspace_bytes, void* stream);
/* The same call with per-call options (tests force every kernel / tile width / work distribution with it;
 * opts == NULL is apex4_w4a4_gemm).  Options that the problem does not admit (the decode kernel for
 * M > 32 or a group size it does not cover) return APEX4_ERR_INVALID_ARG. */
int apex4_w4a4_gemm_ex(const void* qA_packed, const void* sA_f16, const void* qW_packed,
                       const void* sW_f16, void* Y, int out_dtype, int M, int N, int K, int group_size,
                       int gran, int layer, void* workspace, size_t workspace_bytes, void* stream,
                       const apex4_debug_opts* opts);

/* ---- K-split (row-parallel) tensor parallelism, the reduce-scatter fused into the GEMM ------ */
/* This rank holds the K-slice [k0, k1) of X and W (cut on group boundaries: qA/sA from apex4_quantize_act on the
 * slice, qW/sW packed from the slice, K_local = k1 - k0).  Output column n belongs to rank n / (N / world);
 * owner_y_f32[r] (a HOST array of `world` DEVICE pointers) is rank r's FP32 accumulation buffer [M, N / world]
 * row-major -- this rank's own memory for r == rank, peer memory mapped over NVLink (CUDA IPC / cudaMemcpyPeer-
 * capable mapping, P2P access enabled) for the others.  The epilogue of the GEMM kernels ADDS each finished
 * FP32 partial tile into its owner's buffer with red.global.add.f32 (system scope) as the tiles complete, so the
 * exchange overlaps the math tile by tile: one kernel is GEMM + reduce-scatter; no Y is stored.
 * Protocol (the caller's, e.g. paper_2606_08761_b200/tp.py): every rank zero-fills its own buffer; barrier; every
 * rank calls this; barrier (after stream completion); each rank reads / casts its [M, N / world] slice.
 * N % world == 0, (N / world) % 8 == 0, world <= 8; workspace as for apex4_w4a4_gemm at (M, N, K_local).
 * Per-group integer sums are those of the single-GPU path; only the FP32 summation order over ranks (and
 * tiles, atomics) varies -- inside the output tolerance (R12), not bitwise reproducible. */
int apex4_w4a4_gemm_tp_push(const void* qA_packed, const void* sA_f16, const void* qW_packed, const void* sW_f16,
                            void* const* owner_y_f32, int world, int M, int N, int K_local, int group_size, int gran,
                            int layer, void* workspace, size_t workspace_bytes, void* stream);

/* The same GEMM for callers that cannot allocate device memory (CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the stream-K workspace comes from a static __device__ array of
 * APEX4_STATIC_WORKSPACE_BYTES inside the library (held by every GPU that loads the library until the process
 * exits) instead of from the caller.  The call allocates and frees nothing; kernels, dispatch and results are those
 * of apex4_w4a4_gemm (bit-identical).  A problem whose apex4_workspace_bytes() exceeds
 * APEX4_STATIC_WORKSPACE_BYTES returns APEX4_ERR_WORKSPACE and launches nothing (use apex4_w4a4_gemm with your own
 * workspace); with one workspace slot per CTA pair that cannot happen on a 148-SM B200 (<= 14.6 MB), it is the
 * guard for devices with more SMs.  All calls share the one array: the bytes a call needs are cleared on `stream` before its launch, and
 * calls that OVERLAP on the GPU (different streams without a dependency, or concurrent host threads on different
 * streams) race on it -- serialise them.  Per device: the array's address is resolved on first use with that device
 * current. */
#define APEX4_STATIC_WORKSPACE_BYTES (16u << 20)
int apex4_w4a4_gemm_static_ws(const void* qA_packed, const void* sA_f16, const void* qW_packed,
                              const void* sW_f16, void* Y, int out_dtype, int M, int N, int K, int group_size,
                              int gran, int layer, void* stream);

/* End-to-end convenience over the three calls above with HOST activations and HOST output:
 * x_host_f16 [M,K] (HOST, pinned for true asynchrony) -> cudaMemcpyAsync -> apex4_quantize_act ->
 * apex4_w4a4_gemm (weights qW/sW pre-packed on the DEVICE) -> cudaMemcpyAsync -> y_host [M,N] (HOST).
 * scratch: DEVICE memory of apex4_linear_host_scratch_bytes() bytes, zero-filled once by the caller
 * (its head is the GEMM workspace) and reusable across calls of the same shape.  Enqueues only. */
size_t apex4_linear_host_scratch_bytes(int M, int N, int K, int group_size, int gran, int layer);
int apex4_w4a4_linear_host(const void* x_host_f16, const void* qW_packed, const void* sW_f16,
                           void* y_host, int M, int N, int K, int group_size, int gran, int layer,
                           int out_dtype, void* scratch, size_t scratch_bytes, void* stream);

/* Verification export: the exact per-group INT32 sums P[m,n,gamma] the tensor cores produced, for the
 * window m in [m0,m1), n in [n0,n1): P_out [(m1-m0), (n1-n0), G] int32 row-major.  Runs the same
 * kernel as apex4_w4a4_gemm would for (M, N, K, g, opts) -- same tiles, same pipeline, whole tiles per
 * CTA pair -- with the accumulators dumped by the epilogue instead of dequantised; takes no scales.
 * P_out is zero-filled by the call (cudaMemsetAsync on `stream`) before the kernel runs. */
int apex4_debug_group_sums(const void* qA_packed, const void* qW_packed, int M, int N, int K,
                           int group_size, int gran, int layer, int m0, int m1, int n0, int n1,
                           int32_t* P_out, void* stream, const apex4_debug_opts* opts);
/* Host-side: what a call with these arguments launches.  out5 (HOST) = {kernel (0 decode, 1 pair),
 * token-tile width, stream-K flag, CTAs or CTA pairs, k units per tile / row blocks per batch}. */
int apex4_debug_get_dispatch(int M, int N, int K, int group_size, int gran, int layer,
                             const apex4_debug_opts* opts, int* out5);

/* ---- rho microbenchmark (Eq. 1-2; Table 1) -------------------- */
/* Measures on the current device: dense INT8 tcgen05.mma rate (TOPS), FP32 FMA rate (TFLOPS),
 * INT32->FP32 conversion rate (Gop/s) and rho = int8_tops / fp32_tflops.  (SURVEY 8(b) gives this call four
 * double* outputs; one array carries them and the raw per-SM-per-clock figures.)  out[] is a HOST array of
 * at least 8 doubles: {int8_tops, fp32_tflops, i2f_gops, rho, tmem_ld_gbs, sm_clock_mhz, int8_mac_per_clk_per_sm,
 * tmem_ld_bytes_per_clk_per_sm}.
 * Synchronises the stream; allocates and frees its own small device scratch (the only call that
 * does). */
int apex4_measure_rho(double* out_host, void* stream);

/* The Blackwell form of the paper's Tensor-Core / CUDA-Core tension inside the epilogue (a5): how much the TMEM
 * <-> register traffic of the dequant step (tcgen05.ld of the accumulators, tcgen05.st of the magic bias) and its
 * FP32 FMAs slow each other down on one SM.  out_host (HOST, >= 16 doubles): for mode m = 1..7 (bit 0 loads, bit 1
 * stores, bit 2 FFMA2) out[2m] = clocks a TMEM warp needs per 16 accumulator columns, out[2m+1] = clocks an FFMA2
 * warp needs per 32 FFMA2 (the FMAs of 16 columns), two warps of each kind per SM sub-partition.  Synchronises the
 * stream; allocates and frees ~2 KB of device scratch. */
int apex4_measure_epilogue_pipes(double* out_host, void* stream);

/* The epilogue's own instruction stream in isolation: eight warps per SM take a 192-column accumulator buffer
 * through registers as the pair kernel's group loop does (tcgen05.ld double-buffered, the tcgen05.st re-bias, token
 * scales from shared memory, two FMAs per element on 96 accumulators per thread) with no barriers, no MMA, no
 * wideners.  out_host (HOST, >= 8 doubles): clocks per group for {loads, loads + stores, loads + FMAs,
 * loads + stores + FMAs, loads + scale loads + FMAs, everything, and -- for the alternative tcgen05.ld.16x256b fragment
 * layout (four rows x four tokens per thread and chunk: a quarter of the token-scale loads) -- loads, everything}.  The gap between out[5] and the pair
 * kernel's measured group period is what the epilogue loses to the warps it shares a sub-partition with and to the
 * accumulator hand-off.  Synchronises the stream; allocates and frees ~1 KB of device scratch. */
int apex4_measure_epilogue_stream(double* out_host, void* stream);

/* ---- experiment: is an FP8 tensor-core path exact on INT4 codes? ------------------------------- */
/* Runs one 128 x 256 tile over K (multiple of 128, <= 32768) through tcgen05.mma kind::i8 and through
 * kind::f8f6f4 with the same codes as E4M3 operands and compares the two TMEM accumulators element by element.
 * pattern: 0 uniform codes, 1 all -8, 2 alternating 7 / -8, 3 large sums with odd increments, 4 random signs at
 * +-7, 5 deterministic ramp.  encoding: 0 = codes as normal E4M3 numbers, 1 = sign | magnitude (E4M3 subnormals,
 * value code * 2^-9).  out_host (HOST, >= 5 doubles) = {mismatching elements, max |fp32 - int|, max |int sum|,
 * elements compared, mismatches of the INT8 sums against 64 K (pattern 1 only)}.  Synchronises the stream and
 * allocates / frees 40 bytes of device scratch.  Not a product path: apex4_w4a4_gemm always uses kind::i8. */
int apex4_e4m3_exactness(int K, int pattern, int encoding, unsigned seed, double* out_host, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* APEX4_H_ */
