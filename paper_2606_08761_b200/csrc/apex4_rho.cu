// apex4_rho.cu -- measures this GPU's own rho (Eq. 1-2; Table 1):
// tensor-core throughput (dense INT8 tcgen05.mma kind::i8, the pipe the W4A4 path runs on, since
// sm_100a has no 4-bit integer MMA) against CUDA-core throughput (FP32 FMA), plus the two other
// rates that bound the dequant step a5: INT32->FP32 conversion and TMEM read bandwidth.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/apex4.h"
#include "apex4_ptx.cuh"

namespace apex4 {

constexpr int kChains = 8;

__global__ void __launch_bounds__(256) fma_rate_kernel(float* out, int iters, float b, float c) {
  float a[kChains];
#pragma unroll
  for (int j = 0; j < kChains; ++j) a[j] = threadIdx.x * 0.001f + j;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int j = 0; j < kChains; ++j) a[j] = fmaf(a[j], b, c);
  }
  float s = 0.f;
#pragma unroll
  for (int j = 0; j < kChains; ++j) s += a[j];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(256) fma2_rate_kernel(float* out, int iters, float b, float c) {
  uint64_t a[kChains];
  const uint64_t b2 = pack_f2(b, b), c2 = pack_f2(c, c);
#pragma unroll
  for (int j = 0; j < kChains; ++j) a[j] = pack_f2(threadIdx.x * 0.001f + j, 1.f + j);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int j = 0; j < kChains; ++j) a[j] = fma2(a[j], b2, c2);
  }
  float s = 0.f;
#pragma unroll
  for (int j = 0; j < kChains; ++j) { float lo, hi; unpack_f2(a[j], lo, hi); s += lo + hi; }
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(256) i2f_rate_kernel(float* out, int iters) {
  int x[kChains];
#pragma unroll
  for (int j = 0; j < kChains; ++j) x[j] = threadIdx.x * 7 + j;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int j = 0; j < kChains; ++j) x[j] = __float_as_int(__int2float_rn(x[j]));
  }
  int s = 0;
#pragma unroll
  for (int j = 0; j < kChains; ++j) s ^= x[j];
  out[blockIdx.x * blockDim.x + threadIdx.x] = __int_as_float(s);
}

// One CTA per SM: a single thread issues back-to-back 128x256x32 INT8 MMAs from resident shared
// memory into two alternating TMEM accumulators; four warps then stream the accumulators out with
// tcgen05.ld to time TMEM reads.
constexpr int kMmaSmem = 1024 + 16384 + 32768 + 64;
__global__ void __launch_bounds__(128, 1) mma_rate_kernel(int mma_iters, int ld_iters,
                                                          long long* cycles_mma, long long* cycles_ld,
                                                          uint32_t* sink) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* gen = smem_raw + (base - smem_u32(smem_raw));
  for (int i = threadIdx.x; i < (16384 + 32768) / 4; i += blockDim.x)
    reinterpret_cast<uint32_t*>(gen)[i] = 0x01010101u;
  const uint32_t barA = base + 16384 + 32768, tptr = barA + 16;
  if (threadIdx.x == 0) { mbar_init(barA, 1); fence_mbar_init(); }
  fence_proxy_async_smem();
  if (threadIdx.x < 32) tmem_alloc<512>(tptr);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *reinterpret_cast<volatile uint32_t*>(gen + 16384 + 32768 + 16);
  long long t0 = 0, t1 = 0;
  if (threadIdx.x == 0) {
    constexpr uint32_t idesc = umma_idesc_i8(128, 256);
    const uint64_t ad = umma_desc_sw128(base), bd = umma_desc_sw128(base + 16384);
    t0 = clock64();
    for (int it = 0; it < mma_iters; ++it) {
#pragma unroll
      for (int ks = 0; ks < 4; ++ks)
        mma_i8_ss(tmem + (it & 1) * 256, ad + 2 * ks, bd + 2 * ks, idesc, ks ? 1u : 0u);
    }
    tc_commit(barA);
    mbar_wait(barA, 0);
    t1 = clock64();
    cycles_mma[blockIdx.x] = t1 - t0;
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  {
    const int warp = threadIdx.x >> 5;
    const uint32_t taddr = tmem + (static_cast<uint32_t>(warp * 32) << 16);
    uint32_t acc = 0;
    const long long s0 = clock64();
    for (int it = 0; it < ld_iters; ++it) {
      uint32_t v[32];
      tmem_ld_32x32(taddr + (it & 15) * 32, v);
      tmem_ld_wait();
#pragma unroll
      for (int j = 0; j < 32; j += 8) acc ^= v[j];
    }
    const long long s1 = clock64();
    if (threadIdx.x == 0) cycles_ld[blockIdx.x] = s1 - s0;
    if (acc == 0x12345678u) sink[0] = acc;
  }
  tc_fence_before();
  __syncthreads();
  if (threadIdx.x < 32) { tc_fence_after(); tmem_dealloc<512>(tmem); }
}

// Epilogue-pipe interference probe (profiles/r2_gemm_pair_ncu.md): 16 warps on every SM; warps 0-7 stream the
// TMEM traffic of the pair kernel's epilogue (tcgen05.ld 32x32b.x16 + wait and / or two tcgen05.st 32x32b.x8 per 16
// columns), warps 8-15 a chain-free FFMA2 stream (32 per 16 columns, the two FMAs per element pair).  mode bit 0 =
// loads, bit 1 = stores, bit 2 = FFMA2.  out[0] / out[1] = clocks of a TMEM warp / an FFMA2 warp.
__global__ void __launch_bounds__(512, 1) epilogue_pipes_kernel(int mode, int iters, long long* out, float* sink) {
  __shared__ uint32_t tptr;
  const int warp = threadIdx.x >> 5;
  if (warp == 0) tmem_alloc<512>(smem_u32(&tptr));
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tb = tptr + (static_cast<uint32_t>((warp & 3) * 32) << 16);
  const bool do_ld = mode & 1, do_st = mode & 2, do_fma = mode & 4;
  const long long t0 = clock64();
  if (warp < 8) {
    uint32_t v[16], acc = 0, m[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) m[i] = 0x4B400000u + i;
    for (int it = 0; it < iters; ++it) {
      const uint32_t a = tb + (warp >> 2) * 96 + (it % 6) * 16;
      if (do_ld) { tmem_ld_32x16(a, v); tmem_ld_wait16(v); acc ^= v[0] ^ v[7] ^ v[15]; }
      if (do_st) { tmem_st_32x8(a, m); tmem_st_32x8(a + 8, m); }
    }
    if (do_st) tmem_st_wait();
    sink[threadIdx.x] = __uint_as_float(acc);
  } else if (do_fma) {
    uint64_t a[8];
    const uint64_t b2 = pack_f2(1.0001f, 0.9999f), c2 = pack_f2(0.5f, 0.25f);
#pragma unroll
    for (int j = 0; j < 8; ++j) a[j] = pack_f2(threadIdx.x * 0.001f + j, 1.f + j);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int j = 0; j < 8; ++j) a[j] = fma2(a[j], b2, c2);
    }
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < 8; ++j) { float lo, hi; unpack_f2(a[j], lo, hi); s += lo + hi; }
    sink[threadIdx.x] = s;
  }
  const long long t1 = clock64();
  if (blockIdx.x == 0 && (threadIdx.x & 31) == 0 && (warp == 0 || warp == 8)) out[warp >> 3] = t1 - t0;
  tc_fence_before();
  __syncthreads();
  if (warp == 0) { tc_fence_after(); tmem_dealloc<512>(tptr); }
}

int measure_epilogue_pipes(double* out, cudaStream_t st) {
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  long long* cyc = nullptr;
  float* sink = nullptr;
  if (cudaMalloc(&cyc, 2 * sizeof(long long)) != cudaSuccess) return APEX4_ERR_CUDA;
  if (cudaMalloc(&sink, 512 * sizeof(float)) != cudaSuccess) { cudaFree(cyc); return APEX4_ERR_CUDA; }
  const int iters = 3000;
  int rc = APEX4_OK;
  // out[2 m], out[2 m + 1], m = 1..7: clocks per 16 columns of a TMEM warp / per 32 FFMA2 of an FFMA2 warp in mode m
  for (int i = 0; i < 16; ++i) out[i] = 0.0;
  for (int mode = 1; mode < 8 && rc == APEX4_OK; ++mode) {
    for (int rep = 0; rep < 2; ++rep) {
      cudaMemsetAsync(cyc, 0, 2 * sizeof(long long), st);
      epilogue_pipes_kernel<<<sms, 512, 0, st>>>(mode, iters, cyc, sink);
    }
    long long h[2];
    if (cudaMemcpyAsync(h, cyc, sizeof(h), cudaMemcpyDeviceToHost, st) != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess) {
      rc = APEX4_ERR_CUDA;
      break;
    }
    out[2 * mode] = (mode & 3) ? static_cast<double>(h[0]) / iters : 0.0;
    out[2 * mode + 1] = (mode & 4) ? static_cast<double>(h[1]) / iters : 0.0;
  }
  cudaFree(cyc);
  cudaFree(sink);
  return cudaGetLastError() == cudaSuccess ? rc : APEX4_ERR_CUDA;
}

// The epilogue's own instruction stream, in isolation (profiles/r2_gemm_pair_ncu.md): eight warps (two per
// sub-partition) take a 192-column accumulator buffer through registers exactly as the pair kernel's group loop
// does -- tcgen05.ld 32x32b.x16 double-buffered, two tcgen05.st 32x32b.x8 of the bias behind each load, the chunk's 16
// token scales from shared memory, t = fma(word, a, b), acc = fma(t, sA, acc) on 96 accumulators -- with no barriers,
// no MMA and no wideners.  MODE bit 0 = the re-bias stores, bit 1 = the token-scale loads, bit 2 = the FMAs.
// LAYOUT 1 is the alternative fragment layout that was considered for the kernel: two tcgen05.ld.16x256b.x2 per 16-column
// chunk give a thread four weight rows x four tokens instead of one row x sixteen, so it needs one 16-byte load of token
// scales per chunk instead of four (and four {a, b} row pairs per group instead of one).
__device__ __forceinline__ void tmem_ld_16x256_x2(uint32_t taddr, uint32_t* v) {
  asm volatile("tcgen05.ld.sync.aligned.16x256b.x2.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
               : "r"(taddr)
               : "memory");
}
template <int MODE, int LAYOUT = 0>
__global__ void __launch_bounds__(256, 1) epilogue_stream_kernel(int groups, long long* out, float* sink) {
  __shared__ uint32_t tptr;
  __shared__ __align__(16) float sa[8][192];
  __shared__ __align__(8) float rowab[128][2];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x < 128) { rowab[threadIdx.x][0] = 1.0f / 256; rowab[threadIdx.x][1] = -49152.0f; }
  if (warp == 0) tmem_alloc<512>(smem_u32(&tptr));
  for (int i = threadIdx.x; i < 8 * 192; i += blockDim.x) (&sa[0][0])[i] = 1.0f + 1e-3f * static_cast<float>(i);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const int h = warp >> 2;
  const uint32_t tb0 = tptr + (static_cast<uint32_t>((warp & 3) * 32) << 16) + h * 96;
  uint64_t acc[48];
#pragma unroll
  for (int i = 0; i < 48; ++i) acc[i] = 0ull;
  uint32_t mg[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) mg[i] = 0x4B400000u;
  asm volatile("" : "+r"(mg[0]), "+r"(mg[1]), "+r"(mg[2]), "+r"(mg[3]), "+r"(mg[4]), "+r"(mg[5]), "+r"(mg[6]), "+r"(mg[7]));
  for (int b = 0; b < 2; ++b)
    for (int c = 0; c < 96; c += 8) tmem_st_32x8(tb0 + b * 192 + c, mg);
  tmem_st_wait();
  uint32_t v[2][16];
  float a = 1.0f / 256;
  const float bb = -49152.0f;
  auto load_chunk = [&](uint32_t addr, uint32_t (&d)[16]) {
    if constexpr (LAYOUT == 0) {
      tmem_ld_32x16(addr, d);
    } else {
      tmem_ld_16x256_x2(addr, d);                       // lanes 0-15 of the warp's quarter
      tmem_ld_16x256_x2(addr + (16u << 16), d + 8);     // lanes 16-31
    }
  };
  const long long t0 = clock64();
  load_chunk(tb0, v[0]);
  for (int g = 0; g < groups; ++g) {
    const uint32_t tb = tb0 + (g & 1) * 192;
    const uint32_t sAf = smem_u32(&sa[g & 7][h * 96]);
    const uint64_t a2 = pack_f2(a, a), b2 = pack_f2(bb, bb);
    float ra[4], rb[4];                                 // LAYOUT 1: {a, b} of the thread's four rows
    if constexpr (LAYOUT == 1) {
#pragma unroll
      for (int i = 0; i < 4; ++i) unpack_f2(lds64(smem_u32(&rowab[(warp & 3) * 32 + (lane >> 2) + 8 * i][0])), ra[i], rb[i]);
    }
#pragma unroll
    for (int c = 0; c < 6; ++c) {
      uint32_t* vc = v[c & 1];
      uint64_t sq[8];
      if (MODE & 2) {
        if constexpr (LAYOUT == 0) {
#pragma unroll
          for (int i = 0; i < 4; ++i) lds_2x64(sAf + 64 * c + 16 * i, sq[2 * i], sq[2 * i + 1]);
        } else {
          lds_2x64(sAf + 64 * c + 16 * (lane & 3), sq[0], sq[1]);   // the thread's four columns of the chunk (slot permuted)
        }
      } else {
#pragma unroll
        for (int i = 0; i < 8; ++i) sq[i] = pack_f2(1.f + i, 2.f + c);
      }
      tmem_ld_wait16(vc);
      load_chunk(c < 5 ? tb + 16 * (c + 1) : tb0 + ((g + 1) & 1) * 192, v[(c + 1) & 1]);
      if (MODE & 1) {
        tmem_st_32x8(tb + 16 * c, mg);
        tmem_st_32x8(tb + 16 * c + 8, mg);
      }
      if (MODE & 4) {
        if constexpr (LAYOUT == 0) {
#pragma unroll
          for (int jj = 0; jj < 8; ++jj) fma2_acc(acc[c * 8 + jj], fma2v(pack_u2(vc[2 * jj], vc[2 * jj + 1]), a2, b2), sq[jj]);
        } else {
          // registers of one load: {row 0 pair 0, row 1 pair 0, row 0 pair 1, row 1 pair 1}; the second load: rows 2, 3
#pragma unroll
          for (int q = 0; q < 8; ++q) {
            const int row = 2 * (q >> 2) + (q & 1), pr = (q >> 1) & 1;
            fma2_acc(acc[c * 8 + q], fma2v(pack_u2(vc[2 * q], vc[2 * q + 1]), pack_f2(ra[row], ra[row]), pack_f2(rb[row], rb[row])), sq[pr]);
          }
        }
      } else {
        acc[c] ^= pack_u2(vc[0] ^ vc[15], vc[8]) ^ sq[0] ^ sq[7];
      }
    }
    a += 1e-6f;
  }
  tmem_ld_wait16(v[0]);
  tmem_st_wait();
  const long long t1 = clock64();
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < 48; ++i) { float lo, hi; unpack_f2(acc[i], lo, hi); s += lo + hi; }
  sink[threadIdx.x] = s + __uint_as_float(v[0][0]);
  if (blockIdx.x == 0 && threadIdx.x == 0) out[0] = t1 - t0;
  tc_fence_before();
  __syncthreads();
  if (warp == 0) { tc_fence_after(); tmem_dealloc<512>(tptr); }
}

template <int MODE, int LAYOUT = 0>
static double run_epilogue_stream(long long* cyc, float* sink, cudaStream_t st) {
  const int groups = 2000;
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  for (int rep = 0; rep < 2; ++rep) epilogue_stream_kernel<MODE, LAYOUT><<<sms, 256, 0, st>>>(groups, cyc, sink);
  long long h = 0;
  if (cudaMemcpyAsync(&h, cyc, sizeof(h), cudaMemcpyDeviceToHost, st) != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess) return -1.0;
  return static_cast<double>(h) / groups;
}

int measure_epilogue_stream(double* out, cudaStream_t st) {
  long long* cyc = nullptr;
  float* sink = nullptr;
  if (cudaMalloc(&cyc, sizeof(long long)) != cudaSuccess) return APEX4_ERR_CUDA;
  if (cudaMalloc(&sink, 256 * sizeof(float)) != cudaSuccess) { cudaFree(cyc); return APEX4_ERR_CUDA; }
  // clocks per 192-column group: loads only; + stores; loads + FMAs; + stores; loads + scales + FMAs; everything
  out[0] = run_epilogue_stream<0>(cyc, sink, st);
  out[1] = run_epilogue_stream<1>(cyc, sink, st);
  out[2] = run_epilogue_stream<4>(cyc, sink, st);
  out[3] = run_epilogue_stream<5>(cyc, sink, st);
  out[4] = run_epilogue_stream<6>(cyc, sink, st);
  out[5] = run_epilogue_stream<7>(cyc, sink, st);
  // the 16x256b fragment layout: loads only; everything
  out[6] = run_epilogue_stream<0, 1>(cyc, sink, st);
  out[7] = run_epilogue_stream<7, 1>(cyc, sink, st);
  cudaFree(cyc);
  cudaFree(sink);
  for (int i = 0; i < 8; ++i) if (out[i] < 0.0) return APEX4_ERR_CUDA;
  return cudaGetLastError() == cudaSuccess ? APEX4_OK : APEX4_ERR_CUDA;
}

__global__ void clock_probe_kernel(long long* out) {
  unsigned long long g0, g1;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
  const long long c0 = clock64();
  do {
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
  } while (g1 - g0 < 200000ull);   // 200 us
  const long long c1 = clock64();
  out[0] = c1 - c0;
  out[1] = static_cast<long long>(g1 - g0);
}

static float time_ms(cudaEvent_t a, cudaEvent_t b) {
  float ms = 0.f;
  cudaEventElapsedTime(&ms, a, b);
  return ms;
}

int measure_rho(double* out, cudaStream_t st) {
  for (int i = 0; i < 8; ++i) out[i] = 0.0;
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  float* buf = nullptr;
  long long* cyc = nullptr;
  const int blocks = sms * 8, threads = 256;
  if (cudaMalloc(&buf, sizeof(float) * blocks * threads) != cudaSuccess) return APEX4_ERR_CUDA;
  if (cudaMalloc(&cyc, sizeof(long long) * (2 * sms + 2)) != cudaSuccess) { cudaFree(buf); return APEX4_ERR_CUDA; }
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const int iters = 4096;
  int rc = APEX4_OK;
  // FP32 FMA (scalar and packed)
  double best_fma = 0, best_fma2 = 0, best_i2f = 0;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, st);
    fma_rate_kernel<<<blocks, threads, 0, st>>>(buf, iters, 1.0001f, 0.5f);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) { rc = APEX4_ERR_CUDA; break; }
    double fl = 2.0 * blocks * threads * double(iters) * kChains / (time_ms(e0, e1) * 1e-3);
    if (rep && fl > best_fma) best_fma = fl;
    cudaEventRecord(e0, st);
    fma2_rate_kernel<<<blocks, threads, 0, st>>>(buf, iters, 1.0001f, 0.5f);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) { rc = APEX4_ERR_CUDA; break; }
    fl = 4.0 * blocks * threads * double(iters) * kChains / (time_ms(e0, e1) * 1e-3);
    if (rep && fl > best_fma2) best_fma2 = fl;
    cudaEventRecord(e0, st);
    i2f_rate_kernel<<<blocks, threads, 0, st>>>(buf, iters);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) { rc = APEX4_ERR_CUDA; break; }
    fl = 1.0 * blocks * threads * double(iters) * kChains / (time_ms(e0, e1) * 1e-3);
    if (rep && fl > best_i2f) best_i2f = fl;
  }
  // INT8 tcgen05 MMA + TMEM read
  double best_mma = 0, ld_bytes_per_clk = 0;
  if (rc == APEX4_OK) {
    cudaFuncSetAttribute(mma_rate_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kMmaSmem);
    const int mma_iters = 8192, ld_iters = 4096;
    for (int rep = 0; rep < 3; ++rep) {
      cudaEventRecord(e0, st);
      mma_rate_kernel<<<sms, 128, kMmaSmem, st>>>(mma_iters, ld_iters, cyc, cyc + sms,
                                                  reinterpret_cast<uint32_t*>(buf));
      cudaEventRecord(e1, st);
      if (cudaEventSynchronize(e1) != cudaSuccess) { rc = APEX4_ERR_CUDA; break; }
    }
    if (rc == APEX4_OK) {
      long long h[2];
      cudaMemcpy(h, cyc, sizeof(long long), cudaMemcpyDeviceToHost);
      cudaMemcpy(h + 1, cyc + sms, sizeof(long long), cudaMemcpyDeviceToHost);
      // per-SM MACs per clock from the issuing thread's own cycle counter
      const double macs = double(mma_iters) * 4 * 128.0 * 256.0 * 32.0;
      out[6] = macs / double(h[0]);                               // INT8 MAC / clk / SM
      ld_bytes_per_clk = double(ld_iters) * 4 * 4096.0 / double(h[1]);   // 4 warps x 4 KB per ld
      out[7] = ld_bytes_per_clk;                                  // TMEM read B / clk / SM
    }
  }
  // SM clock while idle-ish (context for the per-clock numbers)
  double mhz = 0;
  if (rc == APEX4_OK) {
    clock_probe_kernel<<<1, 1, 0, st>>>(cyc + 2 * sms);
    long long h[2];
    if (cudaMemcpy(h, cyc + 2 * sms, 2 * sizeof(long long), cudaMemcpyDeviceToHost) == cudaSuccess && h[1] > 0)
      mhz = double(h[0]) / double(h[1]) * 1e3;
    else rc = APEX4_ERR_CUDA;
  }
  if (rc == APEX4_OK) {
    // chip-level INT8 rate: time a long MMA-only launch with events
    const int mma_iters = 32768;
    cudaEventRecord(e0, st);
    mma_rate_kernel<<<sms, 128, kMmaSmem, st>>>(mma_iters, 1, cyc, cyc + sms,
                                                reinterpret_cast<uint32_t*>(buf));
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) == cudaSuccess) {
      const double ops = 2.0 * sms * double(mma_iters) * 4 * 128.0 * 256.0 * 32.0;
      best_mma = ops / (time_ms(e0, e1) * 1e-3);
    } else rc = APEX4_ERR_CUDA;
  }
  out[0] = best_mma * 1e-12;                                  // INT8 TOPS (dense, kind::i8)
  out[1] = (best_fma2 > best_fma ? best_fma2 : best_fma) * 1e-12;   // FP32 TFLOPS (best of FFMA / FFMA2)
  out[2] = best_i2f * 1e-9;                                   // INT32->FP32 Gop/s
  out[3] = out[1] > 0 ? out[0] / out[1] : 0;                  // rho = tensor ops / CUDA-core flops
  out[4] = ld_bytes_per_clk * sms * mhz * 1e6 * 1e-9;         // TMEM read GB/s (chip)
  out[5] = mhz;
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(buf);
  cudaFree(cyc);
  return cudaGetLastError() == cudaSuccess ? rc : APEX4_ERR_CUDA;
}

}  // namespace apex4
