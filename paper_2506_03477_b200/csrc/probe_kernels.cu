// Issue-rate probes that measure the roofline denominators of the two MMA pipes the path uses, on
// the device the library runs on (MEASURED_PEAKS.json has no FP64 / TF32 figure):
//   FP64: register-resident DMMA.8x8x4 loop (no memory traffic) -> FP64 tensor-pipe peak.
//   TF32 / F16: back-to-back tcgen05.mma 128x128xK (A in TMEM, B in shared memory, no global traffic).
// They do no work of the method; bench.py reports them as `peak` beside the achieved rate.
#include <cuda_fp16.h>

#include "kernels.h"
#include "ptx.cuh"

namespace qsgw {

namespace {

constexpr int kProbeThreads = 256;
constexpr int kProbeAcc = 16;    // independent accumulator pairs per warp (hides the DMMA latency)

__global__ void __launch_bounds__(kProbeThreads) dmma_peak_kernel(int iters, double* sink) {
  double c0[kProbeAcc], c1[kProbeAcc];
#pragma unroll
  for (int i = 0; i < kProbeAcc; ++i) {
    c0[i] = 0.0;
    c1[i] = 0.0;
  }
  const double a = 1.0 + 1e-9 * threadIdx.x, b = 1.0 - 1e-9 * threadIdx.x;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < kProbeAcc; ++i) dmma884(c0[i], c1[i], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < kProbeAcc; ++i) s += c0[i] + c1[i];
  if (s == 123.456) sink[0] = s;   // never true: keeps the loop alive
}

}  // namespace

// Runs the FP64 probe on `s`; returns real TFLOP/s (2 flop per FMA, 256 FMA per DMMA.8x8x4).
cudaError_t probe_fp64_mma(cudaStream_t s, double* out_tflops, double* out_ms) {
  int dev = 0, n_sm = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return e;
  double* sink = nullptr;
  e = cudaMalloc(&sink, sizeof(double));
  if (e != cudaSuccess) return e;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const int blocks = n_sm * 4, iters = 40000;
  dmma_peak_kernel<<<blocks, kProbeThreads, 0, s>>>(2000, sink);   // warm-up (clocks ramp)
  float best = 1e30f;
  for (int rep = 0; rep < 3; ++rep) {
    cudaEventRecord(e0, s);
    dmma_peak_kernel<<<blocks, kProbeThreads, 0, s>>>(iters, sink);
    cudaEventRecord(e1, s);
    e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  if (e != cudaSuccess) return e;
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const double flop = 2.0 * 256.0 * kProbeAcc * (double)iters * (kProbeThreads / 32) * blocks;
  if (out_tflops) *out_tflops = flop / (best * 1e-3) / 1e12;
  if (out_ms) *out_ms = best;
  return cudaSuccess;
}


namespace {

constexpr int kProbeTile = 128 * 128;     // bytes of one 128-row x 128-byte K-major operand tile

// Issue-rate probe of the 5th-generation tensor pipe: every SM issues back-to-back 128x128 MMAs of one K step
// (kind::tf32: K = 8, kind::f16: K = 16).  The operand contents are arbitrary finite numbers.
template <bool F16>
__global__ void __launch_bounds__(128, 1) umma_peak_kernel(int iters) {
  extern __shared__ unsigned char smem_dyn[];
  const uint32_t raw = smem_u32(smem_dyn);
  const uint32_t base = (raw + 1023u) & ~1023u;
  unsigned char* sm = smem_dyn + (base - raw);
  uint64_t* bar = reinterpret_cast<uint64_t*>(sm + kProbeTile);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bar + 1);
  const int tid = threadIdx.x, warp = tid >> 5;
  if (F16) {
    for (int i = tid; i < kProbeTile / 2; i += 128) reinterpret_cast<__half*>(sm)[i] = __float2half(1.0f + 0.001f * (i & 255));
  } else {
    for (int i = tid; i < kProbeTile / 4; i += 128) reinterpret_cast<float*>(sm)[i] = 1.0f + 0.001f * (i & 255);
  }
  if (tid == 0) {
    mbar_init(bar, 1);
    mbar_fence_init();
  }
  if (warp == 0) tmem_alloc(tmem_slot, 512);
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tbase = *tmem_slot;
  uint32_t v[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    if (F16) {
      const __half2 t = __floats2half2_rn(0.5f + 0.01f * i, 0.25f + 0.01f * i);
      v[i] = *reinterpret_cast<const uint32_t*>(&t);
    } else {
      v[i] = cvt_tf32_rna(0.5f + 0.01f * i);
    }
  }
  tmem_st16(tbase + 256 + ((uint32_t)(32 * warp) << 16), v);
  tmem_st16(tbase + 272 + ((uint32_t)(32 * warp) << 16), v);
  tmem_wait_st();
  tc_fence_before();
  __syncthreads();
  if (tid == 0) {
    tc_fence_after();
    const uint32_t idesc = F16 ? umma_idesc_f16(128, 128, 0) : umma_idesc_tf32(128, 128, 0);
    const uint64_t bd = umma_desc_k_sw128(base);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int g = 0; g < 4; ++g) {
        const uint32_t acc = (it | g) ? 1u : 0u;
        if (F16) {
          umma_f16_ts(tbase, tbase + 256 + 8 * g, bd + (uint64_t)(2 * g), idesc, acc);
          umma_f16_ts(tbase + 128, tbase + 256 + 8 * g, bd + (uint64_t)(2 * g), idesc, acc);
        } else {
          umma_tf32_ts(tbase, tbase + 256 + 8 * g, bd + (uint64_t)(2 * g), idesc, acc);
          umma_tf32_ts(tbase + 128, tbase + 256 + 8 * g, bd + (uint64_t)(2 * g), idesc, acc);
        }
      }
    }
    umma_commit(bar);
    mbar_wait(bar, 0);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tbase, 512);
}

template <bool F16>
cudaError_t probe_umma(cudaStream_t s, double* out_tflops, double* out_ms) {
  int dev = 0, n_sm = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(umma_peak_kernel<F16>, cudaFuncAttributeMaxDynamicSharedMemorySize, 20480);
  if (e != cudaSuccess) return e;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const int iters = 40000;
  umma_peak_kernel<F16><<<n_sm, 128, 20480, s>>>(iters / 4);
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, s);
    umma_peak_kernel<F16><<<n_sm, 128, 20480, s>>>(iters);
    cudaEventRecord(e1, s);
    e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (e != cudaSuccess) return e;
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const double flop = 2.0 * 128.0 * 128.0 * (F16 ? 16.0 : 8.0) * 8.0 * (double)iters * n_sm;
  if (out_tflops) *out_tflops = flop / (best * 1e-3) / 1e12;
  if (out_ms) *out_ms = best;
  return cudaSuccess;
}

}  // namespace

cudaError_t probe_tf32_mma(cudaStream_t s, double* out_tflops, double* out_ms) { return probe_umma<false>(s, out_tflops, out_ms); }
cudaError_t probe_f16_mma(cudaStream_t s, double* out_tflops, double* out_ms) { return probe_umma<true>(s, out_tflops, out_ms); }

}  // namespace qsgw
