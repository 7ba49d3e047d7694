// Issue-rate probes that measure the roofline denominators of the two MMA pipes the path uses, on
// the device the library runs on (MEASURED_PEAKS.json has no FP64 / TF32 figure):
//   FP64: register-resident DMMA.8x8x4 loop (no memory traffic) -> FP64 tensor-pipe peak.
// They do no work of the method; bench.py reports them as `peak` beside the achieved rate.
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

}  // namespace qsgw
