// FP64 peak probe: the denominator of the solve's roofline (bench.py --probe-fp64, `roofline_solve`).  MEASURED_PEAKS.json
// carries HBM and bf16 numbers only, so the FP64 pipe is measured here, on the device the bench runs on: register-resident
// chains of DFMA (vector FP64) and of mma.sync.m8n8k4.f64 (DMMA, the tensor path of the dense tile updates), enough
// independent chains per thread to cover the pipe latency, CUDA events around a launch that fills every SM.
#include "sim3ba_internal.cuh"

namespace sim3ba {

namespace {

constexpr int kProbeThreads = 256;
constexpr int kProbeChains = 8;

__global__ void __launch_bounds__(kProbeThreads)
k_probe_dfma(double* out, int iters, double a, double b) {
  double v[kProbeChains];
#pragma unroll
  for (int k = 0; k < kProbeChains; ++k) v[k] = (double)(threadIdx.x + k);
  for (int it = 0; it < iters; ++it)
#pragma unroll
    for (int k = 0; k < kProbeChains; ++k) v[k] = fma(v[k], a, b);
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < kProbeChains; ++k) s += v[k];
  if (s == 123.456) out[blockIdx.x * kProbeThreads + threadIdx.x] = s;   // never true: keeps the chains alive
}

__global__ void __launch_bounds__(kProbeThreads)
k_probe_dmma(double* out, int iters, double a, double b) {
  double c0[kProbeChains], c1[kProbeChains];
#pragma unroll
  for (int k = 0; k < kProbeChains; ++k) { c0[k] = (double)k; c1[k] = (double)(threadIdx.x & 3); }
  for (int it = 0; it < iters; ++it)
#pragma unroll
    for (int k = 0; k < kProbeChains; ++k)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                   : "+d"(c0[k]), "+d"(c1[k]) : "d"(a), "d"(b));
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < kProbeChains; ++k) s += c0[k] + c1[k];
  if (s == 123.456) out[blockIdx.x * kProbeThreads + threadIdx.x] = s;
}

}  // namespace

// TFLOP/s of the two probes (best of `reps` launches)
cudaError_t run_probe_fp64(cudaStream_t st, double* dfma_tflops, double* dmma_tflops) {
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return e;
  const int grid = sms * 8, iters = 4096, reps = 5;
  double* d_out = nullptr;
  e = cudaMalloc(reinterpret_cast<void**>(&d_out), (size_t)grid * kProbeThreads * sizeof(double));
  if (e != cudaSuccess) return e;
  cudaEvent_t ev0, ev1;
  cudaEventCreate(&ev0);
  cudaEventCreate(&ev1);
  double best[2] = {0.0, 0.0};
  for (int which = 0; which < 2; ++which)
    for (int r = 0; r < reps + 1; ++r) {   // the first launch warms up
      cudaEventRecord(ev0, st);
      if (which == 0) k_probe_dfma<<<grid, kProbeThreads, 0, st>>>(d_out, iters, 0.999999, 1e-9);
      else k_probe_dmma<<<grid, kProbeThreads, 0, st>>>(d_out, iters, 0.999999, 1e-9);
      cudaEventRecord(ev1, st);
      e = cudaEventSynchronize(ev1);
      if (e != cudaSuccess) break;
      float ms = 0.f;
      cudaEventElapsedTime(&ms, ev0, ev1);
      // DFMA: 2 flop per thread and instruction; DMMA m8n8k4: 2 * 8 * 8 * 4 = 512 flop per warp and instruction
      const double flop = which == 0 ? 2.0 * kProbeChains * (double)iters * grid * kProbeThreads
                                     : 512.0 * kProbeChains * (double)iters * grid * (kProbeThreads / 32);
      if (r > 0 && ms > 0.f) best[which] = std::max(best[which], flop / (ms * 1e-3) / 1e12);
    }
  cudaEventDestroy(ev0);
  cudaEventDestroy(ev1);
  cudaFree(d_out);
  if (e == cudaSuccess) e = cudaGetLastError();
  *dfma_tflops = best[0];
  *dmma_tflops = best[1];
  return e;
}

}  // namespace sim3ba
