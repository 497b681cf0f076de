// Kernel 5 of the Sim(3) GN step: retraction T_WCi <- Exp(tau_i) T_WCi (a8).
// FP64, one thread per keyframe; gauge keyframes are skipped (their tau is exactly zero).
#include "sim3ba_internal.cuh"
#include "sim3_math.cuh"

namespace sim3ba {

namespace {

__global__ void k_retract(double* __restrict__ poses, const double* __restrict__ tau, const uint8_t* __restrict__ fixed,
                          const int32_t* __restrict__ fail_flag, int N) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= N || fixed[k] || *fail_flag) return;
  double p[8], t[7];
#pragma unroll
  for (int a = 0; a < 8; ++a) p[a] = poses[8 * k + a];
#pragma unroll
  for (int a = 0; a < 7; ++a) t[a] = tau[7 * k + a];
  retract_pose(p, t);
#pragma unroll
  for (int a = 0; a < 8; ++a) poses[8 * k + a] = p[a];
}

}  // namespace

cudaError_t launch_retract(Ctx* c) {
  k_retract<<<(c->N + 127) / 128, 128, 0, c->stream>>>(c->poses, c->tau, c->fixed_mask, c->fail_flag, c->N);
  ++c->launches;
  return cudaGetLastError();
}

}  // namespace sim3ba
