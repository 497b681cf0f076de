// Packed fp32x2 arithmetic (sm_100: FFMA2 / FMUL2 / FADD2, one issue slot for two lanes) and the approximate
// MUFU reciprocals, shared by the per-match kernels (k_accumulate.cu, k_depth.cu).  The two lanes of every
// float2 are TWO DIFFERENT MATCHES (A, B) of the same thread.
#pragma once
#include <cuda_runtime.h>

namespace sim3ba {

using f2 = float2;
__device__ __forceinline__ f2 operator*(f2 a, f2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ f2 operator+(f2 a, f2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ f2 operator-(f2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ f2 bc(float s) { return make_float2(s, s); }

// MUFU.RSQ / MUFU.RCP without the denormal pre/post-scaling of rsqrtf() / 1/x: arguments are clamped or
// may legitimately give +inf (handled by the min() that follows)
__device__ __forceinline__ float rsq(float v) {
  float r;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(v));
  return r;
}
__device__ __forceinline__ float rcp(float v) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(v));
  return r;
}

}  // namespace sim3ba
