// a6: damped assembly of ONE 64x64 tile of the 7N system, shared by the
// stand-alone assembly kernel (first attempt) and the persistent solve kernel (epsilon retries).
//
// Every edge e = (i, j) contributes H_ii += A_e, H_jj += A_e, H_ij -= A_e, H_ji -= A_e ("two diagonal
// and one off-diagonal 7x7 blocks").  The scatter is a GATHER: the CTA that owns a tile
// computes each of its elements from the per-edge blocks through the bookkeeping CSRs built at create
// (keyframe -> incident edges, unordered keyframe pair -> edges), so there are no atomics, the
// summation order is fixed and no tile is written twice.  Gauge keyframes get identity
// rows/columns; rows >= n are identity padding.  Damping of Eq. (7): diag <- diag (1 + lambda) + eps.
// Only row >= col is meaningful; the strict upper triangle of diagonal tiles is written as zero.
#pragma once
#include "sim3ba_internal.cuh"

namespace sim3ba {

struct AsmArgs {
  double* L; int npad, n, N;
  const double* blocks35;
  const int32_t *kf_ptr, *kf_edge, *pair_kf, *pairhi_ptr, *pair_ptr, *pair_edge;
  const uint8_t* fixed;
  const double* dense;   // non-NULL: caller-supplied dense H [n][n] (sim3ba_load_system) instead of the blocks
  const double* g;
  double* rhs;           // rhs = -g (written by the diagonal tiles), NULL: not written
  double lambda;
};

__device__ __forceinline__ int tri7(int r, int c) { return r * 7 - r * (r - 1) / 2 + (c - r); }   // r <= c

static __device__ __noinline__ double asm_element(const AsmArgs& a, int R, int C, double eps) {
  if (C > R) return 0.0;
  if (R >= a.n) return (R == C) ? 1.0 : 0.0;
  const int kr = R / 7, kc = C / 7;
  if (a.fixed[kr] || a.fixed[kc]) return (R == C) ? 1.0 : 0.0;
  double v = 0.0;
  if (a.dense) {
    v = a.dense[(size_t)R * a.n + C];
  } else {
    const int ar = R - 7 * kr, ac = C - 7 * kc;
    if (kr == kc) {
      const int idx = tri7(ac, ar);
      for (int p = a.kf_ptr[kr]; p < a.kf_ptr[kr + 1]; ++p) v += a.blocks35[(size_t)a.kf_edge[p] * 35 + idx];
    } else {
      const int idx = ar <= ac ? tri7(ar, ac) : tri7(ac, ar);
      for (int p = a.pairhi_ptr[kr]; p < a.pairhi_ptr[kr + 1]; ++p) {
        if (a.pair_kf[2 * p + 1] != kc) continue;
        for (int q = a.pair_ptr[p]; q < a.pair_ptr[p + 1]; ++q) v += a.blocks35[(size_t)a.pair_edge[q] * 35 + idx];
        v = -v;
        break;
      }
    }
  }
  if (R == C) v = v * (1.0 + a.lambda) + eps;
  return v;
}

// 256 threads: thread (row = tid / 4, quarter = tid % 4) writes 16 consecutive doubles of its row
static __device__ __noinline__ void assemble_tile(const AsmArgs& a, int ti, int tj, double eps, int tid) {
  const int rr = tid >> 2, q = tid & 3;
  const int R = ti * kNB + rr;
  double* dst = a.L + (size_t)R * a.npad + (size_t)tj * kNB + 16 * q;
#pragma unroll 1
  for (int k = 0; k < 16; k += 2) {
    const int C = tj * kNB + 16 * q + k;
    double2 v;
    v.x = asm_element(a, R, C, eps);
    v.y = asm_element(a, R, C + 1, eps);
    *reinterpret_cast<double2*>(dst + k) = v;
  }
  if (a.rhs && ti == tj && tid < kNB) {
    const int r = ti * kNB + tid;
    a.rhs[r] = (r < a.n) ? -a.g[r] : 0.0;
  }
}

}  // namespace sim3ba
