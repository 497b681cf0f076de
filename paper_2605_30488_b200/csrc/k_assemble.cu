// Kernel 3 of the Sim(3) GN step: block-sparse -> dense assembly (a6).
//
// Every edge e = (i, j) contributes H_ii += A_e, H_jj += A_e, H_ij -= A_e, H_ji -= A_e,
// g_j += b_e, g_i -= b_e ("two diagonal and one off-diagonal 7x7 blocks").  The
// scatter is a GATHER over the bookkeeping CSRs built at create (keyframe -> incident edges,
// unique keyframe pair -> edges), so no atomics are needed and the summation order is fixed.
// Gauge keyframes get an identity diagonal block, zero off-diagonal blocks and zero
// gradient, so tau_fixed = 0 exactly.  Damping of Eq. (7): diag <- diag (1 + lambda) + eps.
// Only the lower triangle (row >= col) is written; the destination is zero-filled first.
#include "sim3ba_internal.cuh"

namespace sim3ba {

namespace {

__device__ __forceinline__ int tri_index(int r, int c) {  // upper-triangular row-major, r <= c
  return r * 7 - r * (r - 1) / 2 + (c - r);
}

__global__ void __launch_bounds__(64)
k_scatter_blocks(double* __restrict__ dst, int ld, const double* __restrict__ blocks35,
                 const int32_t* __restrict__ kf_ptr, const int32_t* __restrict__ kf_edge,
                 const int32_t* __restrict__ pair_kf, const int32_t* __restrict__ pair_ptr,
                 const int32_t* __restrict__ pair_edge, const uint8_t* __restrict__ fixed, int N, int n_pairs,
                 int n, int npad, double lambda, double eps) {
  const int b = blockIdx.x, t = threadIdx.x;
  const int r = t / 7, c = t % 7;
  if (b < N) {  // diagonal block of keyframe b
    if (t >= 49 || r < c) return;
    double v = 0.0;
    if (fixed[b]) {
      v = (r == c) ? 1.0 : 0.0;
    } else {
      const int idx = tri_index(c, r);
      for (int p = kf_ptr[b]; p < kf_ptr[b + 1]; ++p) v += blocks35[(size_t)kf_edge[p] * 35 + idx];
    }
    if (r == c) v = v * (1.0 + lambda) + eps;
    dst[(size_t)(7 * b + r) * ld + 7 * b + c] = v;
  } else if (b < N + n_pairs) {  // off-diagonal block (hi, lo), hi > lo
    if (t >= 49) return;
    const int p = b - N;
    const int hi = pair_kf[2 * p], lo = pair_kf[2 * p + 1];
    if (fixed[hi] || fixed[lo]) return;  // stays zero
    const int idx = r <= c ? tri_index(r, c) : tri_index(c, r);
    double v = 0.0;
    for (int q = pair_ptr[p]; q < pair_ptr[p + 1]; ++q) v += blocks35[(size_t)pair_edge[q] * 35 + idx];
    dst[(size_t)(7 * hi + r) * ld + 7 * lo + c] = -v;
  } else {  // identity padding rows n..npad-1
    for (int k = n + t; k < npad; k += blockDim.x) dst[(size_t)k * ld + k] = 1.0;
  }
}

// dense source (sim3ba_load_system): dst = lower(src) with gauge rows/cols -> identity and damping
__global__ void k_damp_copy(double* __restrict__ dst, const double* __restrict__ src, const uint8_t* __restrict__ fixed,
                            int n, int npad, double lambda, double eps) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  const int r = blockIdx.y;
  if (c >= npad) return;
  double v = 0.0;
  if (r >= n || c >= n) {
    v = (r == c) ? 1.0 : 0.0;
  } else if (c <= r) {
    if (fixed[r / 7] || fixed[c / 7]) v = (r == c) ? 1.0 : 0.0;
    else v = src[(size_t)r * n + c];
    if (r == c) v = v * (1.0 + lambda) + eps;
  }
  dst[(size_t)r * npad + c] = v;
}

// g from the per-edge b_e (gather over the keyframe -> edge CSR); the last block sums the per-edge robust costs instead
__global__ void __launch_bounds__(128)
k_gradient_cost(double* __restrict__ g, const double* __restrict__ blocks35, const int32_t* __restrict__ edges,
                const int32_t* __restrict__ kf_ptr, const int32_t* __restrict__ kf_edge, const uint8_t* __restrict__ fixed, int N,
                const double* __restrict__ edge_cost, int E, double* __restrict__ total) {
  if (blockIdx.x == gridDim.x - 1) {
    __shared__ double s[128];
    double v = 0.0;
    for (int e = threadIdx.x; e < E; e += 128) v += edge_cost[e];
    s[threadIdx.x] = v;
    __syncthreads();
    for (int o = 64; o > 0; o >>= 1) {
      if (threadIdx.x < o) s[threadIdx.x] += s[threadIdx.x + o];
      __syncthreads();
    }
    if (threadIdx.x == 0) *total = s[0];
    return;
  }
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= 7 * N) return;
  const int k = idx / 7, comp = idx % 7;
  double v = 0.0;
  if (!fixed[k]) {
    for (int p = kf_ptr[k]; p < kf_ptr[k + 1]; ++p) {
      const int e = kf_edge[p];
      const double b = blocks35[(size_t)e * 35 + 28 + comp];
      v += (edges[2 * e + 1] == k) ? b : -b;
    }
  }
  g[idx] = v;
}

__global__ void k_load_gradient(double* __restrict__ g, const double* __restrict__ src, const uint8_t* __restrict__ fixed, int n) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < n) g[idx] = fixed[idx / 7] ? 0.0 : src[idx];
}

}  // namespace

cudaError_t launch_assemble(Ctx* c, double* dst, double lambda, double eps, bool from_dense) {
  if (from_dense) {
    dim3 grid((c->npad + 255) / 256, c->npad);
    k_damp_copy<<<grid, 256, 0, c->stream>>>(dst, c->Hd, c->fixed_mask, c->n, c->npad, lambda, eps);
    ++c->launches;
    return cudaGetLastError();
  }
  cudaError_t err = cudaMemsetAsync(dst, 0, (size_t)c->npad * c->npad * sizeof(double), c->stream);
  if (err != cudaSuccess) return err;
  k_scatter_blocks<<<c->N + c->n_pairs + 1, 64, 0, c->stream>>>(dst, c->npad, c->blocks35, c->kf_ptr, c->kf_edge,
                                                                c->pair_kf, c->pair_ptr, c->pair_edge, c->fixed_mask,
                                                                c->N, c->n_pairs, c->n, c->npad, lambda, eps);
  ++c->launches;
  return cudaGetLastError();
}

cudaError_t launch_gradient(Ctx* c) {
  k_gradient_cost<<<(7 * c->N + 127) / 128 + 1, 128, 0, c->stream>>>(c->g, c->blocks35, c->edges, c->kf_ptr, c->kf_edge, c->fixed_mask, c->N,
                                                                     c->edge_cost, c->E, c->total_cost);
  ++c->launches;
  return cudaGetLastError();
}

cudaError_t launch_load_gradient(Ctx* c, const double* d_g) {
  k_load_gradient<<<(c->n + 127) / 128, 128, 0, c->stream>>>(c->g, d_g, c->fixed_mask, c->n);
  ++c->launches;
  return cudaGetLastError();
}

}  // namespace sim3ba
